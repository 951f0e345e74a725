#!/usr/bin/env python
"""Benchmark of the ARKCoS hot path on B200: output Mpix/s per map at HEALPix Nside=2048 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--cfg 4]

One "step" = one arkcos_convolve of the whole hot path (kernel rows -> ring FFT -> band MAC -> inverse FFT) over the
config-4 workload (HEALPix nside 2048, white noise + 1000 point sources, Gaussian FWHM 5', theta_max 15').
Prints ONE JSON line (rank 0).  N > 1: every rank convolves its own map (maps are independent problems, no
collective on the data path) -> "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1104_0672_b200 import inputs  # noqa: E402
from paper_1104_0672_b200.sharding import shard_range  # noqa: E402

METRIC = "output Mpix/s per map at HEALPix Nside=2048"
# dram__bytes_read.sum + dram__bytes_write.sum per launch (bytes) from the ncu --set full captures summarised in
# profiles/ (config 4, one map); None where no capture exists
TRAFFIC = {  # profiles/r1_v8_final.md (ncu --set full, config 4, one map); FFT entries = sum over the size classes
    "band_mac_eq_kernel": 224e6 + 111e6,
    "band_mac_capchunk_kernel<4,20>": 138e6 + 30e6,
    "ring_fft3_forward_kernel (all transform sizes)": 306e6 + 149e6 + 42e6 + 1e6 + 11e6 + 3e6,
    "ring_fft3_inverse_kernel (all transform sizes)": 309e6 + 149e6 + 42e6 + 1e6 + 11e6 + 3e6,
}
UNIT = "Mpix/s"


def workload(cfg: int, which: int = 1):
    c = inputs.config(cfg)
    if cfg == 5:
        k = c["kernels"][which]
        c = dict(c, **k)
    tab = inputs.kernel_table(c)
    pix = c["pix"]
    npix = pix[1] * pix[2] if pix[0] == "ecp" else 12 * pix[1] ** 2
    nmaps = c["nmaps"]
    x = inputs.white_noise_maps(npix, cfg, nmaps)
    if c.get("point_sources"):
        x = inputs.add_point_sources(x)
    name = {1: "cfg1 ECP 64x128 Gaussian FWHM 5deg", 2: "cfg2 ECP 1024x2048 Gaussian FWHM 30'",
            3: "cfg3 HEALPix nside=512 Gaussian FWHM 10'",
            4: "cfg4 HEALPix nside=2048 (50.3 Mpix), Gaussian FWHM 5' cut at 15', white noise + 1000 point sources, 1 map",
            5: "cfg5 HEALPix nside=2048, 16 maps, Mexican hat s=4' cut at 20'"}[cfg]
    return c, tab, x, npix, nmaps, name


def oracle_sample_rings(R: int, nsample: int) -> np.ndarray:
    return np.unique(np.linspace(0, R - 1, nsample).round().astype(np.int32))


def time_oracle(c, tab, x, nsample_rings, nthreads=0):
    """The oracle as it stands (brute-force direct sum, fp64) on a sample of output rings."""
    from oracle import geometry, direct
    pix = c["pix"]
    geom = geometry.ecp(pix[1], pix[2]) if pix[0] == "ecp" else geometry.healpix_ring(pix[1])
    rings = oracle_sample_rings(geom.nrings, nsample_rings)
    xx = x.astype(np.float64)
    t0 = time.perf_counter()
    out, nthr = direct.direct_sum(geom, tab, c["theta_max"], xx, out_rings=rings, nthreads=nthreads, return_threads=True)
    dt = time.perf_counter() - t0
    npx = int(geom.n[rings].sum())
    return dict(seconds=dt, pixels=npx, maps=xx.shape[0], threads=nthr, rings=int(rings.size), nrings=geom.nrings)


class ClockSampler:
    """Samples SM clock and clock-event reasons of one GPU every few milliseconds (NVML, background thread) while the
    timed region runs; falls back to `nvidia-smi -lms` when NVML is not importable."""
    NAMES = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index: int, period_s: float = 0.004):
        import threading
        self.sm, self.reasons, self.max_mhz, self.err = [], set(), None, None
        self._stop = threading.Event()
        self._index, self._period = index, period_s
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def _run(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self._index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            while not self._stop.is_set():
                self.sm.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                mask = int(pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                for name, bit in self.NAMES.items():
                    if mask & bit:
                        self.reasons.add(name)
                time.sleep(self._period)
        except Exception as e:  # noqa: BLE001  (NVML missing or refused: report it, the bench still runs)
            self.err = repr(e)

    def stop(self) -> dict:
        self._stop.set()
        self._t.join()
        out = {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
               "reasons": sorted(self.reasons), "samples": len(self.sm)}
        if self.err:
            out["error"] = self.err
        return out


def run_reference(args):
    """--impl reference: the oracle on the host cores, rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    c, tab, x, npix, nmaps, name = workload(args.cfg)
    # size the per-step sample so that the whole run stays near two minutes on this host: calibrate on 32 rings
    cal = time_oracle(c, tab, x, 32)
    for _ in range(max(args.warmup - 1, 0)):
        time_oracle(c, tab, x, 4)
    per_ring = cal["seconds"] / max(cal["rings"], 1)
    nsample = int(min(args.oracle_rings, max(8, 120.0 / (per_ring * max(args.steps, 1)))))
    tot_t, tot_px, info = 0.0, 0, None
    for _ in range(args.steps):
        info = time_oracle(c, tab, x, nsample)
        tot_t += info["seconds"]
        tot_px += info["pixels"] * info["maps"]
    val = tot_px / tot_t / 1e6
    sample = (f"{info['rings']} of {info['nrings']} output rings, evenly spaced in ring index "
              f"({info['pixels']} output pixels x {info['maps']} map(s) per step)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": {"workload": name},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": info["threads"], "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1104_0672_b200 import arkcos

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c, tab, x, npix, nmaps, name = workload(args.cfg, args.cfg5_kernel)
    if world > 1:                       # every rank its own map(s): same shape, different seed
        mine = shard_range(nmaps * world, world, rank)
        x = np.stack([inputs.white_noise(npix, args.cfg, k) for k in mine])
    dtype = arkcos.F32
    t0 = time.perf_counter()
    plan = arkcos.Plan(c["pix"], tab, c["theta_max"], dtype, max_nmaps=nmaps)
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t0
    stats = plan.stats()
    d_in = torch.from_numpy(x).cuda()
    d_out = torch.empty_like(d_in)
    stream = torch.cuda.current_stream().cuda_stream

    def step():
        plan.convolve(d_in.data_ptr(), d_out.data_ptr(), nmaps, stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    if args.profile:                    # launches only (for ncu): no end-to-end leg, no CPU oracle, no JSON line
        for _ in range(args.steps):
            step()
        barrier()
        return
    if args.quick:                      # device-resident timing only: whole step, stages, band kernels one after the other
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            step()
        e1.record()
        barrier()
        out = {"ms_per_step": e0.elapsed_time(e1) / args.steps}
        plan.set_timing(2)
        acc, stage = None, {}
        for _ in range(args.steps):
            step()
            cur = [b[2] for b in plan.band_kernels(with_timing=True)]
            acc = cur if acc is None else [a + b for a, b in zip(acc, cur)]
            for k, v in plan.get_timing().items():
                stage[k] = stage.get(k, 0.0) + v / args.steps
        out["stage_ms_serial"] = stage
        out["band_ms"] = {b[0]: a / args.steps for b, a in zip(plan.band_kernels(), acc) if a > 0.5e-3 * args.steps}
        print(json.dumps(out))
        return
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    # same steps again with the library's per-stage events (the stream torch handed us is the launching stream)
    plan.set_timing(True)
    stage = {"rows": 0.0, "fft_forward": 0.0, "band": 0.0, "fft_inverse": 0.0}
    for _ in range(args.steps):
        step()
        for k, v in plan.get_timing().items():
            stage[k] += v / args.steps
    plan.set_timing(False)
    clocks = sampler.stop() if sampler else None
    t = torch.tensor([ms], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    ms_step = ms / args.steps
    value = world * npix * nmaps / (ms_step * 1e-3) / 1e6

    # end to end through the host-buffer entry point: pinned host -> device, convolve, device -> host, every step
    h_in = torch.from_numpy(x).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    plan.convolve_host(h_in.data_ptr(), h_out.data_ptr(), nmaps, stream)
    barrier()
    e0.record()
    for _ in range(args.steps):
        plan.convolve_host(h_in.data_ptr(), h_out.data_ptr(), nmaps, stream)
    e1.record()
    barrier()
    t = torch.tensor([e0.elapsed_time(e1)], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_sync_ms = float(t.item()) / args.steps
    # the streaming form of the same call (arkcos_convolve_host_async): every step still uploads its input and
    # downloads its result inside the timed region, but the upload of step k+1 and the download of step k-1 overlap
    # the kernels of step k (two staging sets in the plan)
    plan.convolve_host_async(h_in.data_ptr(), h_out.data_ptr(), nmaps)
    plan.synchronize()
    barrier()
    e0.record()
    for _ in range(args.steps):
        plan.convolve_host_async(h_in.data_ptr(), h_out.data_ptr(), nmaps)
    plan.synchronize()
    e1.record()
    barrier()
    t = torch.tensor([e0.elapsed_time(e1)], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_ms = float(t.item()) / args.steps
    e2e = {"value": world * npix * nmaps / (e2e_ms * 1e-3) / 1e6, "unit": UNIT, "ms_per_step": e2e_ms,
           "h2d_bytes_per_step": int(x.nbytes), "d2h_bytes_per_step": int(x.nbytes),
           "api": "arkcos_convolve_host_async x steps + arkcos_plan_synchronize (copies of neighbouring steps overlap)",
           "blocking_call_ms_per_step": e2e_sync_ms,
           "blocking_call_value": world * npix * nmaps / (e2e_sync_ms * 1e-3) / 1e6}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # per-kernel durations: the band kernels normally overlap on side streams; timing mode 2 runs them one after the
    # other with events in between (same launches, same stream torch handed us)
    plan.set_timing(2)
    band_ms = None
    for _ in range(args.steps):
        step()
        cur = [b[2] for b in plan.band_kernels(with_timing=True)]
        band_ms = cur if band_ms is None else [a + b for a, b in zip(band_ms, cur)]
    band_info = plan.band_kernels()
    plan.set_timing(False)
    band_ms = [v / args.steps for v in band_ms]

    # roofline of the dominant kernel (largest measured duration)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    fp32_peak = arkcos.arkcos_probe_fp32_peak(10)
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    alu_src = "FFMA chain measured in this run (arkcos_probe_fp32_peak); nominal 148*128*2*1.965 GHz = 74.4"
    kernels = []
    for (kname, flops, _), ms_k in zip(band_info, band_ms):
        if flops > 0:
            ach = flops * nmaps / (ms_k * 1e-3) / 1e12
            kernels.append({"kernel": kname, "ms": ms_k, "bound": "alu", "achieved": ach, "peak": fp32_peak,
                            "unit": "TFLOP/s", "frac": ach / fp32_peak, "traffic": TRAFFIC.get(kname), "peak_source": alu_src})
    for kname, key in (("ring_fft3_forward_kernel (all transform sizes)", "fft_forward"),
                       ("ring_fft3_inverse_kernel (all transform sizes)", "fft_inverse")):
        byts = 2.0 * 4.0 * npix * nmaps           # a ring FFT reads and writes every map element once (4 B each way)
        ach = byts / (stage[key] * 1e-3) / 1e9
        kernels.append({"kernel": kname, "ms": stage[key], "bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s",
                        "frac": ach / hbm, "traffic": TRAFFIC.get(kname), "peak_source": hbm_src})
    roof = dict(max(kernels, key=lambda k: k["ms"]))
    roof["stage_ms"] = stage
    roof["all_kernels"] = [{k: v for k, v in kk.items() if k != "peak_source"} for kk in kernels]
    launches_per_step = plan.launches_per_convolve

    # beside the headline (kernel rows regenerated every step, Table 1): the plan-cached mode for many maps
    # with one kernel, rows and their transforms computed once at plan time
    plan_c = arkcos.Plan(c["pix"], tab, c["theta_max"], dtype, max_nmaps=nmaps, cache_kernel_spectra=1)
    for _ in range(3):
        plan_c.convolve(d_in.data_ptr(), d_out.data_ptr(), nmaps, stream)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        plan_c.convolve(d_in.data_ptr(), d_out.data_ptr(), nmaps, stream)
    e1.record()
    torch.cuda.synchronize()
    cached_ms = e0.elapsed_time(e1) / args.steps
    cached = {"ms_per_step": cached_ms, "value": npix * nmaps / (cached_ms * 1e-3) / 1e6, "unit": UNIT,
              "workspace_gb": plan_c.stats()["workspace_bytes"] / 1e9, "note": "options.cache_kernel_spectra = 1; not the headline"}
    del plan_c

    cpu = time_oracle(c, tab, x, args.oracle_rings)
    cpu_val = cpu["pixels"] * cpu["maps"] / cpu["seconds"] / 1e6
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": name, "l2": "input map 201 MB + spectra 403 MB per step exceed the 126 MB L2; no flush",
                       "kernel_rows": "regenerated every step", "ell_nyquist": plan.ell_nyquist,
                       "plan_create_s": plan_s, "ring_pairs": stats["ring_pairs"], "row_samples": stats["row_samples"],
                       "model_gflop": {"band": stats["mac_flops"] / 1e9, "fft": stats["fft_flops"] / 1e9}},
            "roofline": roof,
            "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cpu["threads"], "kind": "oracle",
                             "sample": f"{cpu['rings']} of {cpu['nrings']} output rings evenly spaced in ring index, "
                                       f"{cpu['pixels']} pixels, {cpu['seconds']:.1f} s"},
            "cached_spectra_mode": cached, "e2e": e2e, "gpu_launches": launches_per_step * args.steps, "clocks": clocks,
            "paper_context": "2.2 s on a GTX 480 incl. PCIe copies = 22.9 Mpix/s (PAPER.md:195)"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=4)
    ap.add_argument("--profile", action="store_true", help="warm-up + steps of arkcos_convolve only (the command ncu wraps)")
    ap.add_argument("--cfg5-kernel", type=int, default=1, help="--cfg 5: 0 = top-hat disc, 1 = cut Mexican hat")
    ap.add_argument("--quick", action="store_true", help="device-resident timing of the step, its stages and band kernels only")
    ap.add_argument("--oracle-rings", type=int, default=2048, help="output rings in the CPU-oracle sample")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
