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


def ncu_table(which: str) -> dict:
    """Numbers taken from the ncu captures summarised under profiles/ (text files; absent -> empty):
    dram_bytes: kernel -> dram__bytes_read.sum + dram__bytes_write.sum per launch; fp32_thread_inst: step totals."""
    path = os.path.join(ROOT, "profiles", "r2_final_ncu.csv")
    out = {}
    try:
        import csv
        for row in csv.DictReader(open(path)):
            if which == "dram_bytes" and row.get("dram_bytes"):
                out[row["kernel"]] = float(row["dram_bytes"])
            if which == "fp32_thread_inst" and row["kernel"] == "STEP TOTAL" and row.get("fp32_gflop"):
                out["step_gflop"] = float(row["fp32_gflop"])
    except OSError:
        pass
    return out


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
    # a stream of our own (events and launches on the same, non-default stream; the library replays a CUDA graph there)
    torch.cuda.set_stream(torch.cuda.Stream())
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c, tab, x, npix, nmaps, name = workload(args.cfg, args.cfg5_kernel)
    if world > 1:                       # every rank its own map(s): same shape, different seed
        mine = shard_range(nmaps * world, world, rank)
        x = np.stack([inputs.white_noise(npix, args.cfg, k) for k in mine])
    dtype = arkcos.F32
    t0 = time.perf_counter()
    plan = arkcos.Plan(c["pix"], tab, c["theta_max"], dtype, max_nmaps=nmaps, exact_caps=int(args.exact_caps))
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
        plan.set_timing(1)
        ov = {}
        for _ in range(args.steps):
            step()
            for k, v in plan.get_timing().items():
                ov[k] = ov.get(k, 0.0) + v / args.steps
        out["stage_ms_overlapped"] = ov
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

    # per-launch durations: the band kernels and the ring-FFT launches normally overlap on side streams; timing mode 2
    # runs them one after the other with events in between (same launches, same stream torch handed us)
    plan.set_timing(2)
    band_ms, fwd_ms, inv_ms = None, None, None
    add = lambda acc, cur: cur if acc is None else [x + y for x, y in zip(acc, cur)]   # noqa: E731
    for _ in range(args.steps):
        step()
        band_ms = add(band_ms, [b[2] for b in plan.band_kernels(with_timing=True)])
        fk = plan.fft_kernels(with_timing=True)
        fwd_ms, inv_ms = add(fwd_ms, [f[2] for f in fk]), add(inv_ms, [f[3] for f in fk])
    band_info, fft_info = plan.band_kernels(), plan.fft_kernels()
    plan.set_timing(False)
    band_ms, fwd_ms, inv_ms = ([v / args.steps for v in lst] for lst in (band_ms, fwd_ms, inv_ms))

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    fp32_peak = arkcos.arkcos_probe_fp32_peak(10)
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    alu_src = ("FFMA chain measured in this run (arkcos_probe_fp32_peak); nominal 148*128*2*1.965 GHz = 74.4.  achieved = "
               "work-model flops of the kernel's rings (cosine transform of the rows + multiply-accumulate, DESIGN.md "
               "section 5) / duration; the tensor-core kernels run the cosine transform as 3xTF32 products, their FP32 pipe "
               "only the multiply-accumulate")
    tc = plan.tensor_cores()
    traffic = ncu_table("dram_bytes")
    plan_fft_bpt = 2 if c["pix"][-1] <= 4096 else 4      # blocks-per-transform template argument of the shared-memory FFT kernel
    kernels = []
    for (kname, flops, _), ms_k in zip(band_info, band_ms):
        if flops > 0 and ms_k > 0:
            ach = flops * nmaps / (ms_k * 1e-3) / 1e12
            launch = kname
            kernels.append({"kernel": launch, "ms": ms_k, "bound": "alu", "achieved": ach, "peak": fp32_peak,
                            "unit": "TFLOP/s", "frac": ach / fp32_peak, "traffic": traffic.get(launch), "peak_source": alu_src})
    for direction, mss in (("forward", fwd_ms), ("inverse", inv_ms)):
        for (kname, px, _, _), ms_k in zip(fft_info, mss):
            if px > 0 and ms_k > 0:
                byts = 2.0 * 4.0 * px * nmaps      # a ring FFT reads and writes every map element once (4 B each way)
                ach = byts / (ms_k * 1e-3) / 1e9
                # the launch's name as ncu prints it (profiles/r2_final_ncu.csv)
                q = kname[kname.index("<") + 1:kname.index(">")] if "<" in kname else ""
                if "direct1" in kname:
                    launch = f"ring_fft3_direct1_kernel<{q},{1 if direction == 'forward' else 0}>"
                elif "bluestein" in kname:
                    launch = f"ring_fft3_{direction}_kernel<{q}>"
                else:
                    launch = f"ring_fft_{direction}_kernel<float,{plan_fft_bpt}>"
                kernels.append({"kernel": launch, "ms": ms_k, "bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s",
                                "frac": ach / hbm, "traffic": traffic.get(launch), "peak_source": hbm_src})
    roof = dict(max(kernels, key=lambda k: k["ms"]))      # the longest single launch of the step
    roof["stage_ms"] = stage
    roof["all_kernels"] = [{k: v for k, v in kk.items() if k != "peak_source"} for kk in kernels]
    launches_per_step = plan.launches_per_convolve
    wm = plan.work_model()

    # whole-step fractions (SURVEY.md section 8d reporting rule): the work model as executed and as the method needs it
    t_s = ms_step * 1e-3
    gf_exec = (stats["mac_flops"] + stats["fft_flops"]) * nmaps / 1e9
    gf_alg = (stats["mac_flops"] + wm["fft_flops_min"]) * nmaps / 1e9
    inst = ncu_table("fp32_thread_inst")
    step_roof = {"model_gflop_executed": gf_exec, "model_gflop_algorithmic": gf_alg,
                 "frac_fp32_executed": gf_exec / t_s / 1e3 / fp32_peak, "frac_fp32_algorithmic": gf_alg / t_s / 1e3 / fp32_peak,
                 "tensor_gflop_issued": wm["tensor_flops"] * nmaps / 1e9,
                 "hbm_bytes_unfused": 6 * 4 * npix * nmaps, "frac_hbm_unfused": 6 * 4 * npix * nmaps / t_s / 1e9 / hbm,
                 "fp32_peak_tflops": fp32_peak, "hbm_peak_gbs": hbm,
                 "ncu_fp32_gflop_executed": inst.get("step_gflop"),
                 "note": "model_gflop_executed counts the Bluestein transforms as run and the rows' cosine transforms as FP32 "
                         "flops although the tensor-core kernels issue them as 3xTF32 products (tensor_gflop_issued, padded "
                         "tiles); ncu_fp32_gflop_executed = 2 FFMA + FMUL + FADD thread instructions of one step from "
                         "profiles/ (null until that capture exists)"}

    # beside the headline (kernel rows regenerated every step, Table 1): the plan-cached mode for many maps
    # with one kernel, rows and their transforms computed once at plan time
    def timed(p, n_maps, d_i, d_o, reps):
        for _ in range(2):
            p.convolve(d_i.data_ptr(), d_o.data_ptr(), n_maps, stream)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            p.convolve(d_i.data_ptr(), d_o.data_ptr(), n_maps, stream)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    plan_c = arkcos.Plan(c["pix"], tab, c["theta_max"], dtype, max_nmaps=nmaps, cache_kernel_spectra=1)
    cached_ms = timed(plan_c, nmaps, d_in, d_out, args.steps)
    cached = {"ms_per_step": cached_ms, "value": npix * nmaps / (cached_ms * 1e-3) / 1e6, "unit": UNIT,
              "workspace_gb": plan_c.stats()["workspace_bytes"] / 1e9, "note": "options.cache_kernel_spectra = 1; not the headline"}
    del plan_c

    # several kernels on one map (arkcos_convolve_multi): K Gaussians of different widths
    extra = {}
    if args.cfg == 4 and not args.no_extras:
        K = 8
        fw = [c["fwhm"] * (0.7 + 0.1 * k) for k in range(K)]
        plans = [arkcos.Plan(c["pix"], inputs.gaussian_table(f, 3.0 * f), 3.0 * f, dtype) for f in fw]
        d_multi = torch.empty((K, npix), device="cuda", dtype=torch.float32)
        run_multi = lambda: arkcos.arkcos_convolve_multi(plans, d_in.data_ptr(), d_multi.data_ptr(), 1, stream)   # noqa: E731
        run_sep = lambda: [p.convolve(d_in.data_ptr(), d_multi[k].data_ptr(), 1, stream) for k, p in enumerate(plans)]   # noqa: E731
        res = {}
        for label, fn in (("multi", run_multi), ("separate", run_sep)):
            fn()
            torch.cuda.synchronize()
            e0.record()
            for _ in range(5):
                fn()
            e1.record()
            torch.cuda.synchronize()
            res[label] = e0.elapsed_time(e1) / 5
        extra["multi_kernel"] = {"kernels": K, "workload": "cfg4 map, Gaussians FWHM 3.5' .. 7', cut at 3 FWHM",
                                 "ms_arkcos_convolve_multi": res["multi"], "ms_separate_calls": res["separate"]}
        del plans, d_multi
        torch.cuda.empty_cache()
        # config 5 (BASELINE.json configs[4]): 16 maps, hard-edged kernels; kernel spectra computed per call, cached, exact caps
        c5 = inputs.config(5)
        x5 = torch.from_numpy(inputs.white_noise_maps(npix, 5, c5["nmaps"])).cuda()
        o5 = torch.empty_like(x5)
        blk = {}
        for kspec in c5["kernels"]:
            tab5 = inputs.kernel_table(kspec)
            row = {}
            for mode, opts in (("computed", {}), ("cached_spectra", {"cache_kernel_spectra": 1}), ("computed_exact_caps", {"exact_caps": 1})):
                p5 = arkcos.Plan(c5["pix"], tab5, kspec["theta_max"], dtype, max_nmaps=c5["nmaps"], **opts)
                ms5 = timed(p5, c5["nmaps"], x5, o5, 3)
                row[mode] = {"ms_per_16_maps": ms5, "gpix_per_s": npix * c5["nmaps"] / (ms5 * 1e-3) / 1e9,
                             "workspace_gb": p5.stats()["workspace_bytes"] / 1e9, "tensor_cores": p5.tensor_cores()["used"]}
                del p5
                torch.cuda.empty_cache()
            blk[kspec["kernel"]] = row
        extra["cfg5"] = blk
        del x5, o5
        torch.cuda.empty_cache()
        # nside 4096 (the paper's next size; not a BASELINE.json config): rings of up to 16384 pixels
        ns = 4096
        np4 = 12 * ns * ns
        fw4, tm4 = 2.5 * inputs.ARCMIN, 7.5 * inputs.ARCMIN
        x4 = torch.randn(np4, dtype=torch.float32, device="cuda", generator=torch.Generator(device="cuda").manual_seed(4096))
        o4 = torch.empty_like(x4)
        p4 = arkcos.Plan(("healpix", ns), inputs.gaussian_table(fw4, tm4), tm4, dtype)
        ms4 = timed(p4, 1, x4, o4, 10)
        extra["nside4096"] = {"workload": "HEALPix nside=4096 (201 Mpix), Gaussian FWHM 2.5' cut at 7.5', 1 map",
                              "ms_per_map": ms4, "gpix_per_s": np4 / (ms4 * 1e-3) / 1e9}
        del p4, x4, o4

    cpu = time_oracle(c, tab, x, args.oracle_rings)
    cpu_val = cpu["pixels"] * cpu["maps"] / cpu["seconds"] / 1e6
    cpu1 = time_oracle(c, tab, x, max(16, args.oracle_rings // 32), nthreads=1)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": name, "l2": "input map 201 MB + spectra 403 MB per step exceed the 126 MB L2; no flush",
                       "kernel_rows": "regenerated every step", "ell_nyquist": plan.ell_nyquist,
                       "plan_create_s": plan_s, "ring_pairs": stats["ring_pairs"], "row_samples": stats["row_samples"],
                       "model_gflop": {"band": stats["mac_flops"] / 1e9, "fft": stats["fft_flops"] / 1e9,
                                       "fft_own_lengths": wm["fft_flops_min"] / 1e9},
                       "band_kernels": "tcgen05 3xTF32 row transform + FP32 multiply-accumulate" if tc["used"] else "FP32 only",
                       "tensor_core_blocks": tc["blocks"]},
            "roofline": roof, "step_roofline": step_roof,
            "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cpu["threads"], "kind": "oracle",
                             "sample": f"{cpu['rings']} of {cpu['nrings']} output rings evenly spaced in ring index, "
                                       f"{cpu['pixels']} pixels, {cpu['seconds']:.1f} s",
                             "one_thread": {"value": cpu1["pixels"] * cpu1["maps"] / cpu1["seconds"] / 1e6, "unit": UNIT,
                                            "sample": f"{cpu1['rings']} rings, {cpu1['pixels']} pixels, {cpu1['seconds']:.1f} s"}},
            "cached_spectra_mode": cached, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
            "gpu_launches_note": "kernels only; plus %d cudaMemsetAsync per step that clear the ranges the cap fold accumulates into"
                                 % (wm["memsets_per_map"] * nmaps),
            "clocks": clocks, "paper_context": "2.2 s on a GTX 480 incl. PCIe copies = 22.9 Mpix/s (PAPER.md:195)"}
    line.update(extra)
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
    ap.add_argument("--exact-caps", action="store_true", help="plan with options.exact_caps = 1 (with --profile / --quick: the direct-space kernel)")
    ap.add_argument("--no-extras", action="store_true", help="skip the multi-kernel and config-5 blocks")
    ap.add_argument("--quick", action="store_true", help="device-resident timing of the step, its stages and band kernels only")
    ap.add_argument("--oracle-rings", type=int, default=2048, help="output rings in the CPU-oracle sample")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
