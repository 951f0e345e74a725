"""Helpers shared by the tests that run the scheme oracle with a plan's settings."""
import numpy as np

from oracle import hybrid


def plan_mprime(plan, geom, theta_max, ell_nyquist=None):
    """The class-C grid lengths M'_i the plan chose (arkcos_plan_ring_info), checked against the bound of reading R10
    (oracle/hybrid.py mprime_resolving): never shorter than the resolving grid, even, and rounded up by less than 256."""
    mp = np.array([plan.ring_info(i)["mprime"] for i in range(geom.nrings)], dtype=np.int64)
    lo = hybrid.mprime_resolving(geom, theta_max, plan.ell_nyquist if ell_nyquist is None else ell_nyquist)
    assert np.all(mp >= lo) and np.all(mp % 2 == 0) and np.all(mp - lo < 256), (mp[:8], lo[:8])
    return mp
