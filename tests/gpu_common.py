"""Shared helpers of the GPU parity tests: run the same seeded problem through the C ABI (CUDA) and
through the CPU oracle.  Imported only by tests."""
from __future__ import annotations

import os

import numpy as np

import oracle
from paper_1812_06632_b200 import soc

N_THREADS = max(1, min(16, os.cpu_count() or 1))


def oracle_grid(P):
    return oracle.Grid(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child)


def gpu_packages(G, P, ifreq, sources, n_packages, seed, weight=1.0, pkg_begin=0, pkg_count=None, flags=soc.SOC_GEOM_FP64,
                 want_replay=True, absorbed=None):
    """Returns (absorbed numpy, result dict, replay structured array or None)."""
    import torch
    if pkg_count is None:
        pkg_count = n_packages - pkg_begin
    A = torch.zeros(G.n_total, dtype=torch.float64, device="cuda") if absorbed is None else absorbed
    rep = torch.zeros(max(1, pkg_count) * soc.REPLAY_DTYPE.itemsize, dtype=torch.uint8, device="cuda") if want_replay else None
    res = G.simulate_packages(ifreq, sources, n_packages, seed, weight, pkg_begin, pkg_count, A, rep, flags=flags)
    torch.cuda.synchronize()
    rep_np = None
    if want_replay:
        rep_np = rep.cpu().numpy().view(soc.REPLAY_DTYPE)[:pkg_count]
    return A.cpu().numpy(), res.as_dict(), rep_np


def oracle_packages(og, P, ifreq, sources, n_packages, seed, weight=1.0, pkg_begin=0, pkg_count=None, want_replay=True,
                    threads=N_THREADS, f32state=False):
    """f32state=False: THE oracle (fp64 throughout) -- production-mode, closed-form and temperature comparisons.
    f32state=True: the named variant with the package state snapped to fp32 (oracle/soc_oracle.c header), pinned to
    the fp64 oracle by tests/test_oracle_pins.py -- package-by-package replay parity only."""
    A, res, rep, _ = oracle.simulate(og, P.kabs[ifreq], P.ksca[ifreq], P.g[ifreq], ifreq, sources, n_packages, seed, weight,
                                     pkg_begin, pkg_count, want_replay=want_replay, threads=threads, f32state=f32state)
    return A, res, rep


def replay_match(rep_gpu, rep_orc):
    """Fraction of packages whose (hash, steps, scatters) agree."""
    same = (rep_gpu["hash"] == rep_orc["hash"]) & (rep_gpu["steps"] == rep_orc["steps"]) & \
           (rep_gpu["scatters"] == rep_orc["scatters"])
    return float(same.mean()) if len(same) else 1.0


def rel_l1(a_gpu, a_orc):
    s = np.abs(a_orc).sum()
    return float(np.abs(a_gpu - a_orc).sum() / s) if s > 0 else float(np.abs(a_gpu).sum())
