"""The photon kernels under the bounds-checked build (libsoc_b200_checked.so, -DSOC_CHECKED): every index into a global or
shared array is tested against the array's length and violations are counted.  compute-sanitizer is closed on this GPU
pool ("runs under it have left GPUs needing a reset"), so this is the memcheck stand-in the pool's own message asks for:
bounds checks of our own, small cases, comparison with the CPU reference (the parity tests).  Runs in a subprocess so that
the product library of the other tests is not replaced."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r'''
import sys, numpy as np, torch
sys.path.insert(0, "%(root)s"); sys.path.insert(0, "%(root)s/tests")
from paper_1812_06632_b200 import inputs, soc
from gpu_common import gpu_packages
from helpers import random_octree
assert soc.checked_violations() == 0, "not the checked build"
REPLAY, PROD = soc.SOC_GEOM_FP64, soc.SOC_GEOM_FP32
def run(P, srcs, flags, kernel=0, n=None, seed=1):
    G = soc.Grid.from_problem(P)
    G.set_option("kernel", kernel)
    for f, src in srcs:
        gpu_packages(G, P, f, src, n or P.n_packages, seed, flags=flags, want_replay=True)
    G.close()
# config 1 (all three regular-grid kernels), ragged package counts
P = inputs.make_config("1", n_packages=30011)
for flags, k in ((REPLAY, 0), (PROD, 1), (PROD, 2)):
    run(P, [(0, P.sources(0))], flags, k)
# two point sources next to the boundary: hot-cell cube partly outside the grid; odd grid sizes (ghost bricks)
rho = np.ones(7 * 5 * 3, dtype=np.float32)
Q = inputs.Problem("adhoc", 7, 5, 3, np.array([105]), rho, None, np.array([1e14]), np.array([0.3]), np.array([0.6]), np.array([0.2]),
                   np.array([1.0]), np.zeros((0, 3)), np.zeros((1, 0)), 20000)
src = dict(bg_intensity=1.0, ps_pos=np.array([[0.5, 0.5, 0.5], [6.5, 4.5, 2.5]]), ps_lum=np.array([3.0, 1.0]))
for flags, k in ((REPLAY, 0), (PROD, 1), (PROD, 2)):
    run(Q, [(0, src)], flags, k, n=20001)
# random octree, 4 levels, with empty cells, point sources inside refined regions
n_cells, rho, child = random_octree((5, 4, 6), 4, 0.3, seed=2, p_empty=0.1)
R = inputs.Problem("adhoc", 5, 4, 6, np.asarray(n_cells, dtype=np.int64), rho, child, np.array([1e14]), np.array([0.4]), np.array([0.9]),
                   np.array([0.5]), np.array([1.0]), np.zeros((0, 3)), np.zeros((1, 0)), 30000)
src = dict(bg_intensity=2.0, ps_pos=np.array([[2.3, 1.7, 3.1], [0.5, 3.5, 5.5]]), ps_lum=np.array([30.0, 5.0]))
for flags in (REPLAY, PROD):
    run(R, [(0, src)], flags, n=30001, seed=9)
# spectrum with overlapped frequencies + temperatures + dust re-emission + iterate on a small octree
S = inputs.make_config("4p", n=8, n_packages=20000, n_freq=5)
S.kabs *= 200; S.ksca *= 200; S.t_scale /= 200; S.bg_intensity = S.bg_intensity * 300
G = soc.Grid.from_problem(S)
A = torch.zeros(S.n_total, dtype=torch.float64, device="cuda"); T = torch.zeros(S.n_total, dtype=torch.float32, device="cuda")
G.iterate([S.sources(f) for f in range(S.n_freq)], S.n_packages, 1, [20000, 30000], S.t_scale, S.table_T, S.e_min, S.e_max, A, T,
          mode="weighted", cap=500, reference_field=True, ali=True)
G.iterate([S.sources(f) for f in range(S.n_freq)], S.n_packages, 1, [20000], S.t_scale, S.table_T, S.e_min, S.e_max, A, T,
          mode="uniform", flags=REPLAY)
G.close()
C3 = inputs.make_config("3", n=12, n_packages=20000, n_freq=5)
C3.kabs *= 100; C3.ksca *= 100; C3.t_scale /= 100; C3.ps_lum = C3.ps_lum * 500
G = soc.Grid.from_problem(C3)
for k in (1, 2):
    G.set_option("kernel", k)
    A = torch.zeros(C3.n_total, dtype=torch.float64, device="cuda"); T = torch.zeros(C3.n_total, dtype=torch.float32, device="cuda")
    G.iterate([C3.sources(f) for f in range(C3.n_freq)], C3.n_packages, 1, [30000], C3.t_scale, C3.table_T, C3.e_min, C3.e_max, A, T,
              mode="weighted", cap=300, ali=True)
G.close()
# slab-blocked launches (queues, suspension, dump at the end of a phase), with and without the "stats" counters
C5 = inputs.make_config("5", n=20, n_packages=60000, n_freq=4)
G = soc.Grid.from_problem(C5)
G.set_option("kernel", 2)
for n_slabs, sweeps, stats in ((2, 0, 0), (5, 3, 0), (3, 1, 1)):
    G.set_option("slabs", n_slabs); G.set_option("slab_sweeps", sweeps); G.set_option("stats", stats)
    for f in range(C5.n_freq):
        gpu_packages(G, C5, f, C5.sources(f), C5.n_packages, 2, flags=PROD, want_replay=False)
G.close()
print("VIOLATIONS", soc.checked_violations(), "LAUNCHES", soc.launch_count())
'''


def test_no_out_of_range_index_in_the_photon_kernels():
    lib = os.path.join(ROOT, "paper_1812_06632_b200", "libsoc_b200_checked.so")
    if not os.path.exists(lib):
        from paper_1812_06632_b200 import build
        build.build(checked=True)
    env = dict(os.environ, SOC_B200_LIB=lib)
    out = subprocess.run([sys.executable, "-c", SCRIPT % dict(root=ROOT)], capture_output=True, text=True, timeout=1200, env=env)
    assert out.returncode == 0, out.stderr[-3000:]
    line = [ln for ln in out.stdout.splitlines() if ln.startswith("VIOLATIONS")][-1].split()
    assert int(line[1]) == 0, out.stdout[-2000:]
    assert int(line[3]) > 50
