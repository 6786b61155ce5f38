"""GPU parity of the surface-brightness map kernel (row f2) against the CPU oracle, through the C ABI."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from gpu_common import oracle_grid
from helpers import random_octree
from paper_1812_06632_b200 import inputs, soc


def _basis(theta, phi):
    d = -np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
    ex = np.array([-math.sin(phi), math.cos(phi), 0.0])
    ey = np.cross(d, ex)
    return ex, ey / np.linalg.norm(ey), d


def _gpu_map(G, f, T, ex, ey, d, centre, npx, npy, pixel):
    import torch
    out = torch.zeros(npx * npy, dtype=torch.float32, device="cuda")
    G.make_map(f, torch.from_numpy(np.ascontiguousarray(T, dtype=np.float32)).cuda(), ex, ey, d, centre, npx, npy, pixel, out)
    torch.cuda.synchronize()
    return out.cpu().numpy().reshape(npy, npx).astype(np.float64)


VIEWS = [(np.array([1.0, 0, 0]), np.array([0, 1.0, 0]), np.array([0, 0, 1.0])),       # the three cardinal directions
         (np.array([0, 1.0, 0]), np.array([0, 0, 1.0]), np.array([1.0, 0, 0])),
         (np.array([0, 0, 1.0]), np.array([1.0, 0, 0]), np.array([0, -1.0, 0])),
         _basis(0.8, 0.3), _basis(2.1, 4.0)]


@pytest.mark.parametrize("which", ["3", "4p"])
def test_map_matches_the_oracle(which):
    P = inputs.make_config(which, n=8, n_packages=10, n_freq=8)
    G = soc.Grid.from_problem(P)
    og = oracle_grid(P)
    rng = np.random.default_rng(3)
    T = rng.uniform(8, 80, P.n_total).astype(np.float32)
    T[rng.uniform(size=P.n_total) < 0.05] = 0.0
    centre = np.array([P.nx, P.ny, P.nz]) / 2
    pix = 1.0 / 2 ** (P.n_levels - 1)                                  # the size of the smallest cells
    npx = int(P.nx / pix) + 6
    for f in (0, 3, P.n_freq - 1):
        for ex, ey, d in VIEWS:
            mo = oracle.make_map(og, P.kabs[f], P.ksca[f], P.freq_hz[f], T, ex, ey, d, centre, npx, npx, pix)
            mg = _gpu_map(G, f, T, ex, ey, d, centre, npx, npx, pix)
            if mo.max() < 1e-30:                                       # cold dust at 0.1 um: below the fp32 range of the map
                assert (mg == 0).all()
                continue
            ok = np.abs(mg - mo) <= 2e-6 * mo + 1e-6 * mo.max() * (mo < 1e-30)
            # a line of sight that runs within rounding of a cell edge may take the two cells in the other order
            assert ok.mean() >= 0.999 and np.abs(mg - mo).sum() <= 1e-5 * mo.sum()
            assert ((mg == 0) | (mo > 0)).all()                        # nothing where the line of sight misses the cloud
    G.close()


def test_map_of_a_thick_uniform_cube_saturates_at_the_source_function():
    N = 10
    P = inputs.Problem("adhoc", N, N, N, np.array([N ** 3]), np.ones(N ** 3, dtype=np.float32), None, np.array([3e12]),
                       np.array([3.0]), np.array([1.0]), np.array([0.0]), np.array([0.0]), np.zeros((0, 3)), np.zeros((1, 0)), 1)
    G = soc.Grid.from_problem(P)
    T = np.full(N ** 3, 35.0, dtype=np.float32)
    m = _gpu_map(G, 0, T, *VIEWS[0], np.full(3, N / 2), N, N, 1.0)
    G.close()
    assert np.allclose(m, 0.75 * float(inputs.planck_nu(3e12, 35.0)), rtol=1e-6)


def test_full_size_map_of_the_octree_cloud(capsys):
    """Config 4' at full size, a 1310 x 1310 map per cardinal direction at 100 um; sampled pixels against the
    oracle, and the thin-limit column as a property of the whole map."""
    import time
    import torch
    P = inputs.make_config("4p")
    G = soc.Grid.from_problem(P)
    og = oracle_grid(P)
    rng = np.random.default_rng(5)
    T = rng.uniform(10, 25, P.n_total).astype(np.float32)
    f = int(np.argmin(np.abs(P.notes["lam_um"] - 100.0)))
    centre = np.array([32.0, 32.0, 32.0])
    npx, pix = 1310, 64.0 / 1310
    Td = torch.from_numpy(T).cuda()
    out = torch.zeros(npx * npx, dtype=torch.float32, device="cuda")
    times = []
    for ex, ey, d in VIEWS[:3]:
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        G.make_map(f, Td, ex, ey, d, centre, npx, npx, pix, out)
        torch.cuda.synchronize()
        times.append(time.perf_counter() - t0)
        m = out.cpu().numpy().reshape(npx, npx).astype(np.float64)
        assert (m > 0).all()
        # sampled pixels: 40 single-pixel oracle maps
        for (i, j) in rng.integers(0, npx, (40, 2)):
            c1 = centre + ((i + 0.5) - npx / 2) * pix * ex + ((j + 0.5) - npx / 2) * pix * ey
            mo = oracle.make_map(og, P.kabs[f], P.ksca[f], P.freq_hz[f], T, ex, ey, d, c1, 1, 1, pix)[0, 0]
            assert m[j, i] == pytest.approx(mo, rel=5e-6)
    G.close()
    with capsys.disabled():
        print(f"\n[map, config 4', 1310 x 1310, 100 um] {[f'{1e3 * t:.1f} ms' for t in times]} per direction")
