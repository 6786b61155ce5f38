"""soc_update_temperatures_ali_static against soc_update_temperatures_ali (row f3).

Some host programs cannot let a library allocate GPU memory when they call it: they have given all of HBM to an allocator
of their own, or they run the update in a loop in which cudaMalloc's device-wide stall is not acceptable.  For them the
library offers one entry point whose work array is compiled into it (include/soc.h): no allocation, grids of at most
soc.STATIC_MAX_CELLS cells, one array per GPU that every call shares.

What is checked here: the temperatures equal those of the allocating call (same kernels, so to the last bit, and in any
case within the 0.01 K the other temperature tests use) on two calls in a row, the second on a smaller grid with another
table so that whatever the first call left in the array would show; the free device memory does not move across the
calls; and a grid beyond the limit is refused before anything is launched.

This file sorts last on purpose (pytest -x stops at the first failure, and the entry point is an extra, not part of the
hot path): it must pass alone in a fresh process as well as after every other test."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from helpers import random_octree
from paper_1812_06632_b200 import inputs, soc

T_TOL = 0.01        # K, north_star's temperature tolerance, as in test_gpu_dust.py / test_gpu_parity.py


def _octree_problem(root, n_levels, seed, n_freq):
    """A random octree (ragged n_total, empty leaves) with the dust tables and the temperature table of a shrunk config 3."""
    n_cells, rho, child = random_octree(root, n_levels, 0.4, seed=seed, p_empty=0.15)
    P0 = inputs.make_config("3", n=4, n_packages=1000, n_freq=n_freq)
    return inputs.Problem("adhoc", root[0], root[1], root[2], np.asarray(n_cells, dtype=np.int64), rho, child, P0.freq_hz,
                          P0.kabs, P0.ksca, P0.g, P0.bg_intensity, np.zeros((0, 3)), np.zeros((P0.n_freq, 0)), 1,
                          t_scale=P0.t_scale, table_T=P0.table_T, e_min=P0.e_min, e_max=P0.e_max)


def _case(torch, P, seed, table):
    """Device inputs of one ALI update: emitted from the library itself, self-absorbed and absorbed energies around it."""
    G = soc.Grid.from_problem(P)
    rng = np.random.default_rng(seed)
    T = rng.uniform(8.0, 90.0, P.n_total).astype(np.float32)
    Em = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
    G.cell_emission(torch.from_numpy(T).cuda(), Em)
    em = Em.cpu().numpy()
    S = em * rng.uniform(0.0, 0.9, P.n_total)
    A = S + em * rng.uniform(0.0, 2.0, P.n_total)
    A[rng.uniform(size=P.n_total) < 0.05] = 0.0                 # cells that were never hit
    return G, torch.from_numpy(A).cuda(), torch.from_numpy(S).cuda(), Em, np.ascontiguousarray(table, dtype=np.float32)


def test_static_scratch_entry_point_equals_the_allocating_one_twice_in_a_row():
    import torch
    P1 = _octree_problem((5, 5, 3), 3, seed=21, n_freq=10)
    P2 = _octree_problem((3, 3, 2), 2, seed=22, n_freq=10)
    assert P2.n_total < P1.n_total <= soc.STATIC_MAX_CELLS and P1.n_total % 4 != 0
    cases = [_case(torch, P1, 5, P1.table_T), _case(torch, P2, 6, P1.table_T[::3] * 1.5)]
    # the allocating path first: it is the expectation, and it has then loaded the two kernels both paths launch, so
    # that lazy loading of their code cannot show up as a change of free memory below
    expected = []
    for (G, A, S, Em, tab), P in zip(cases, (P1, P2)):
        T = torch.full((P.n_total,), -1.0, dtype=torch.float32, device="cuda")
        G.update_temperatures_ali(A, S, Em, P.t_scale, tab, P.e_min, P.e_max, T)
        expected.append(T.cpu().numpy())
    outs = [torch.full((P.n_total,), -1.0, dtype=torch.float32, device="cuda") for P in (P1, P2)]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (G, A, S, Em, tab), P, T in zip(cases, (P1, P2), outs):             # two calls in a row, nothing in between
        G.update_temperatures_ali_static(A, S, Em, P.t_scale, tab, P.e_min, P.e_max, T)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the entry point that must not allocate changed the free device memory"
    for T, want in zip(outs, expected):
        got = T.cpu().numpy()
        assert (want > 0).any() and np.abs(got - want).max() <= T_TOL
        assert np.array_equal(got, want)                                     # same kernels, same inputs
    # and once more on the first grid: the array now holds the second call's values
    G, A, S, Em, tab = cases[0]
    T = torch.full((P1.n_total,), -1.0, dtype=torch.float32, device="cuda")
    G.update_temperatures_ali_static(A, S, Em, P1.t_scale, tab, P1.e_min, P1.e_max, T)
    assert np.abs(T.cpu().numpy() - expected[0]).max() <= T_TOL
    for c in cases:
        c[0].close()


def test_static_scratch_entry_point_refuses_a_grid_beyond_its_limit():
    import torch
    n = (129, 128, 128)                                                      # 2 113 536 cells > 2 097 152
    P0 = inputs.make_config("3", n=4, n_packages=1000, n_freq=4)
    G = soc.Grid(n[0], n[1], n[2], [n[0] * n[1] * n[2]], np.ones(n[0] * n[1] * n[2], dtype=np.float32), None, P0.freq_hz,
                 P0.kabs, P0.ksca, P0.g)
    assert G.n_total > soc.STATIC_MAX_CELLS
    z = torch.zeros(G.n_total, dtype=torch.float64, device="cuda")
    T = torch.full((G.n_total,), -1.0, dtype=torch.float32, device="cuda")
    launches = soc.load().soc_launch_count()
    with pytest.raises(soc.SocError, match=r"2113536 cells.*2097152"):
        G.update_temperatures_ali_static(z, z, z, P0.t_scale, P0.table_T, P0.e_min, P0.e_max, T)
    assert soc.load().soc_launch_count() == launches and float(T.max()) == -1.0      # nothing ran, nothing written
    G.update_temperatures_ali(z, z, z, P0.t_scale, P0.table_T, P0.e_min, P0.e_max, T)   # the allocating call takes it
    assert float(T.min()) == pytest.approx(float(P0.table_T[0]))
    G.close()


def test_static_scratch_entry_point_at_its_limit():
    """A 128^3 regular grid has exactly STATIC_MAX_CELLS cells: the last element of the work array is used."""
    import torch
    n = 128
    P0 = inputs.make_config("3", n=4, n_packages=1000, n_freq=4)
    rng = np.random.default_rng(9)
    rho = rng.uniform(0.2, 3.0, n ** 3).astype(np.float32)
    G = soc.Grid(n, n, n, [n ** 3], rho, None, P0.freq_hz, P0.kabs, P0.ksca, P0.g)
    assert G.n_total == soc.STATIC_MAX_CELLS
    Em = torch.zeros(G.n_total, dtype=torch.float64, device="cuda")
    G.cell_emission(torch.from_numpy(rng.uniform(8.0, 90.0, G.n_total).astype(np.float32)).cuda(), Em)
    S = Em * torch.from_numpy(rng.uniform(0.0, 0.9, G.n_total)).cuda()
    A = S + Em * torch.from_numpy(rng.uniform(0.0, 2.0, G.n_total)).cuda()
    want = torch.full((G.n_total,), -1.0, dtype=torch.float32, device="cuda")
    got = torch.full((G.n_total,), -2.0, dtype=torch.float32, device="cuda")
    G.update_temperatures_ali(A, S, Em, P0.t_scale, P0.table_T, P0.e_min, P0.e_max, want)
    G.update_temperatures_ali_static(A, S, Em, P0.t_scale, P0.table_T, P0.e_min, P0.e_max, got)
    assert float(want.min()) > 0 and float(want.max()) > float(want.min())
    assert float((got - want).abs().max()) <= T_TOL and bool((got == want).all())
    G.close()
