"""Pins for the CPU oracle.  CPU only.

Every test compares the oracle with something that is not the oracle: published known answers,
closed forms, conservation laws, quadrature, or an independent geometric check.

`oracle.simulate` is THE oracle: fp64 throughout (north_star), pinned here at fp64 tolerances.
`oracle.simulate(..., f32state=True)` is the named variant whose package state is snapped to fp32 at every
store (oracle/soc_oracle.c header, "Precision"); the tests at the end of this file pin it to the fp64 oracle,
which is its only licence (F32 below = one fp32 ulp at 1).
"""
import math
import os

import numpy as np
import pytest

import oracle
from helpers import Geometry, fully_refined, random_octree

GOLD = os.path.join(os.path.dirname(__file__), "golden")
F32 = 2.0 ** -23      # one fp32 ulp at 1


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------------------ P1 RNG
def test_philox_known_answers():
    for r in _rows("philox_kat.txt"):
        w = [int(x, 16) for x in r]
        assert list(oracle.philox4x32_10(w[0:4], w[4:6])) == w[6:10]


def test_stream_layout_points():
    for r in _rows("stream_points.txt"):
        seed, ifreq, pkg, blk = (int(x) for x in r[:4])
        assert list(oracle.stream_block(seed, ifreq, pkg, blk)) == [int(x, 16) for x in r[4:8]]
    # each of (seed lo/hi, ifreq, package lo/hi, block) must reach the generator
    base = tuple(oracle.stream_block(1, 7, 12345, 0))
    for args in [(2, 7, 12345, 0), (1 + (1 << 32), 7, 12345, 0), (1, 8, 12345, 0), (1, 7, 12346, 0),
                 (1, 7, 12345 + (1 << 32), 0), (1, 7, 12345, 1)]:
        assert tuple(oracle.stream_block(*args)) != base


def test_uniform_conversion():
    # u = ((x >> 9) + 0.5) 2^-23: printed values of SURVEY 8c.11 P1, range, and exact in fp32
    w = [0x34263357, 0x8AA03099, 0x7D7A3C7A, 0xC08982B7]
    u = [oracle.uniform(x) for x in w]
    assert np.allclose(u, [0.203707874, 0.541506827, 0.490146458, 0.752098262], atol=5e-10, rtol=0)
    assert oracle.uniform(0) == 2.0 ** -24 and oracle.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert oracle.uniform(0x1FF) == oracle.uniform(0)          # low 9 bits are dropped
    for x in w + [0, 0xFFFFFFFF]:
        assert float(np.float32(oracle.uniform(x))) == oracle.uniform(x)
    us = np.array([oracle.uniform(v) for p in range(2000) for v in oracle.stream_block(3, 0, p, 0)])
    assert abs(us.mean() - 0.5) < 4 * (1 / 12) ** 0.5 / len(us) ** 0.5
    assert abs(us.var() - 1 / 12) < 0.004


# ------------------------------------------------------------------------------ P6 scattering
@pytest.mark.parametrize("g", [0.6, -0.3, 0.95, 0.01, 1e-4])
def test_hg_matches_textbook_inverse_cdf(g):
    u = (np.arange(2000) + 0.5) / 2000
    ours = np.array([oracle.hg_cos(g, x) for x in u])
    book = (1 + g * g - ((1 - g * g) / (1 - g + 2 * g * u)) ** 2) / (2 * g)
    assert np.abs(ours - book).max() < (1e-9 if g > 1e-3 else 1e-6)   # the textbook form itself loses digits as g -> 0


@pytest.mark.parametrize("g", [0.0, 0.3, 0.6, -0.5])
def test_hg_moments_and_limits(g):
    u = (np.arange(200000) + 0.5) / 200000          # midpoint rule over the CDF variable
    c = np.array([oracle.hg_cos(g, x) for x in u[::20]])
    assert abs(c.mean() - g) < 2e-4
    assert abs((c * c).mean() - (1 + 2 * g * g) / 3) < 2e-4
    assert abs(oracle.hg_cos(g, 1e-12) + 1) < 1e-9 and abs(oracle.hg_cos(g, 1 - 1e-12) - 1) < 1e-9
    if g == 0.0:
        assert oracle.hg_cos(0.0, 0.3) == pytest.approx(2 * 0.3 - 1, abs=1e-16)


def test_rotation_is_a_rotation():
    rng = np.random.default_rng(0)
    dirs = list(rng.standard_normal((50, 3))) + [np.array(v, float) for v in
                                                  [(0, 0, 1), (0, 0, -1), (1, 0, 0), (0, -1, 0), (1e-9, 0, -1)]]
    for d in dirs:
        d = d / np.linalg.norm(d)
        cost, phi = rng.uniform(-1, 1), rng.uniform(0, 2 * np.pi)
        n = oracle.rotate(d, cost, phi)
        assert abs(np.linalg.norm(n) - 1) < 1e-14
        assert abs(n @ d - cost) < 1e-12
    # the azimuth really goes around d: four quarter turns at cos = 0 are mutually orthogonal / opposite
    d = np.array([0.3, -0.5, 0.8]); d /= np.linalg.norm(d)
    q = [oracle.rotate(d, 0.0, k * np.pi / 2) for k in range(4)]
    assert abs(q[0] @ q[1]) < 1e-12 and abs(q[0] @ q[2] + 1) < 1e-12 and abs(q[1] @ q[3] + 1) < 1e-12
    assert np.linalg.det(np.stack([q[0], q[1], d])) == pytest.approx(1.0, abs=1e-12)   # right-handed


# ------------------------------------------------------------------------------ P2 slab
def _uniform_grid(shape, rho=1.0):
    nx, ny, nz = shape
    return oracle.Grid(nx, ny, nz, [nx * ny * nz], np.full(nx * ny * nz, rho, dtype=np.float32))


@pytest.mark.parametrize("axis,sign", [(0, 1), (0, -1), (1, 1), (1, -1), (2, 1), (2, -1)])
def test_beam_through_pure_absorber(axis, sign):
    shape = (7, 5, 9)
    n = shape[axis]
    g = _uniform_grid(shape, rho=2.0)
    kabs = 0.15
    tau_c = kabs * 2.0
    pos = np.array([3.25, 2.5, 4.75]); pos[axis] = 0.0 if sign > 0 else n
    d = np.zeros(3); d[axis] = sign
    A, res, rep, _ = oracle.simulate(g, kabs, 0.0, 0.0, 0, dict(beam=np.concatenate([pos, d])), 1, 1, want_replay=True)
    A3 = A.reshape(shape[2], shape[1], shape[0])
    idx = [int(pos[0]), int(pos[1]), int(pos[2])]
    line = []
    for i in (range(n) if sign > 0 else range(n - 1, -1, -1)):
        idx[axis] = i
        line.append(A3[idx[2], idx[1], idx[0]])
    expect = np.exp(-tau_c * np.arange(n)) * (1 - np.exp(-tau_c))
    assert np.allclose(line, expect, rtol=1e-13, atol=0)
    assert res.escaped == pytest.approx(math.exp(-n * tau_c), rel=1e-13)        # transmission = exp(-tau)
    assert A.sum() == pytest.approx(sum(line), rel=1e-14)                       # nothing deposited elsewhere
    assert rep["steps"][0] == n and res.scatterings == 0


def test_oblique_beam_path_length():
    # absorbed = 1 - exp(-kappa rho L) with L the geometric chord of the box; visits the right cells
    shape = (6, 4, 5)
    g = _uniform_grid(shape, 1.5)
    d = np.array([0.6, 0.3, -0.5]); d /= np.linalg.norm(d)
    pos = np.array([0.0, 1.2, 4.4])
    A, res, _, tr = oracle.simulate(g, 0.2, 0.0, 0.0, 0, dict(beam=np.concatenate([pos, d])), 1, 1, trace_cap=100)
    tmax = min(((shape[j] if d[j] > 0 else 0) - pos[j]) / d[j] for j in range(3))
    assert res.absorbed == pytest.approx(1 - math.exp(-0.2 * 1.5 * tmax), rel=1e-13)
    assert tr["ds"].sum() == pytest.approx(tmax, rel=1e-13)
    for s in tr:   # each visited cell is the cell of the segment mid-point
        mid = 0.5 * (s["p0"] + s["p1"])
        ijk = np.floor(mid).astype(int)
        assert s["gid"] == ijk[0] + shape[0] * (ijk[1] + shape[1] * ijk[2])


# ------------------------------------------------------------------------------ P4 conservation
@pytest.mark.parametrize("hier", [False, True])
def test_energy_conservation(hier):
    if hier:
        n_cells, rho, child = random_octree((5, 4, 6), 4, 0.3, seed=11, p_empty=0.1)
        g = oracle.Grid(5, 4, 6, n_cells, rho, child)
        pos = np.array([[2.3, 1.7, 3.1], [0.5, 3.5, 5.5]])
    else:
        rng = np.random.default_rng(5)
        g = oracle.Grid(8, 8, 8, [512], rng.lognormal(0, 1, 512).astype(np.float32))
        pos = np.array([[4.5, 4.5, 4.5], [1.5, 6.5, 2.5]])
    src = dict(bg_intensity=2.0, ps_pos=pos, ps_lum=np.array([30.0, 5.0]))
    A, res, rep, _ = oracle.simulate(g, 0.4, 0.9, 0.5, 3, src, 20001, 9, weight=0.25, want_replay=True)  # odd: uneven split over the 2 sources
    assert abs(res.emitted - res.absorbed - res.escaped) <= 1e-9 * res.emitted
    assert A.sum() == pytest.approx(0.25 * res.absorbed, rel=1e-12)             # weight multiplies the deposit
    assert rep["e_escaped"].sum() == pytest.approx(res.escaped, rel=1e-12)
    surf = 2 * (g.ny * g.nz + g.nz * g.nx + g.nx * g.ny)
    assert res.emitted == pytest.approx(math.pi * 2.0 * surf + 35.0, rel=1e-12)  # pi I S + sum L
    if hier:
        assert (A[g.child >= 0] == 0).all()                                     # parents hold no dust
        assert (A[g.rho == 0] == 0).all()


def test_subset_replay_equals_full_run():
    g = _uniform_grid((6, 6, 6))
    src = dict(bg_intensity=1.0, ps_pos=np.array([[3.5, 3.5, 3.5]]), ps_lum=np.array([10.0]))
    A, res, rep, _ = oracle.simulate(g, 0.1, 0.5, 0.3, 0, src, 3000, 4, want_replay=True)
    A2 = np.zeros_like(A)
    reps = []
    for b, n in [(0, 1000), (1000, 1499), (2499, 501)]:
        _, _, r, _ = oracle.simulate(g, 0.1, 0.5, 0.3, 0, src, 3000, 4, pkg_begin=b, pkg_count=n, absorbed=A2,
                                     want_replay=True)
        reps.append(r)
    assert np.array_equal(np.concatenate(reps), rep)
    assert np.allclose(A2, A, rtol=1e-12, atol=0)
    A3, res3, rep3, _ = oracle.simulate(g, 0.1, 0.5, 0.3, 0, src, 3000, 4, want_replay=True, threads=3)
    assert np.array_equal(rep3, rep) and np.allclose(A3, A, rtol=1e-12, atol=0)
    assert res3.cell_steps == res.cell_steps


# ------------------------------------------------------------------------------ P3 optically thin bath
@pytest.mark.parametrize("hier", [False, True])
def test_optically_thin_bath(hier):
    """Isotropic bath I: A_c = 4 pi I kabs rho_c V_c for ANY scattering opacity, g and density structure
    (mean-chord-length invariance), as long as tau_abs << 1."""
    I, kabs, ksca, gg, n = 1.7, 1e-6, 0.6, 0.6, 150000
    if hier:
        n_cells, rho, child = random_octree((5, 5, 5), 3, 0.25, seed=3)
        g = oracle.Grid(5, 5, 5, n_cells, rho, child)
        geo = Geometry((5, 5, 5), n_cells, child)
        gid, level, _, h = geo.leaf_boxes()
        vol = np.zeros(g.n_total); vol[gid] = h ** 3
    else:
        rng = np.random.default_rng(2)
        g = oracle.Grid(6, 6, 6, [216], rng.lognormal(0, 1, 216).astype(np.float32))
        vol = np.ones(216)
    A, res, _, _ = oracle.simulate(g, kabs, ksca, gg, 0, dict(bg_intensity=I), n, 21, threads=4)
    expect = 4 * math.pi * I * kabs * g.rho.astype(np.float64) * vol
    assert res.scatterings / n > 1.0                                   # the invariance is really exercised
    assert A.sum() / expect.sum() == pytest.approx(1.0, abs=0.006)
    order = np.argsort(g.rho)
    leaves = order[vol[order] > 0]
    for q in np.array_split(leaves, 4):                                # flat across density quartiles
        assert A[q].sum() / expect[q].sum() == pytest.approx(1.0, abs=0.015)
    if hier:                                                           # and across hierarchy levels
        for lv in np.unique(level):
            sel = gid[level == lv]
            assert A[sel].sum() / expect[sel].sum() == pytest.approx(1.0, abs=0.02)
    # absorbed is proportional to tau in the thin limit
    A2, _, _, _ = oracle.simulate(g, 2 * kabs, ksca, gg, 0, dict(bg_intensity=I), n, 21, threads=4)
    assert A2.sum() / A.sum() == pytest.approx(2.0, rel=1e-4)


# ------------------------------------------------------------------------------ P5 point source
def test_point_source_in_uniform_absorber():
    N, kr = 21, 0.1
    g = _uniform_grid((N, N, N), 1.0)
    n = 200000
    src = dict(ps_pos=np.array([[N / 2, N / 2, N / 2]]), ps_lum=np.array([1.0]))
    A, res, _, _ = oracle.simulate(g, kr, 0.0, 0.0, 0, src, n, 2, threads=4)
    # escape fraction = < exp(-kr d(Omega)) > with d the distance from the centre to the cube surface
    mu = (np.arange(2000) + 0.5) / 2000 * 2 - 1
    ph = (np.arange(4000) + 0.5) / 4000 * 2 * np.pi
    st = np.sqrt(1 - mu ** 2)[:, None]
    comp = np.stack([st * np.cos(ph)[None, :], st * np.sin(ph)[None, :], np.broadcast_to(mu[:, None], (2000, 4000))])
    dist = (N / 2) / np.abs(comp).max(axis=0)
    w = np.exp(-kr * dist)
    assert res.escaped == pytest.approx(w.mean(), abs=5 * w.std() / n ** 0.5)
    # energy absorbed between radii r1 < r2 (inside the cube) = exp(-kr r1) - exp(-kr r2): test with cells whose
    # 8 corners all lie within / outside the shell -> bracket
    c = np.arange(N) + 0.5 - N / 2
    zz, yy, xx = np.meshgrid(c, c, c, indexing="ij")
    rmin = np.sqrt(np.maximum(np.abs(xx) - 0.5, 0) ** 2 + np.maximum(np.abs(yy) - 0.5, 0) ** 2 + np.maximum(np.abs(zz) - 0.5, 0) ** 2)
    rmax = np.sqrt((np.abs(xx) + 0.5) ** 2 + (np.abs(yy) + 0.5) ** 2 + (np.abs(zz) + 0.5) ** 2)
    A3 = A.reshape(N, N, N)
    for R in (4.0, 8.0):
        inner = A3[rmax <= R].sum()        # cells fully inside radius R
        outer = A3[rmin < R].sum()         # cells touching radius R
        exact = 1 - math.exp(-kr * R)
        assert inner <= exact * 1.002 and outer >= exact * 0.998
    assert res.cell_steps / n > N / 2      # every package crosses at least half the grid


def test_point_source_in_empty_cell():
    # the source sits in a zero-density cell -- legal, nothing absorbed there
    rho = np.ones(125, dtype=np.float32); rho[62] = 0.0
    g = oracle.Grid(5, 5, 5, [125], rho)
    A, res, _, _ = oracle.simulate(g, 0.3, 0.2, 0.0, 0, dict(ps_pos=np.array([[2.5, 2.5, 2.5]]), ps_lum=np.array([1.0])),
                                   5000, 1)
    assert A[62] == 0.0 and res.absorbed > 0 and abs(res.emitted - res.absorbed - res.escaped) < 1e-12


# ------------------------------------------------------------------------------ P7 emission laws
def test_background_emission_laws():
    nx, ny, nz = 3, 5, 8
    rng = np.random.default_rng(1)
    n = 60000
    U = rng.random((n, 5))
    faces = np.zeros(6)
    mus = []
    for u in U:
        ijk, f, d = oracle.emit_background(nx, ny, nz, u)
        assert abs(np.linalg.norm(d) - 1) < 1e-14
        assert (0 <= ijk).all() and (ijk < (nx, ny, nz)).all() and (f >= 0).all() and (f <= 1).all()
        on = [a for a in range(3) if (f[a] == 0.0 and ijk[a] == 0 and d[a] > 0) or
              (f[a] == 1.0 and ijk[a] == (nx, ny, nz)[a] - 1 and d[a] < 0)]
        assert len(on) >= 1
        a = on[0]
        faces[2 * a + (1 if d[a] < 0 else 0)] += 1
        mus.append(abs(d[a]))
    area = np.array([ny * nz, ny * nz, nz * nx, nz * nx, nx * ny, nx * ny], float)
    p = area / area.sum()
    assert np.all(np.abs(faces / n - p) < 5 * np.sqrt(p * (1 - p) / n))     # faces in proportion to area
    assert np.mean(mus) == pytest.approx(2 / 3, abs=5 * (1 / 18) ** 0.5 / n ** 0.5)   # cosine law
    assert np.mean(np.square(mus)) == pytest.approx(0.5, abs=0.006)
    # entry points uniform over a face: mean tangential coordinate of x- face hits
    ijk, f, d = oracle.emit_background(nx, ny, nz, [0.0, 0.75, 0.5, 0.25, 0.125])
    assert list(ijk) == [0, 3, 4] and np.allclose(f, [0, 0.75, 0.0]) and d[0] == pytest.approx(0.5)
    assert d[1] == pytest.approx(math.sqrt(0.75) * math.cos(math.pi / 4)) and d[2] == pytest.approx(math.sqrt(0.75) * math.sin(math.pi / 4))


def test_point_emission_is_isotropic():
    rng = np.random.default_rng(4)
    D = np.array([oracle.emit_point([1.25, 2.5, 0.75], u)[2] for u in rng.random((40000, 2))])
    assert np.allclose(np.linalg.norm(D, axis=1), 1, atol=1e-14)
    assert np.all(np.abs(D.mean(axis=0)) < 5 * (1 / 3) ** 0.5 / 200)
    assert np.allclose((D[:, :, None] * D[:, None, :]).mean(axis=0), np.eye(3) / 3, atol=0.01)
    ijk, f, _ = oracle.emit_point([1.25, 2.5, 0.75], [0.5, 0.5])
    assert list(ijk) == [1, 2, 0] and np.allclose(f, [0.25, 0.5, 0.75])


@pytest.mark.parametrize("hier", [False, True])
def test_mean_cells_crossed_in_empty_grid(hier):
    """Flux argument: a package of an isotropic field crosses on average 1 + 2 A_int / S cells of an EMPTY
    grid, A_int = total interior leaf-interface area (= N for a cubic regular grid)."""
    shape = (4, 6, 5)
    if hier:
        n_cells, rho, child = random_octree(shape, 3, 0.3, seed=8)
    else:
        n_cells, rho, child = np.array([120]), np.zeros(120, np.float32), None
    g = oracle.Grid(*shape, n_cells, np.zeros_like(rho), child)
    a_int = Geometry(shape, n_cells, child).interior_interface_area()
    S = 2 * (shape[1] * shape[2] + shape[2] * shape[0] + shape[0] * shape[1])
    if not hier:
        assert a_int == 3 * 4 * 6 * 5 - (6 * 5 + 4 * 5 + 4 * 6)
    n = 120000
    _, res, rep, _ = oracle.simulate(g, 1.0, 1.0, 0.0, 0, dict(bg_intensity=1.0), n, 17, want_replay=True, threads=4)
    sd = rep["steps"].std() / n ** 0.5
    assert res.cell_steps / n == pytest.approx(1 + 2 * a_int / S, abs=5 * sd)
    assert res.escaped == pytest.approx(res.emitted, rel=1e-12) and res.scatterings == 0


# ------------------------------------------------------------------------------ P8 geometric replay
@pytest.mark.parametrize("seed", [1, 2])
def test_bruteforce_geometric_replay_on_tiny_octree(seed):
    shape = (3, 4, 3)
    n_cells, rho, child = random_octree(shape, 4, 0.35, seed=seed, p_empty=0.15)
    g = oracle.Grid(*shape, n_cells, rho, child)
    geo = Geometry(shape, n_cells, child)
    kabs, ksca = 0.3, 1.1
    src = dict(bg_intensity=1.0, ps_pos=np.array([[1.3, 2.2, 0.7]]), ps_lum=np.array([5.0]))
    n = 1500
    A, res, rep, tr = oracle.simulate(g, kabs, ksca, 0.4, 1, src, n, seed, want_replay=True, trace_cap=400000)
    assert len(tr) == res.cell_steps
    A_chk = np.zeros_like(A)
    k = 0
    for p in range(n):
        steps = tr[k:k + rep["steps"][p]]
        k += len(steps)
        assert (steps["pkg"] == p).all()
        tau_acc = 0.0
        for i, s in enumerate(steps):
            seglen = np.linalg.norm(s["p1"] - s["p0"])
            assert seglen == pytest.approx(s["ds"], abs=1e-12)
            if i > 0:                                    # contiguous path
                assert np.allclose(steps[i - 1]["p1"], s["p0"], atol=1e-12)
            if seglen > 1e-9:                            # the mid-point lies in the leaf that was charged
                gid, level, org, h = geo.locate(*(0.5 * (s["p0"] + s["p1"])))
                assert gid == s["gid"] and level == s["level"]
                assert (np.minimum(s["p0"], s["p1"]) >= org - 1e-12).all() and (np.maximum(s["p0"], s["p1"]) <= org + h + 1e-12).all()
            assert geo.is_leaf(s["gid"])
            assert s["tau_sca"] == pytest.approx(s["ds"] * float(rho[s["gid"]]) * ksca, rel=1e-12, abs=1e-300)
            tau_acc += s["tau_sca"]
            if s["kind"] == 1:                           # free path really has the drawn optical depth
                assert tau_acc == pytest.approx(s["tau_drawn"], rel=1e-9)
                tau_acc = 0.0
            else:
                assert tau_acc < s["tau_drawn"] * (1 + 1e-12)
        last = steps[-1]
        assert last["kind"] in (2, 3)
        if last["kind"] == 3:                            # escaped: ends on the outer boundary
            on = [abs(last["p1"][j]) < 1e-12 or abs(last["p1"][j] - shape[j]) < 1e-12 for j in range(3)]
            assert any(on)
    # the absorbed energy is what the recorded path lengths imply (weights follow from the packages' E0)
    n_bg = n // 2
    S = 2 * (shape[1] * shape[2] + shape[2] * shape[0] + shape[0] * shape[1])
    k = 0
    for p in range(n):
        E = math.pi * 1.0 * S / n_bg if p < n_bg else 5.0 / (n - n_bg)
        for s in tr[k:k + rep["steps"][p]]:
            dep = E * -math.expm1(-s["ds"] * float(rho[s["gid"]]) * kabs)
            A_chk[s["gid"]] += dep
            E -= dep
        k += rep["steps"][p]
    assert np.allclose(A, A_chk, rtol=1e-10, atol=1e-14)


# ------------------------------------------------------------------------------ P9 hierarchy == regular
def test_fully_refined_hierarchy_equals_regular_grid():
    N = 6
    rng = np.random.default_rng(7)
    rho2n = rng.lognormal(0, 0.8, (2 * N, 2 * N, 2 * N)).astype(np.float32)
    n_cells, rho, child, gid_of = fully_refined(rho2n)
    gh = oracle.Grid(N, N, N, n_cells, rho, child)
    gr = oracle.Grid(2 * N, 2 * N, 2 * N, [8 * N ** 3], rho2n.ravel())
    n, kabs, ksca, gg, I = 20000, 0.35, 0.8, 0.45, 3.0
    # the regular grid's length unit is half a root cell: kappa halves, and I/4 keeps the package energy
    Ah, rh, reph, _ = oracle.simulate(gh, kabs, ksca, gg, 2, dict(bg_intensity=I), n, 5, want_replay=True)
    Ar, rr, repr_, _ = oracle.simulate(gr, kabs / 2, ksca / 2, gg, 2, dict(bg_intensity=I / 4), n, 5, want_replay=True)
    same = (reph["steps"] == repr_["steps"]) & (reph["scatters"] == repr_["scatters"])
    assert same.mean() >= 0.9999
    assert rh.emitted == pytest.approx(rr.emitted, rel=1e-13)
    assert rh.escaped == pytest.approx(rr.escaped, rel=1e-9)
    assert np.allclose(Ah[gid_of.ravel()], Ar, rtol=1e-9, atol=1e-12 * Ar.max())
    assert Ah[: N ** 3].sum() == 0.0


# ------------------------------------------------------------------------------ P10 noise law
def test_noise_scales_as_inverse_sqrt_n():
    g = _uniform_grid((6, 6, 6))
    src = dict(bg_intensity=1.0)

    def rms(n):
        a = [oracle.simulate(g, 0.05, 0.3, 0.2, 0, src, n, s)[0] for s in (1, 2)]
        return np.sqrt(np.mean((a[0] - a[1]) ** 2))
    r1, r2 = rms(4000), rms(64000)
    assert r1 / r2 == pytest.approx(4.0, rel=0.25)       # PAPER.md:125 noise ~ N^-1/2


# ------------------------------------------------------------------------------ a10, a11
def test_trapezoid_weights():
    rng = np.random.default_rng(0)
    nu = np.sort(rng.uniform(1, 10, 17))
    y = rng.random(17)
    w = oracle.trapezoid_weights(nu)
    assert (w * y).sum() == pytest.approx(np.trapezoid(y, nu), rel=1e-13)
    assert oracle.trapezoid_weights([5.0])[0] == 1.0


def test_temperature_lookup_semantics():
    n_cells, rho, child = random_octree((3, 3, 3), 3, 0.4, seed=5, p_empty=0.2)
    g = oracle.Grid(3, 3, 3, n_cells, rho, child)
    n_t, e_min, e_max = 64, 1e-3, 1e5
    beta = 2.0
    table = (10.0 * (np.geomspace(e_min, e_max, n_t) / 1.0) ** (1 / (4 + beta))).astype(np.float32)
    rng = np.random.default_rng(1)
    A = 10 ** rng.uniform(-6, 7, g.n_total)
    A[::7] = 0.0
    T = oracle.update_temperatures(g, A, 2.5, table, e_min, e_max)
    geo = Geometry((3, 3, 3), n_cells, child)
    gid, level, _, h = geo.leaf_boxes()
    vol = np.zeros(g.n_total); vol[gid] = h ** 3
    for i in range(g.n_total):
        if child[i] >= 0 or rho[i] == 0:
            assert T[i] == 0.0
            continue
        e = 2.5 * A[i] / (float(rho[i]) * vol[i])
        if e <= e_min:
            assert T[i] == table[0]                       # also the unhit cells
        elif e >= e_max:
            assert T[i] == table[-1]
        else:                                             # power law table: T = 10 E^(1/6) up to interpolation error
            assert T[i] == pytest.approx(10.0 * e ** (1 / 6), rel=2e-3)
            x = math.log(e / e_min) / math.log(e_max / e_min) * (n_t - 1)
            k = int(x)
            assert T[i] == pytest.approx(table[k] + (x - k) * (float(table[k + 1]) - float(table[k])), rel=1e-6)


def test_grid_validation_rejects_bad_hierarchies():
    ok = random_octree((2, 2, 2), 2, 0.5, seed=1)
    oracle.Grid(2, 2, 2, *ok)
    n_cells, rho, child = (a.copy() for a in ok)
    bad = child.copy(); bad[np.argmax(child >= 0)] += 4                # not a multiple of 8
    with pytest.raises(ValueError):
        oracle.Grid(2, 2, 2, n_cells, rho, bad)
    bad = child.copy(); i = np.where(child >= 0)[0]
    if len(i) >= 2:
        bad[i[1]] = bad[i[0]]                                         # two parents for one octet
        with pytest.raises(ValueError):
            oracle.Grid(2, 2, 2, n_cells, rho, bad)
    r = rho.copy(); r[np.argmax(child < 0)] = -1.0
    with pytest.raises(ValueError):
        oracle.Grid(2, 2, 2, n_cells, r, child)


# ------------------------------------------------------------------------------ extra pins (mutation survivors)
def test_termination_deposits_the_residual():
    # optically very thick absorber: weights fall below 1e-9 E0, the residual stays in the cell (reading S7)
    g = _uniform_grid((4, 4, 4), 1.0)
    A, res, _, _ = oracle.simulate(g, 30.0, 5.0, 0.0, 0, dict(bg_intensity=1.0), 2000, 3)
    assert res.terminated > 1000
    assert A.sum() == pytest.approx(res.emitted - res.escaped, rel=1e-12)
    assert abs(res.emitted - res.absorbed - res.escaped) <= 1e-12 * res.emitted


def test_lowest_axis_wins_an_exact_tie():
    # d_x = d_y exactly and the beam starts on the x = y diagonal: every x/y crossing is an exact tie
    g = _uniform_grid((4, 4, 4), 1.0)
    d = np.array([0.625, 0.625, 0.0]); d[2] = math.sqrt(1 - 2 * 0.625 ** 2)
    beam = np.concatenate([[0.0, 0.0, 0.05], d])
    _, res, _, tr = oracle.simulate(g, 0.1, 0.0, 0.0, 0, dict(beam=beam), 1, 1, trace_cap=64)
    cells = [(int(s["gid"]) % 4, (int(s["gid"]) // 4) % 4, int(s["gid"]) // 16) for s in tr]
    for a, b in zip(cells[:-1], cells[1:]):
        assert sum(abs(np.array(a) - np.array(b))) == 1           # one axis per step
    # x is crossed first, then y by a zero-length step
    assert cells[0] == (0, 0, 0) and cells[1] == (1, 0, 0) and cells[2][:2] == (1, 1)
    xy = [c[:2] for c in cells]
    assert all(c[0] - c[1] in (0, 1) for c in xy)                 # never (i, i+1): y never leads x
    assert (tr["ds"] == 0).sum() >= 2


@pytest.mark.parametrize("gg", [0.0, 0.6])
def test_scattering_angle_distribution_in_the_walk(gg):
    # beam into a uniform scattering medium: direction change at the FIRST scattering of each package
    g = _uniform_grid((9, 9, 9), 1.0)
    d0 = np.array([0.36, 0.48, 0.8])
    n = 15000
    _, res, rep, tr = oracle.simulate(g, 0.0, 0.7, gg, 0, dict(beam=np.concatenate([[4.5, 4.5, 0.0], d0])), n, 6,
                                      want_replay=True, trace_cap=2_000_000)
    first = np.concatenate([[0], np.cumsum(rep["steps"].astype(np.int64))[:-1]])
    cos, perp = [], []
    for p in range(n):
        s = tr[first[p]:first[p] + int(rep["steps"][p])]
        k = np.where(s["kind"] == 1)[0]
        if len(k) == 0 or k[0] + 1 >= len(s):
            continue
        nxt = s[k[0] + 1:]
        nxt = nxt[nxt["ds"] > 1e-9]
        if len(nxt) == 0:
            continue
        d1 = (nxt[0]["p1"] - nxt[0]["p0"]) / nxt[0]["ds"]
        cos.append(d1 @ d0)
        perp.append(d1 - (d1 @ d0) * d0)
    cos, perp = np.array(cos), np.array(perp)
    m = len(cos)
    assert m > 0.8 * n
    assert cos.mean() == pytest.approx(gg, abs=5 * cos.std() / m ** 0.5)
    assert (cos ** 2).mean() == pytest.approx((1 + 2 * gg * gg) / 3, abs=0.01)
    assert np.all(np.abs(perp.mean(axis=0)) < 5 * perp.std(axis=0) / m ** 0.5)    # azimuth covers the full circle
    # ... uniformly: second harmonic of the azimuth vanishes too
    e1 = np.cross(d0, [0, 0, 1.0]); e1 /= np.linalg.norm(e1); e2 = np.cross(d0, e1)
    az = np.arctan2(perp @ e2, perp @ e1)
    assert abs(np.cos(2 * az).mean()) < 5 / (2 * m) ** 0.5 and abs(np.sin(2 * az).mean()) < 5 / (2 * m) ** 0.5


def test_termination_threshold_is_1e9_of_the_initial_weight():
    # beam through a pure absorber with tau = 2.5 per cell: weight after k cells is exp(-2.5 k);
    # exp(-20) = 2.1e-9 survives, exp(-22.5) = 1.7e-10 terminates -> 9 steps, everything absorbed
    g = _uniform_grid((12, 3, 3), 1.0)
    A, res, rep, _ = oracle.simulate(g, 2.5, 0.0, 0.0, 0, dict(beam=[0, 1.5, 1.5, 1, 0, 0]), 1, 1, want_replay=True)
    assert rep["steps"][0] == 9 and res.terminated == 1 and res.escaped == 0.0
    assert A.sum() == pytest.approx(1.0, rel=1e-15) and A.reshape(3, 3, 12)[1, 1, 9:].sum() == 0.0


def test_stream_layout_inside_the_walk():
    """Block 0 (4 words) + block 1 word 0 -> emission; block 2+s word 0 -> free path of segment s,
    word 1 -> HG angle, word 2 -> azimuth at its end (reading S2).  Checked on recorded paths using only
    the (separately pinned) generator, uniform conversion, emission and HG functions."""
    shape = (5, 6, 4)
    g = _uniform_grid(shape, 1.0)
    seed, ifreq, n, gg = 77, 5, 300, 0.5
    _, res, rep, tr = oracle.simulate(g, 0.05, 0.9, gg, ifreq, dict(bg_intensity=1.0), n, seed, want_replay=True,
                                      trace_cap=100000)
    first = np.concatenate([[0], np.cumsum(rep["steps"].astype(np.int64))[:-1]])
    checked = 0
    for p in range(n):
        s = tr[first[p]:first[p] + int(rep["steps"][p])]
        b0, b1 = oracle.stream_block(seed, ifreq, p, 0), oracle.stream_block(seed, ifreq, p, 1)
        u = [oracle.uniform(x) for x in b0] + [oracle.uniform(b1[0])]
        ijk, f, d = oracle.emit_background(*shape, u)
        assert np.allclose(s[0]["p0"], ijk + f, atol=1e-14)
        nz = s[s["ds"] > 1e-9]
        assert np.allclose((nz[0]["p1"] - nz[0]["p0"]) / nz[0]["ds"], d, atol=1e-9)
        seg = 0
        d_prev = d
        for i, st in enumerate(s):
            blk = oracle.stream_block(seed, ifreq, p, 2 + seg)
            assert st["tau_drawn"] == pytest.approx(-math.log(oracle.uniform(blk[0])), rel=1e-14)
            if st["kind"] == 1:
                later = s[i + 1:]
                later = later[later["ds"] > 1e-9]
                if len(later):
                    d_new = (later[0]["p1"] - later[0]["p0"]) / later[0]["ds"]
                    expect = oracle.rotate(d_prev, oracle.hg_cos(gg, oracle.uniform(blk[1])),
                                           2 * math.pi * oracle.uniform(blk[2]))
                    # only compare when no further scattering happened before the next non-zero step
                    if not (s[i + 1:i + 1 + int(np.argmax(s[i + 1:]["ds"] > 1e-9))]["kind"] == 1).any():
                        assert np.allclose(d_new, expect, atol=1e-7)
                        checked += 1
                    d_prev = expect
                seg += 1
    assert checked > 100


# ------------------------------------------------------------------------------ the f32state variant
# soc_oracle_simulate_f32state (package state snapped to fp32 at every store) is licensed only by these pins
# against THE oracle (fp64 throughout) and by the closed forms it must still reach at fp32 tolerance.
def _records_equal(a, b):
    return (a["hash"] == b["hash"]) & (a["steps"] == b["steps"]) & (a["scatters"] == b["scatters"])


def test_f32state_identical_on_non_scattering_paths():
    # straight paths (ksca = 0): snapping moves a position by <= 6e-8 of a cell, which changes the visited
    # cells only for a path within that distance of a cell edge -- none among these 30k packages
    rng = np.random.default_rng(17)
    g = oracle.Grid(8, 8, 8, [512], rng.lognormal(0, 1, 512).astype(np.float32))
    src = dict(bg_intensity=1.0, ps_pos=np.array([[3.3, 4.6, 2.2]]), ps_lum=np.array([40.0]))
    A, r, rep, _ = oracle.simulate(g, 0.3, 0.0, 0.0, 0, src, 30000, 3, want_replay=True)
    B, q, rq, _ = oracle.simulate(g, 0.3, 0.0, 0.0, 0, src, 30000, 3, want_replay=True, f32state=True)
    assert _records_equal(rep, rq).all()
    assert q.emitted == r.emitted and q.cell_steps == r.cell_steps
    # a path of ~10 cells moves by <= 1e-6 of a cell; e^-tau with kabs rho up to ~10 per cell follows it
    assert np.allclose(rq["e_escaped"], rep["e_escaped"], rtol=1e-4, atol=0)
    assert np.abs(B - A).sum() <= 1e-6 * A.sum()
    n_cells, rho, child = random_octree((4, 4, 4), 3, 0.3, seed=5)
    gh = oracle.Grid(4, 4, 4, n_cells, rho, child)
    _, _, rep, _ = oracle.simulate(gh, 0.3, 0.0, 0.0, 0, dict(bg_intensity=1.0), 20000, 3, want_replay=True)
    _, _, rq, _ = oracle.simulate(gh, 0.3, 0.0, 0.0, 0, dict(bg_intensity=1.0), 20000, 3, want_replay=True, f32state=True)
    assert _records_equal(rep, rq).all()


@pytest.mark.parametrize("which", ["1", "2"])
def test_f32state_follows_the_fp64_oracle_on_config_1_2_like_runs(which):
    from paper_1812_06632_b200 import inputs
    P = inputs.make_config("1", n_packages=40000) if which == "1" else inputs.make_config("2", n=32, n_packages=40000)
    g = oracle.Grid(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child)
    src = P.sources(0)
    A, r, rep, _ = oracle.simulate(g, P.kabs[0], P.ksca[0], P.g[0], 0, src, P.n_packages, 1, want_replay=True, threads=4)
    B, q, rq, _ = oracle.simulate(g, P.kabs[0], P.ksca[0], P.g[0], 0, src, P.n_packages, 1, want_replay=True, threads=4,
                                  f32state=True)
    same = _records_equal(rep, rq).mean()
    assert same >= 0.99, same                       # the few that part ways scatter several times (chaotic map)
    assert np.abs(B - A).sum() <= 0.02 * A.sum()
    assert q.absorbed == pytest.approx(r.absorbed, rel=2e-3) and q.escaped == pytest.approx(r.escaped, rel=2e-3)
    assert abs(q.emitted - q.absorbed - q.escaped) <= 1e-9 * q.emitted      # weights and deposits stay fp64


def test_f32state_within_5_sigma_of_the_fp64_oracle_over_8_seeds():
    rng = np.random.default_rng(23)
    g = oracle.Grid(8, 8, 8, [512], rng.lognormal(0, 1, 512).astype(np.float32))
    src = dict(bg_intensity=1.0, ps_pos=np.array([[4.5, 3.5, 4.5]]), ps_lum=np.array([60.0]))
    runs, runs32 = [], []
    for seed in range(1, 9):
        runs.append(oracle.simulate(g, 0.2, 0.8, 0.6, 0, src, 20000, seed, threads=4)[0])
        runs32.append(oracle.simulate(g, 0.2, 0.8, 0.6, 0, src, 20000, seed, threads=4, f32state=True)[0])
    runs, runs32 = np.array(runs), np.array(runs32)
    sigma = runs.std(axis=0, ddof=1)
    assert (sigma > 0).all()
    assert (np.abs(runs32 - runs) <= 5 * sigma[None, :]).all()
    # and the 8-seed means agree far inside the noise of the mean
    assert np.abs(runs32.mean(0) - runs.mean(0)).max() <= 1.0 * (sigma / 8 ** 0.5).max()


def test_f32state_reaches_the_same_closed_forms():
    # slab: transmission exp(-tau) and per-cell deposits (axis-aligned: nothing to round)
    g = _uniform_grid((7, 5, 9), rho=2.0)
    beam = np.array([0.0, 2.5, 4.75, 1.0, 0.0, 0.0])
    A, res, _, _ = oracle.simulate(g, 0.15, 0.0, 0.0, 0, dict(beam=beam), 1, 1, f32state=True)
    assert res.escaped == pytest.approx(math.exp(-7 * 0.3), rel=1e-13)
    # oblique chord: to a few fp32 ulps
    shape = (6, 4, 5)
    g = _uniform_grid(shape, 1.5)
    d = np.array([0.6, 0.3, -0.5]); d /= np.linalg.norm(d)
    pos = np.array([0.0, 1.2, 4.4])
    _, res, _, tr = oracle.simulate(g, 0.2, 0.0, 0.0, 0, dict(beam=np.concatenate([pos, d])), 1, 1, trace_cap=100,
                                    f32state=True)
    tmax = min(((shape[j] if d[j] > 0 else 0) - pos[j]) / d[j] for j in range(3))
    assert tr["ds"].sum() == pytest.approx(tmax, rel=4 * F32)
    assert res.absorbed == pytest.approx(1 - math.exp(-0.2 * 1.5 * tmax), rel=4 * F32)
    # optically thin bath with scattering: A_c = 4 pi I kabs rho_c V_c
    rng = np.random.default_rng(2)
    g = oracle.Grid(6, 6, 6, [216], rng.lognormal(0, 1, 216).astype(np.float32))
    A, res, _, _ = oracle.simulate(g, 1e-6, 0.6, 0.6, 0, dict(bg_intensity=1.7), 150000, 21, threads=4, f32state=True)
    expect = 4 * math.pi * 1.7 * 1e-6 * g.rho.astype(np.float64)
    assert A.sum() / expect.sum() == pytest.approx(1.0, abs=0.006)
    # fully refined hierarchy = regular 2N grid: the ascent rounds (f + bit)/2 to fp32, so a package within an
    # ulp of a cell edge may take the corner cell in the other order
    N = 4
    rho2 = rng.lognormal(0, 0.8, (2 * N, 2 * N, 2 * N)).astype(np.float32)
    n_cells, rho, child, gid_of = fully_refined(rho2)
    gh = oracle.Grid(N, N, N, n_cells, rho, child)
    gr = oracle.Grid(2 * N, 2 * N, 2 * N, [8 * N ** 3], rho2.ravel())
    Ah, rh, reph, _ = oracle.simulate(gh, 0.3, 0.7, 0.4, 2, dict(bg_intensity=1.0), 20000, 5, want_replay=True, f32state=True)
    Ar, rr, repr_, _ = oracle.simulate(gr, 0.15, 0.35, 0.4, 2, dict(bg_intensity=0.25), 20000, 5, want_replay=True, f32state=True)
    assert ((reph["steps"] == repr_["steps"]) & (reph["scatters"] == repr_["scatters"])).mean() >= 0.999
    assert np.abs(Ah[gid_of.ravel()] - Ar).sum() <= 1e-3 * Ar.sum()
