"""Pins for the oracle's surface-brightness maps (row f2; readings M1, M2 of DESIGN.md): closed
forms, the optically thin column, an oblique chord, octree = equivalent regular grid, and a brute-force integration that
does not use the cell walk at all (point location top-down at fine steps along the line of sight)."""
import math

import numpy as np
import pytest

import oracle
from helpers import fully_refined, random_octree
from paper_1812_06632_b200 import inputs

NU = 3.0e12
EX, EY, EZ = np.eye(3)


def B(T):
    return float(inputs.planck_nu(NU, T))


def test_uniform_slab_closed_form_along_the_three_axes():
    shape = (5, 7, 4)
    g = oracle.Grid(*shape, [5 * 7 * 4], np.full(5 * 7 * 4, 1.5, dtype=np.float32))
    T = np.full(g.n_total, 30.0, dtype=np.float32)
    kabs, ksca = 0.2, 0.1
    centre = np.array(shape) / 2
    for axis, (ex, ey, d) in enumerate(((EY, EZ, EX), (EZ, EX, EY), (EX, EY, EZ))):
        npx, npy = shape[(axis + 1) % 3], shape[(axis + 2) % 3]
        m = oracle.make_map(g, kabs, ksca, NU, T, ex, ey, d, centre, npx, npy, 1.0)
        tau = (kabs + ksca) * 1.5 * shape[axis]
        assert np.allclose(m, kabs / (kabs + ksca) * B(30.0) * (1 - math.exp(-tau)), rtol=1e-13)
        m2 = oracle.make_map(g, kabs, ksca, NU, T, ex, ey, -d, centre, npx, npy, 1.0)      # from the other side: the same
        assert np.allclose(m2, m, rtol=1e-13)
    # a pixel whose line of sight misses the cloud sees nothing
    m = oracle.make_map(g, kabs, ksca, NU, T, EX, EY, EZ, centre, 9, 9, 1.0)
    assert (m[:, 0] == 0).all() and (m[:, -1] == 0).all() and (m[0] == 0).all() and m[4, 4] > 0


def test_optically_thin_map_is_the_emission_column():
    """tau << 1: I = sum along the line of sight of kabs rho B_nu(T) ds -- a plain numpy projection of the cell arrays."""
    rng = np.random.default_rng(3)
    n = 6
    rho = rng.lognormal(0, 1, (n, n, n)).astype(np.float32)          # [z][y][x]
    T = rng.uniform(10, 60, (n, n, n)).astype(np.float32)
    g = oracle.Grid(n, n, n, [n ** 3], rho.ravel())
    kabs = 1e-7
    j = kabs * rho.astype(np.float64) * inputs.planck_nu(NU, T.astype(np.float64))
    c = np.full(3, n / 2)
    mz = oracle.make_map(g, kabs, 3e-7, NU, T.ravel(), EX, EY, EZ, c, n, n, 1.0)        # pixel (i, j) = (x, y)
    assert np.allclose(mz, j.sum(axis=0), rtol=1e-5)
    mx = oracle.make_map(g, kabs, 3e-7, NU, T.ravel(), EY, EZ, EX, c, n, n, 1.0)        # pixel (i, j) = (y, z)
    assert np.allclose(mx, j.sum(axis=2), rtol=1e-5)
    my = oracle.make_map(g, kabs, 3e-7, NU, T.ravel(), EZ, EX, EY, c, n, n, 1.0)        # pixel (i, j) = (z, x)
    assert np.allclose(my, j.sum(axis=1).T, rtol=1e-5)


def test_front_cells_hide_the_back_cells():
    """Two slabs of different temperature along z: I = S1 (1 - e^-t1) + e^-t1 S2 (1 - e^-t2); reversed from the other side."""
    n = 4
    rho = np.ones((n, n, n), dtype=np.float32)
    T = np.empty((n, n, n), dtype=np.float32)
    T[:2], T[2:] = 20.0, 50.0
    g = oracle.Grid(n, n, n, [n ** 3], rho.ravel())
    kabs, ksca = 0.5, 0.25
    t = (kabs + ksca) * 2
    w = kabs / (kabs + ksca)
    c = np.full(3, n / 2)
    front = oracle.make_map(g, kabs, ksca, NU, T.ravel(), EX, EY, EZ, c, n, n, 1.0)
    back = oracle.make_map(g, kabs, ksca, NU, T.ravel(), EX, EY, -EZ, c, n, n, 1.0)
    e = math.exp(-t)
    assert np.allclose(front, w * (B(20.0) * (1 - e) + e * B(50.0) * (1 - e)), rtol=1e-13)
    assert np.allclose(back, w * (B(50.0) * (1 - e) + e * B(20.0) * (1 - e)), rtol=1e-13)


def _basis(theta, phi):
    d = -np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])   # into the cloud
    ex = np.array([-math.sin(phi), math.cos(phi), 0.0])
    ey = np.cross(d, ex)
    return ex, ey / np.linalg.norm(ey), d


def test_oblique_view_of_a_thin_uniform_cube_gives_the_chord():
    n = 8
    g = oracle.Grid(n, n, n, [n ** 3], np.ones(n ** 3, dtype=np.float32))
    T = np.full(n ** 3, 25.0, dtype=np.float32)
    ex, ey, d = _basis(0.9, 0.4)
    c = np.full(3, n / 2)
    npx = 24
    m = oracle.make_map(g, 1e-8, 0.0, NU, T, ex, ey, d, c, npx, npx, 0.6)
    for (i, j) in ((12, 12), (3, 17), (20, 5), (0, 0), (9, 14)):
        o = c + ((i + 0.5) - npx / 2) * 0.6 * ex + ((j + 0.5) - npx / 2) * 0.6 * ey
        t0 = np.where(d > 0, (0 - o) / d, (n - o) / d).max()
        t1 = np.where(d > 0, (n - o) / d, (0 - o) / d).min()
        chord = max(0.0, t1 - t0)
        assert m[j, i] == pytest.approx(1e-8 * B(25.0) * chord, rel=1e-6, abs=1e-30)


def test_octree_map_equals_the_map_of_the_equivalent_regular_grid():
    N = 4
    rng = np.random.default_rng(8)
    rho2 = rng.lognormal(0, 0.8, (2 * N, 2 * N, 2 * N)).astype(np.float32)
    T2 = rng.uniform(10, 70, (2 * N, 2 * N, 2 * N)).astype(np.float32)
    n_cells, rho, child, gid_of = fully_refined(rho2)
    gh = oracle.Grid(N, N, N, n_cells, rho, child)
    gr = oracle.Grid(2 * N, 2 * N, 2 * N, [8 * N ** 3], rho2.ravel())
    Th = np.zeros(gh.n_total, dtype=np.float32)
    Th[gid_of.ravel()] = T2.ravel()
    ex, ey, d = _basis(1.1, 2.3)
    # the regular grid's length unit is half a root cell: opacities halve, pixel and centre double
    mh = oracle.make_map(gh, 0.4, 0.3, NU, Th, ex, ey, d, np.full(3, N / 2), 20, 20, 0.35)
    mr = oracle.make_map(gr, 0.2, 0.15, NU, T2.ravel(), ex, ey, d, np.full(3, N), 20, 20, 0.70)
    assert np.allclose(mh, mr, rtol=1e-9, atol=1e-12 * mr.max())
    assert (mh > 0).sum() > 100


def _locate(n_cells, child, root_shape, x):
    """Top-down point location: global id of the leaf that holds the point x (root-cell units)."""
    off = np.concatenate([[0], np.cumsum(n_cells)])
    nx, ny, nz = root_shape
    c = np.minimum(np.floor(x).astype(int), np.array(root_shape) - 1)
    f = x - c
    gid, lvl = c[0] + nx * (c[1] + ny * c[2]), 0
    while child[gid] >= 0:
        b = (f >= 0.5).astype(int)
        f = 2 * f - b
        lvl += 1
        gid = off[lvl] + child[gid] + b[0] + 2 * b[1] + 4 * b[2]
    return gid


def test_bruteforce_integration_along_the_line_of_sight():
    """The same integral by fine sampling: dI = e^-tau kabs rho B ds at 4000 points per line, leaf found top-down from the
    root at every point -- no cell walk, no neighbour search."""
    shape = (3, 3, 3)
    n_cells, rho, child = random_octree(shape, 3, 0.5, seed=12, p_empty=0.1)
    g = oracle.Grid(*shape, n_cells, rho, child)
    rng = np.random.default_rng(1)
    T = rng.uniform(15, 60, g.n_total).astype(np.float32)
    kabs, ksca = 0.6, 0.3
    ex, ey, d = _basis(0.7, 1.9)
    c = np.array(shape) / 2
    npx, pix = 6, 0.55
    m = oracle.make_map(g, kabs, ksca, NU, T, ex, ey, d, c, npx, npx, pix)
    for (i, j) in ((2, 3), (0, 5), (3, 2), (4, 1)):
        o = c + ((i + 0.5) - npx / 2) * pix * ex + ((j + 0.5) - npx / 2) * pix * ey
        t0 = np.where(d > 0, (0 - o) / d, (np.array(shape) - o) / d).max()
        t1 = np.where(d > 0, (np.array(shape) - o) / d, (0 - o) / d).min()
        if t1 <= t0:
            assert m[j, i] == 0.0
            continue
        ns = 4000
        ds = (t1 - t0) / ns
        I = tau = 0.0
        for k in range(ns):
            x = o + (t0 + (k + 0.5) * ds) * d
            gid = _locate(n_cells, child, shape, np.clip(x, 0, np.array(shape) - 1e-12))
            r = float(rho[gid])
            dt = (kabs + ksca) * r * ds
            if dt > 0:
                I += math.exp(-tau) * kabs / (kabs + ksca) * B(float(T[gid])) * -math.expm1(-dt)
            tau += dt
        assert m[j, i] == pytest.approx(I, rel=3e-3)
