"""GPU parity of the dust re-emission source, the package counts, the ALI update and the iteration driver (rows f1, f3)
against the CPU oracle, through the C ABI.  Tolerances as in test_gpu_parity.py."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from gpu_common import N_THREADS, oracle_grid, rel_l1, replay_match
from helpers import random_octree
from paper_1812_06632_b200 import inputs, soc

REPLAY, PROD = soc.SOC_GEOM_FP64, soc.SOC_GEOM_FP32


def _torch():
    import torch
    return torch


def _hot_problem(which="3", n=8, n_freq=8, tau_scale=100.0, lum_scale=500.0, n_packages=30000):
    P = inputs.make_config(which, n=n, n_packages=n_packages, n_freq=n_freq)
    P.kabs = P.kabs * tau_scale
    P.ksca = P.ksca * tau_scale
    P.t_scale = P.t_scale / tau_scale
    if P.n_point:
        P.ps_lum = P.ps_lum * lum_scale
    else:
        P.bg_intensity = P.bg_intensity * lum_scale
    return P


def _temperatures(P, seed=3):
    rng = np.random.default_rng(seed)
    T = rng.uniform(8.0, 90.0, P.n_total).astype(np.float32)
    T[rng.uniform(size=P.n_total) < 0.05] = 0.0          # some cells emit nothing
    return T


def _gpu_dust(G, P, f, T_dev, cnt_dev, n_dust, seed, flags, want_replay, self_abs=None, extra=None, weight=1.0):
    torch = _torch()
    src = dict(dust_T=T_dev, dust_count=cnt_dev, n_dust=n_dust, dust_self=self_abs, n_bg=0)
    n = n_dust
    if extra:
        src.update(extra)
        n = n_dust + extra["_n_const"]
        src["n_bg"] = -1
    A = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
    rep = torch.zeros(n * soc.REPLAY_DTYPE.itemsize, dtype=torch.uint8, device="cuda") if want_replay else None
    r = G.simulate_packages(f, src, n, seed, weight, 0, n, A, rep, flags=flags)
    torch.cuda.synchronize()
    return A.cpu().numpy(), r, (rep.cpu().numpy().view(soc.REPLAY_DTYPE) if want_replay else None)


@pytest.mark.parametrize("which", ["3", "4p"])
def test_emission_counts_match_the_oracle(which):
    torch = _torch()
    P = _hot_problem(which, n=8)
    G = soc.Grid.from_problem(P)
    og = oracle_grid(P)
    T = _temperatures(P)
    Td = torch.from_numpy(T).cuda()
    cnt = torch.zeros(P.n_total, dtype=torch.int32, device="cuda")
    for f in (0, P.n_freq // 2, P.n_freq - 1):
        L = oracle.cell_luminosity(og, P.kabs[f], P.freq_hz[f], T)
        for mode, n_req, cap in (("uniform", 5000, 1), ("weighted", 40000, 300), ("weighted", 0, 10)):
            n_dust, tot = G.emission_counts(f, Td, mode, n_req, cap, cnt)
            co = oracle.emission_counts(og, P.kabs[f], P.freq_hz[f], T, mode, n_req, cap)
            cg = cnt.cpu().numpy()
            assert tot == pytest.approx(L.sum(), rel=1e-12) and n_dust == int(cg.sum())
            # ceil(n_request L_c / sum L) is taken in fp64 on both sides: a cell within an ulp of an integer may differ by 1
            assert (cg != co).sum() <= 2 and np.abs(cg - co).max() <= 1
            assert ((cg > 0) == (L > 0)).all() or n_req == 0
    G.close()


@pytest.mark.parametrize("which,mode", [("3", "uniform"), ("3", "weighted"), ("4p", "weighted")])
def test_dust_emission_replay(which, mode):
    """Replay parity of the dust source: identical cell sequences for >= 99.9 % of the packages, per-cell L1 <= 1e-4, the
    in-cell absorption accumulator (f3) to the same L1; counts from the oracle's policy routine on both sides."""
    torch = _torch()
    P = _hot_problem(which, n=8)
    G = soc.Grid.from_problem(P)
    og = oracle_grid(P)
    T = _temperatures(P)
    Td = torch.from_numpy(T).cuda()
    for f in (1, P.n_freq - 3):
        cnt = oracle.emission_counts(og, P.kabs[f], P.freq_hz[f], T, mode, 60000, cap=500)
        n_dust = int(cnt.sum())
        assert n_dust > 0
        So = np.zeros(P.n_total)
        src = dict(dust_T=T, dust_count=cnt, dust_freq_hz=P.freq_hz[f], dust_self=So, n_bg=0)
        Ao, ro, repo, _ = oracle.simulate(og, P.kabs[f], P.ksca[f], P.g[f], f, src, n_dust, 11, 0.5, want_replay=True,
                                          threads=N_THREADS, f32state=True)
        Sg = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
        Ag, rg, repg = _gpu_dust(G, P, f, Td, torch.from_numpy(cnt).cuda(), n_dust, 11, REPLAY, True, self_abs=Sg, weight=0.5)
        assert replay_match(repg, repo) >= 0.999
        assert rel_l1(Ag, Ao) <= 1e-4 and rel_l1(Sg.cpu().numpy(), So) <= 1e-4
        assert rg.emitted == pytest.approx(ro.emitted, rel=1e-12)
        assert abs(rg.emitted - rg.absorbed - rg.escaped) <= 1e-6 * rg.emitted
        L = oracle.cell_luminosity(og, P.kabs[f], P.freq_hz[f], T)
        assert rg.emitted == pytest.approx(L.sum(), rel=1e-12)
    G.close()


def test_dust_with_constant_sources_in_one_call():
    """Background + point sources + dust in one launch: ids [0, n_bg) background, then point sources, the last n_dust dust."""
    torch = _torch()
    P = _hot_problem("3", n=8)
    G = soc.Grid.from_problem(P)
    og = oracle_grid(P)
    T = _temperatures(P)
    f = 2
    cnt = oracle.emission_counts(og, P.kabs[f], P.freq_hz[f], T, "weighted", 20000, cap=200)
    n_dust, n_const = int(cnt.sum()), 30001
    src_o = dict(P.sources(f), dust_T=T, dust_count=cnt, dust_freq_hz=P.freq_hz[f])
    Ao, ro, repo, _ = oracle.simulate(og, P.kabs[f], P.ksca[f], P.g[f], f, src_o, n_const + n_dust, 5, want_replay=True,
                                      threads=N_THREADS, f32state=True)
    extra = dict(P.sources(f), _n_const=n_const)
    for flags, min_match, max_l1 in ((REPLAY, 0.999, 1e-4), (PROD, 0.98, 2e-2)):
        Ag, rg, repg = _gpu_dust(G, P, f, torch.from_numpy(T).cuda(), torch.from_numpy(cnt).cuda(), n_dust, 5, flags, True, extra=extra)
        assert replay_match(repg, repo) >= min_match and rel_l1(Ag, Ao) <= max_l1
        assert rg.emitted == pytest.approx(ro.emitted, rel=1e-12 if flags == REPLAY else 1e-6)
        assert abs(rg.emitted - rg.absorbed - rg.escaped) <= 1e-6 * rg.emitted
        assert Ag.sum() == pytest.approx(rg.absorbed, rel=5e-6)
    G.close()


def test_slab_blocked_dust_launch_walks_the_same_paths():
    """Dust packages (per-package energies, in-cell absorption of f3) through the slab-blocked launch, alone and together
    with background and point-source packages: the counts of the one-launch photon_q_kernel, per-cell sums to the order of
    the fp32 additions, in-cell absorption likewise."""
    torch = _torch()
    P = _hot_problem("3", n=24, n_packages=60000)
    G = soc.Grid.from_problem(P)
    G.set_option("kernel", 2)
    og = oracle_grid(P)
    T = _temperatures(P)
    Td = torch.from_numpy(T).cuda()
    for f, extra in ((P.n_freq - 3, None), (2, dict(P.sources(2), _n_const=40001))):
        cnt = oracle.emission_counts(og, P.kabs[f], P.freq_hz[f], T, "weighted", 200_000, cap=500)
        n_dust, cd = int(cnt.sum()), torch.from_numpy(cnt).cuda()
        out = []
        for n_slabs in (1, 3):
            G.set_option("slabs", n_slabs)
            Sg = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
            Ag, rg, _ = _gpu_dust(G, P, f, Td, cd, n_dust, 7, PROD, False, self_abs=Sg, extra=extra)
            out.append((Ag, Sg.cpu().numpy(), rg))
        (A1, S1, r1), (A2, S2, r2) = out
        assert (r1.cell_steps, r1.scatterings, r1.terminated) == (r2.cell_steps, r2.scatterings, r2.terminated)
        assert r1.suspensions == 0 and r2.suspensions > 0
        assert r2.emitted == pytest.approx(r1.emitted, rel=1e-12) and r2.escaped == pytest.approx(r1.escaped, rel=1e-9)
        # (in-cell absorption: the fp32 deposit sum of a visit that is split at a hand-over between phases rounds differently)
        assert rel_l1(A2, A1) <= 2e-6 and rel_l1(S2, S1) <= 1e-7
        assert A2.sum() == pytest.approx(r2.absorbed, rel=5e-6)
    G.close()


@pytest.mark.parametrize("which,kernel,n_slabs", [("3", 1, 1), ("3", 2, 1), ("3", 2, 3), ("4p", 0, 1)])
def test_dust_production_mode_within_5_sigma(which, kernel, n_slabs):
    """Production kernels (photon_fast_kernel, photon_q_kernel in one launch and slab-blocked, the octree kernel) with the
    dust source: 8 seeds, every cell within 5 sigma of the oracle's MC noise; in-cell absorption likewise; conservation
    through the cells."""
    torch = _torch()
    P = _hot_problem(which, n=8 if which == "4p" else 12)
    G = soc.Grid.from_problem(P)
    G.set_option("kernel", kernel)
    G.set_option("slabs", n_slabs)
    og = oracle_grid(P)
    T = _temperatures(P)
    Td = torch.from_numpy(T).cuda()
    f = P.n_freq - 3
    cnt = oracle.emission_counts(og, P.kabs[f], P.freq_hz[f], T, "weighted", 150_000, cap=2000)
    n_dust = int(cnt.sum())
    cd = torch.from_numpy(cnt).cuda()
    Ao, So = [], []
    for seed in range(1, 9):
        s = np.zeros(P.n_total)
        src = dict(dust_T=T, dust_count=cnt, dust_freq_hz=P.freq_hz[f], dust_self=s, n_bg=0)
        Ao.append(oracle.simulate(og, P.kabs[f], P.ksca[f], P.g[f], f, src, n_dust, seed, threads=N_THREADS)[0])
        So.append(s)
    Ao, So = np.array(Ao), np.array(So)
    sig_a, sig_s = Ao.std(axis=0, ddof=1), So.std(axis=0, ddof=1)
    for seed in range(1, 9):
        Sg = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
        Ag, rg, _ = _gpu_dust(G, P, f, Td, cd, n_dust, seed, PROD, False, self_abs=Sg)
        assert abs(rg.emitted - rg.absorbed - rg.escaped) <= 1e-6 * rg.emitted
        assert Ag.sum() == pytest.approx(rg.absorbed, rel=5e-6)
        da, ds = np.abs(Ag - Ao[seed - 1]), np.abs(Sg.cpu().numpy() - So[seed - 1])
        # (cells whose luminosity lies > 30 decades below the mean package energy -- cold cells at short wavelengths --
        #  carry no measurable energy: their packages underflow the fp32 unit of the launch, hence the absolute floor)
        floor_a, floor_s = 1e-12 * Ao.max(), 1e-12 * So.max()
        assert (da <= 5 * sig_a + 1e-6 * np.abs(Ao[seed - 1]) + floor_a).all(), float((da / np.where(sig_a > 0, sig_a, np.inf)).max())
        assert (ds <= 5 * sig_s + 1e-6 * np.abs(So[seed - 1]) + floor_s).all(), float((ds / np.where(sig_s > 0, sig_s, np.inf)).max())
        assert rg.emitted == pytest.approx(oracle.cell_luminosity(og, P.kabs[f], P.freq_hz[f], T).sum(), rel=1e-6)
    G.close()


def test_kirchhoff_on_the_gpu():
    """Deep inside an opaque isothermal cloud a cell absorbs what it emits (J = B), production kernel, no oracle."""
    torch = _torch()
    N = 14
    rho = np.random.default_rng(5).uniform(0.8, 1.25, N ** 3).astype(np.float32)
    P = inputs.Problem("adhoc", N, N, N, np.array([N ** 3]), rho, None, np.array([3e12]), np.array([2.0]), np.array([1.5]),
                       np.array([0.4]), np.array([0.0]), np.zeros((0, 3)), np.zeros((1, 0)), 1)
    G = soc.Grid.from_problem(P)
    T = np.full(N ** 3, 40.0, dtype=np.float32)
    Td = torch.from_numpy(T).cuda()
    cnt = torch.zeros(N ** 3, dtype=torch.int32, device="cuda")
    n_dust, tot = G.emission_counts(0, Td, "uniform", 400 * N ** 3, 1, cnt)
    A, r, _ = _gpu_dust(G, P, 0, Td, cnt, n_dust, 9, PROD, False)
    G.close()
    L = 4 * math.pi * 2.0 * rho.astype(np.float64) * inputs.planck_nu(3e12, 40.0)
    i = np.arange(N)
    inner = (i >= 5) & (i < N - 5)
    m = (inner[:, None, None] & inner[None, :, None] & inner[None, None, :]).ravel()
    ratio = A[m] / L[m]
    assert ratio.mean() == pytest.approx(1.0, abs=4 * ratio.std() / math.sqrt(m.sum()) + 2e-3)
    assert r.emitted == pytest.approx(L.sum(), rel=1e-6) and tot == pytest.approx(L.sum(), rel=1e-12)


def test_cell_emission_and_ali_update_match_the_oracle():
    torch = _torch()
    n_cells, rho, child = random_octree((4, 3, 3), 3, 0.4, seed=8, p_empty=0.15)
    P0 = _hot_problem("3", n=4, n_freq=10)
    P = inputs.Problem("adhoc", 4, 3, 3, np.asarray(n_cells, dtype=np.int64), rho, child, P0.freq_hz, P0.kabs, P0.ksca, P0.g,
                       P0.bg_intensity, np.zeros((0, 3)), np.zeros((P0.n_freq, 0)), 1, t_scale=P0.t_scale, table_T=P0.table_T,
                       e_min=P0.e_min, e_max=P0.e_max)
    G = soc.Grid.from_problem(P)
    og = oracle_grid(P)
    T = _temperatures(P, seed=4)
    w = oracle.trapezoid_weights(P.freq_hz)
    Em_o = sum(w[f] * oracle.cell_luminosity(og, P.kabs[f], P.freq_hz[f], T) for f in range(P.n_freq))
    Em = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
    G.cell_emission(torch.from_numpy(T).cuda(), Em)
    assert np.allclose(Em.cpu().numpy(), Em_o, rtol=1e-12, atol=0)
    rng = np.random.default_rng(2)
    S = Em_o * rng.uniform(0, 0.9, P.n_total)
    A = S + Em_o * rng.uniform(0.0, 2.0, P.n_total)
    To = oracle.update_temperatures_ali(og, A, S, Em_o, P.t_scale, P.table_T, P.e_min, P.e_max)
    Tg = torch.zeros(P.n_total, dtype=torch.float32, device="cuda")
    G.update_temperatures_ali(torch.from_numpy(A).cuda(), torch.from_numpy(S).cuda(), Em, P.t_scale, P.table_T, P.e_min, P.e_max, Tg)
    assert np.abs(Tg.cpu().numpy() - To).max() <= 0.01
    G.close()


@pytest.mark.parametrize("ali,reference_field", [(False, False), (True, True)])
def test_iterate_matches_the_oracle(ali, reference_field):
    """soc_iterate in replay mode against oracle.iterate: same package counts, same packages, same running mean, so the
    temperatures of every iteration's end agree to 0.01 K and the histories to 1e-6."""
    torch = _torch()
    P = _hot_problem("3", n=6, n_freq=8, tau_scale=300.0, lum_scale=500.0, n_packages=20000)
    G = soc.Grid.from_problem(P)
    og = oracle_grid(P)
    srcs = [P.sources(f) for f in range(P.n_freq)]
    n_req = [15000, 30000, 60000]                      # variable number of packages per iteration
    out = oracle.iterate(og, P.freq_hz, P.kabs, P.ksca, P.g, srcs, P.n_packages, n_req, P.seed, P.t_scale, P.table_T, P.e_min,
                         P.e_max, mode="weighted", cap=3000, reference_field=reference_field, ref_start=2, ali=ali,
                         threads=N_THREADS, f32state=True)
    A = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
    T = torch.zeros(P.n_total, dtype=torch.float32, device="cuda")
    hist = G.iterate(srcs, P.n_packages, P.seed, n_req, P.t_scale, P.table_T, P.e_min, P.e_max, A, T, mode="weighted", cap=3000,
                     reference_field=reference_field, ref_start=2, ali=ali, flags=REPLAY)
    G.close()
    To = out["T"][-1]
    assert np.abs(T.cpu().numpy() - To).max() <= 0.01
    assert rel_l1(A.cpu().numpy(), out["A_const"] + out["R"]) <= 1e-4
    for i in range(len(n_req) + 1):
        assert hist[i]["emitted"] == pytest.approx(out["emitted"][i], rel=1e-6)
        assert hist[i]["escaped"] == pytest.approx(out["escaped"][i], rel=1e-4)
    assert To.max() > out["T"][0].max() + 0.5          # the iterations matter in this model
    assert [h["n_packages"] for h in hist[1:]] == out["n_dust"] or all(
        abs(h["n_packages"] - n) <= 2 * P.n_freq for h, n in zip(hist[1:], out["n_dust"]))


def test_iterate_production_mode_energy_balance():
    """soc_iterate with the production kernels: the whole-box balance the oracle's pin checks -- the dust emission that
    escapes approaches what the constant sources put into the dust."""
    torch = _torch()
    P = _hot_problem("3", n=8, n_freq=10, tau_scale=400.0, lum_scale=300.0, n_packages=40000)
    G = soc.Grid.from_problem(P)
    A = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
    T = torch.zeros(P.n_total, dtype=torch.float32, device="cuda")
    hist = G.iterate([P.sources(f) for f in range(P.n_freq)], P.n_packages, P.seed, [60000] * 10, P.t_scale, P.table_T, P.e_min,
                     P.e_max, A, T, mode="weighted", cap=4000, reference_field=False)
    G.close()
    a_const = hist[0]["absorbed"]
    ratio = np.array([h["escaped"] for h in hist[1:]]) / a_const
    assert ratio[0] < 0.6 and 0.93 < ratio[-1] < 1.04 and (np.diff(ratio) > -0.03).all()
    for h in hist:
        assert abs(h["emitted"] - h["absorbed"] - h["escaped"]) <= 1e-6 * h["emitted"]


def test_iterate_at_full_size_is_measured(capsys):
    """Config 3 at full size (128^3, 64 frequencies), made opaque and luminous like the paper's iteration tests
    (PAPER.md:139), through soc_iterate with the production kernels: emission-weighted counts with the paper's cap of 10000,
    reference field after a burn-in, ALI.  Properties that hold at any size (conservation per iteration, global balance
    approached) and the throughput of the dust launches, printed."""
    import time
    torch = _torch()
    P = _hot_problem("3", n=128, n_freq=64, tau_scale=30.0, lum_scale=3000.0, n_packages=4_000_000)
    G = soc.Grid.from_problem(P)
    A = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
    T = torch.zeros(P.n_total, dtype=torch.float32, device="cuda")
    n_req = [1_000_000, 2_000_000, 4_000_000, 4_000_000]          # growing package numbers
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    hist = G.iterate([P.sources(f) for f in range(P.n_freq)], P.n_packages, P.seed, n_req, P.t_scale, P.table_T, P.e_min,
                     P.e_max, A, T, mode="weighted", cap=10000, reference_field=True, ref_start=3, ali=True)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    G.close()
    for h in hist:
        assert abs(h["emitted"] - h["absorbed"] - h["escaped"]) <= 1e-6 * h["emitted"]
    a_const = hist[0]["absorbed"]
    ratio = [h["escaped"] / a_const for h in hist[1:]]
    assert ratio[-1] > ratio[0] and 0.5 < ratio[-1] < 1.05
    Tn = T.cpu().numpy()
    assert Tn.max() > 100.0 and np.median(Tn[Tn > 0]) > 5.0       # hot dust near the sources only
    steps = sum(h["cell_steps"] for h in hist)
    with capsys.disabled():
        print(f"\n[soc_iterate, config 3 at 128^3 x 64 frequencies, 4 iterations with ALI + reference field] {dt:.2f} s wall, "
              f"{steps:.3e} cell-steps = {steps / dt:.3e} cell-steps/s incl. counts, scans and temperature updates; packages per "
              f"iteration {[h['n_packages'] for h in hist]}; escaped dust emission / A_const per iteration {[round(r, 3) for r in ratio]}; "
              f"T max {Tn.max():.0f} K")


def test_dust_spectrum_with_counts_per_frequency_does_not_depend_on_the_overlap_option():
    """A dust spectrum passed straight to soc_simulate_spectrum, package counts differing from frequency to frequency
    (emission-weighted).  The prefix sums of the counts and the scan scratch exist once per grid, so two frequencies in
    flight on two streams would search each other's offsets: with dust sources the launches stay serial whatever the
    option says.  overlap = 1 must give the counters of overlap = 0 exactly and the same integral up to the order of the
    additions, every frequency must emit the luminosity of its sending cells, and nothing may turn inf / NaN."""
    torch = _torch()
    P = _hot_problem("3", n=16, n_freq=8, n_packages=60_000)
    G = soc.Grid.from_problem(P)
    Td = torch.from_numpy(_temperatures(P)).cuda()
    srcs, lum = [], []
    for f in range(P.n_freq):
        cnt = torch.zeros(P.n_total, dtype=torch.int32, device="cuda")
        n_dust, tot = G.emission_counts(f, Td, "weighted", 12_000 + 5_000 * f, 40, cnt)
        assert 0 <= n_dust < P.n_packages
        s = dict(P.sources(f))
        if n_dust > 0:                  # (towards the UV no cell of 8-90 K emits: those frequencies carry constant sources only)
            s.update(dust_T=Td, dust_count=cnt, n_dust=n_dust)
        srcs.append(s)
        lum.append(tot)
    with_dust = [s["n_dust"] for s in srcs if s.get("n_dust", 0) > 0]
    assert len(with_dust) >= 4 and len(set(with_dust)) == len(with_dust)      # every dust frequency has its own offsets
    out = []
    for overlap in (0, 1, 1):
        G.set_option("overlap", overlap)
        A = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
        res = G.simulate_spectrum(srcs, P.n_packages, 11, A)
        torch.cuda.synchronize()
        out.append((A.cpu().numpy(), res))
    G.close()
    for A, res in out:
        assert np.isfinite(A).all() and all(np.isfinite(r.emitted) and r.emitted > 0 for r in res)
        assert all(abs(r.emitted - r.absorbed - r.escaped) <= 1e-6 * r.emitted for r in res)
    for A, res in out[1:]:
        assert [(r.cell_steps, r.scatterings, r.terminated) for r in res] == [(r.cell_steps, r.scatterings, r.terminated) for r in out[0][1]]
        assert all(a.emitted == pytest.approx(b.emitted, rel=1e-12) for a, b in zip(res, out[0][1]))
        assert np.allclose(A, out[0][0], rtol=2e-5, atol=0)
    # the dust part of what a frequency emits is the luminosity of all cells (weighted counts: every emitting cell sends)
    Gc = soc.Grid.from_problem(P)
    for f in (0, 2, P.n_freq - 1):
        s = dict(P.sources(f))
        n_const = P.n_packages - srcs[f].get("n_dust", 0)
        A = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
        rc = Gc.simulate_packages(f, s, n_const, 11, 1.0, 0, n_const, A, None, flags=PROD)
        assert out[0][1][f].emitted - rc.emitted == pytest.approx(lum[f], rel=1e-5)
    Gc.close()
