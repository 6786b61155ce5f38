"""CPU-side checks of the boundary and of the host logic (no compute calls, no GPU):

  * the C-ABI library loads and exports every function include/soc.h declares, and the Python binding
    names the same set;
  * argument validation that happens before any CUDA call returns SOC_EINVAL with a message;
  * the multi-GPU plan: shards cover the package ids exactly once, and the one
    collective of the path -- a sum all-reduce of the per-cell fp64 array -- is exercised with world_size 2
    over gloo, the per-rank arrays coming from the CPU oracle run on each rank's shard.
"""
import ctypes as C
import os
import re
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "soc.h")


def _declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(soc_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_1812_06632_b200 import build, soc
    build.build()
    lib = C.CDLL(soc.LIB_PATH)
    names = _declared_functions()
    assert len(names) >= 15
    for n in names:
        assert getattr(lib, n) is not None, n
    assert sorted(soc.EXPORTS) == names, "binding and header disagree on the exported calls"


def test_library_has_sm100a_code_only():
    """The product is sm_100a code: the fat binary holds an sm_100a cubin (cuobjdump) and nothing else."""
    import shutil
    import subprocess
    from paper_1812_06632_b200 import build, soc
    build.build()
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", soc.LIB_PATH], stdout=subprocess.PIPE, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_argument_validation_without_a_device():
    """Checks that run before the first CUDA call: they must fail with SOC_EINVAL and leave a message."""
    from paper_1812_06632_b200 import build, soc
    build.build()
    L = soc.load()
    h = C.c_void_p()
    assert L.soc_grid_create(None, C.byref(h)) == -1
    assert b"NULL" in L.soc_last_error()
    P = dict(nx=2, ny=2, nz=2, n_cells=[7], density=np.ones(8, np.float32), child=None, freq_hz=[1e14], kabs=[1.0],
             ksca=[1.0], g=[0.0])
    desc, keep = soc.make_desc(**P)
    assert L.soc_grid_create(C.byref(desc), C.byref(h)) == -1           # n_cells[0] != nx*ny*nz
    assert b"n_cells" in L.soc_last_error()
    P["n_cells"] = [8]; P["g"] = [1.0]
    desc, keep = soc.make_desc(**P)
    assert L.soc_grid_create(C.byref(desc), C.byref(h)) == -1           # |g| must be < 1
    P["g"] = [0.0]; P["density"] = np.array([1, 1, 1, -1, 1, 1, 1, 1], np.float32)
    desc, keep = soc.make_desc(**P)
    assert L.soc_grid_create(C.byref(desc), C.byref(h)) == -1           # negative density
    assert b"density" in L.soc_last_error()
    ms = C.c_float()
    assert L.soc_probe_throughput(9, 1 << 20, 1000, C.byref(ms)) == -1
    assert L.soc_simulate_frequency(None, 0, None, 1, 1, 1.0, None, None, 0, None) == -1
    assert L.soc_update_temperatures(None, None, 1.0, None, 2, 1.0, 2.0, None, None) == -1
    assert L.soc_update_temperatures_ali_static(None, None, None, None, 1.0, None, 2, 1.0, 2.0, None, None) == -1
    assert b"NULL" in L.soc_last_error()                                 # refused before any device call
    assert L.soc_launch_count() == 0
    assert L.soc_release_cached_memory() == 0                            # nothing cached, no device touched
    assert L.soc_version().startswith(b"soc_b200")


def test_no_cpu_fallback_in_the_product():
    """The package never imports the oracle, and the binding raises when the library is missing."""
    pkg = os.path.join(ROOT, "paper_1812_06632_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|oracle[/.]|soc_oracle", text), f
    from paper_1812_06632_b200 import soc
    saved, soc._lib, soc.LIB_PATH = (soc._lib, soc.LIB_PATH), None, os.path.join(pkg, "does_not_exist.so")
    try:
        with pytest.raises(soc.SocError):
            soc.load()
    finally:
        soc._lib, soc.LIB_PATH = saved


# ------------------------------------------------------------------------------------------------ multi-GPU plan
@pytest.mark.parametrize("world", [1, 2, 3, 8])
@pytest.mark.parametrize("n", [0, 1, 7, 1000, 10_000_019])
def test_strong_plan_covers_every_package_once(world, n):
    from paper_1812_06632_b200 import dist
    shards = [dist.plan("strong", r, world, n, 5) for r in range(world)]
    assert shards[0].pkg_begin == 0 and sum(s.pkg_count for s in shards) == n
    for a, b in zip(shards, shards[1:]):
        assert a.pkg_begin + a.pkg_count == b.pkg_begin
    assert max(s.pkg_count for s in shards) - min(s.pkg_count for s in shards) <= 1
    assert all(s.seed == 5 and s.mean_scale == 1.0 for s in shards)


def test_weak_plan_is_independent_realisations():
    from paper_1812_06632_b200 import dist
    shards = [dist.plan("weak", r, 4, 1000, 11) for r in range(4)]
    assert [s.seed for s in shards] == [11, 12, 13, 14]
    assert all(s.pkg_begin == 0 and s.pkg_count == 1000 and s.mean_scale == 0.25 for s in shards)
    with pytest.raises(ValueError):
        dist.plan("weak", 4, 4, 10, 1)
    with pytest.raises(ValueError):
        dist.plan("ring", 0, 4, 10, 1)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, mode, out_dir):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as td
    import oracle
    from paper_1812_06632_b200 import dist, inputs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    td.init_process_group("gloo", rank=rank, world_size=world)
    P = inputs.make_config("2", n=8, n_packages=4000)
    og = oracle.Grid(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child)
    sh = dist.plan(mode, rank, world, P.n_packages, 3)
    A, res, _, _ = oracle.simulate(og, P.kabs[0], P.ksca[0], P.g[0], 0, P.sources(0), P.n_packages, sh.seed, 1.0,
                                   sh.pkg_begin, sh.pkg_count)
    t = torch.from_numpy(A.copy())
    dist.combine(t, sh)
    np.save(os.path.join(out_dir, f"{mode}_{rank}.npy"), t.numpy())
    td.destroy_process_group()


@pytest.mark.parametrize("mode", ["strong", "weak"])
def test_world_size_2_gloo_all_reduce(mode, tmp_path):
    """Two processes over gloo: the combined per-cell array equals what one process computes alone."""
    import torch.multiprocessing as mp
    import oracle
    from paper_1812_06632_b200 import inputs
    port = _free_port()
    mp.spawn(_worker, args=(2, port, mode, str(tmp_path)), nprocs=2, join=True)
    a0, a1 = np.load(tmp_path / f"{mode}_0.npy"), np.load(tmp_path / f"{mode}_1.npy")
    assert np.array_equal(a0, a1)                                     # every rank holds the combined field
    P = inputs.make_config("2", n=8, n_packages=4000)
    og = oracle.Grid(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child)
    sim = lambda seed: oracle.simulate(og, P.kabs[0], P.ksca[0], P.g[0], 0, P.sources(0), P.n_packages, seed)[0]   # noqa: E731
    if mode == "strong":      # same seed, ids split: the single-process result up to the order of additions
        assert np.allclose(a0, sim(3), rtol=1e-12, atol=0)
    else:                     # seeds 3 and 4: the mean of two realisations
        assert np.allclose(a0, 0.5 * (sim(3) + sim(4)), rtol=1e-12, atol=0)


def _bench_worker(rank, world, port, mode, out_dir):
    """The distributed bookkeeping of bench.py's run_ours (init -> plan -> per-rank pass -> combine -> job_totals) over
    gloo, with the per-rank pass done by the oracle instead of the CUDA library (no GPU here)."""
    sys.path.insert(0, ROOT)
    import json
    import torch
    import torch.distributed as td
    import oracle
    from paper_1812_06632_b200 import dist, inputs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init("gloo", rank, world)
    P = inputs.make_config("3", n=8, n_packages=3000, n_freq=3)
    og = oracle.Grid(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child)
    sh = dist.plan(mode, rank, world, P.n_packages, P.seed)
    w = oracle.trapezoid_weights(P.freq_hz)
    A = np.zeros(P.n_total)
    steps = 0
    for f in range(P.n_freq):
        _, res, _, _ = oracle.simulate(og, P.kabs[f], P.ksca[f], P.g[f], f, P.sources(f), P.n_packages, sh.seed, w[f],
                                       sh.pkg_begin, sh.pkg_count, absorbed=A)
        steps += res.cell_steps
    t = torch.from_numpy(A)
    dist.combine(t, sh)
    job = dist.job_totals(step_ms=10.0 * (rank + 1), cell_steps=steps, launches=P.n_freq + 1, world=world)
    with open(os.path.join(out_dir, f"job_{mode}_{rank}.json"), "w") as fh:
        json.dump(dict(job=job, my_steps=steps, sum=float(t.sum())), fh)
    td.destroy_process_group()


@pytest.mark.parametrize("mode", ["strong", "weak"])
def test_bench_job_bookkeeping_world_size_2_gloo(mode, tmp_path):
    """time = MAX over ranks, cell-steps and launches = SUM over ranks, value = all cell-steps / that time; strong: the
    ranks' steps add up to the single-process count, weak: each rank does the full count."""
    import json
    import torch.multiprocessing as mp
    import oracle
    from paper_1812_06632_b200 import inputs
    mp.spawn(_bench_worker, args=(2, _free_port(), mode, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"job_{mode}_{k}.json")) for k in range(2)]
    assert r[0]["job"] == r[1]["job"]                                  # every rank holds the job totals
    job = r[0]["job"]
    assert job["step_ms"] == 20.0 and job["launches"] == 8
    assert job["cell_steps"] == r[0]["my_steps"] + r[1]["my_steps"]
    assert job["value"] == pytest.approx(job["cell_steps"] / 20e-3, rel=1e-12)
    assert r[0]["sum"] == pytest.approx(r[1]["sum"], rel=1e-14)
    P = inputs.make_config("3", n=8, n_packages=3000, n_freq=3)
    og = oracle.Grid(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child)
    full = sum(oracle.simulate(og, P.kabs[f], P.ksca[f], P.g[f], f, P.sources(f), P.n_packages, P.seed)[1].cell_steps
               for f in range(P.n_freq))
    if mode == "strong":
        assert job["cell_steps"] == full
    else:
        assert r[0]["my_steps"] == full and job["cell_steps"] > 1.9 * full


def test_bench_refuses_a_rank_count_it_cannot_serve():
    """`bench.py --gpus 2` with no launcher and fewer than 2 CUDA devices must fail loudly, not bench one GPU."""
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1"],
                         capture_output=True, text=True, timeout=600, env=env)
    assert out.returncode != 0 and "CUDA device" in (out.stderr + out.stdout)
    assert not [ln for ln in out.stdout.splitlines() if ln.startswith("{")]


def test_bench_reads_dram_traffic_from_the_newest_capture(tmp_path, monkeypatch):
    import importlib.util
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    b = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(b)
    (tmp_path / "profiles").mkdir()
    (tmp_path / "profiles" / "r01_ncu_dram_traffic.csv").write_text(
        "config,kernel,cell_steps,dram_read_bytes,dram_write_bytes,source\n5,k,100,900,100,old.txt\n")
    (tmp_path / "profiles" / "r02_ncu_dram_traffic.csv").write_text(
        "config,kernel,cell_steps,dram_read_bytes,dram_write_bytes,weight,source\n5,k,100,1500,500,1,new.txt\n5,k,100,500,500,1,new.txt\n")
    monkeypatch.setattr(b, "ROOT", str(tmp_path))
    t = b.ncu_traffic("5")
    assert t["bytes_per_cell_step"] == 15.0 and "r02_ncu_dram_traffic.csv" in t["source"] and "new.txt" in t["source"]
    assert b.ncu_traffic("3") is None


def test_bench_reference_arm_prints_the_contract_line():
    """bench.py --impl reference runs the oracle on the host cores and prints ONE JSON line with the keys the
    driver reads (no GPU involved)."""
    import json
    import subprocess
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["impl"] == "reference" and d["value"] > 0 and d["unit"] == "cell-steps/s" and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in d["config"]
