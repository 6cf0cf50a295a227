"""CPU-side checks of the product: the C-ABI library builds, loads and exports every
symbol include/cm.h declares (no compute calls without a GPU), the register DFT blocks
are right (compiled for the host), and the shared-memory exchange layouts are free of
bank conflicts."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    import paper_2301_06763_b200 as pkg
    so = pkg.build()
    L = ctypes.CDLL(so)
    hdr = open(os.path.join(ROOT, "include", "cm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(cm_[a-z_A-Z0-9]+)\s*\(", hdr)))
    assert len(declared) >= 10
    for name in declared:
        assert hasattr(L, name), f"{name} declared in cm.h but not exported"
    assert sorted(pkg.EXPORTS) == declared
    assert pkg.lib().cm_error_string(pkg.CM_ENOTREADY).decode().startswith("cm_green_precompute")


def test_argument_validation_needs_no_gpu():
    import paper_2301_06763_b200 as pkg
    for kw in [dict(N=26, levels=2, dx0=1.0), dict(N=12, levels=2, dx0=1.0), dict(N=520, levels=2, dx0=1.0), dict(N=16, levels=2, dx0=-1.0), dict(N=16, levels=2, dx0=1.0, refinement=4)]:
        with pytest.raises(pkg.CMError) as ei:
            pkg.cm_plan_create(**kw)
        assert ei.value.code == pkg.CM_EINVAL
    assert pkg.cm_slot_to_freq(16, 0) == 0 and pkg.cm_slot_to_freq(16, 16) == 1
    for N in (16, 64, 256):
        f = sorted(pkg.cm_slot_to_freq(N, s) for s in range(2 * N))
        assert f == list(range(2 * N))


def test_product_never_touches_the_oracle():
    """The product path must not import, link or execute anything under oracle/."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2301_06763_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2301_06763_b200" not in txt and "libcm.so" not in txt


def test_register_dft_blocks_on_host(tmp_path):
    exe = tmp_path / "hfb"
    subprocess.run(["g++", "-std=c++17", "-O1", "-o", str(exe), os.path.join(ROOT, "tests", "host_fft_blocks.cpp")],
                   check=True)
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout


def _conflict_degree(addrs_complex):
    """16-byte accesses: hardware serves a warp in quarter-warps of 8 lanes; degree = max
    number of distinct 128-byte rows hit by the same 16-byte column within a quarter."""
    worst = 1
    a = np.asarray(addrs_complex)
    for q in range(0, 32, 8):
        cols = {}
        for x in a[q:q + 8]:
            cols.setdefault(x % 8, set()).add(x // 8)
        worst = max(worst, max(len(v) for v in cols.values()))
    return worst


@pytest.mark.parametrize("T", [2, 4, 8, 16])
def test_exchange_layouts_are_conflict_free(T):
    """Mirrors LayBatch / LayRow of csrc/cm_kernels.cuh (values parsed from the source)."""
    src = open(os.path.join(ROOT, "paper_2301_06763_b200", "csrc", "cm_kernels.cuh")).read()
    assert "static constexpr int PS = 16 * T + 1;" in src and "static constexpr int RS = T + 1;" in src
    assert "16 * (T + 1) + (T == 4 ? 4 : (T == 2 ? 2 : 0))" in src
    lanes = np.arange(32)
    # batch-fastest: px = lane & 7, j = (lane >> 3) % T, g = lane // (8 T)
    RS, PS = T, 16 * T + 1
    px, j, g = lanes & 7, (lanes >> 3) % T, lanes // (8 * T)
    pen = (g * 8 + px) * PS
    for k1 in range(16):
        assert _conflict_degree(pen + k1 * RS + j) == 1                       # stage-1 side
    for cc in range(16 // T):
        for jj in range(T):
            assert _conflict_degree(pen + (cc * T + j) * RS + jj) == 1        # stage-2 side
    # j-fastest: j = lane % T, row = lane // T
    RS, PS = T + 1, 16 * (T + 1) + (4 if T == 4 else (2 if T == 2 else 0))
    j, row = lanes % T, lanes // T
    for k1 in range(16):
        assert _conflict_degree(row * PS + k1 * RS + j) == 1
    for cc in range(16 // T):
        for jj in range(T):
            assert _conflict_degree(row * PS + (cc * T + j) * RS + jj) == 1


# ------------------------------------------------------------------ multi-rank host logic (replicas only), CPU, gloo
def _rank_main(rank, world, port, out_dir):
    import json
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)

    def all_reduce_max(x):
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slower replica
    agg = bench.aggregate_over_ranks(ms_local, cells_per_rank=1000, world=world, all_reduce_max=all_reduce_max)
    assert bench.dist_env() == (rank, world, rank)
    bench.ensure_world(world, [])                      # consistent: returns
    with open(os.path.join(out_dir, f"rank{rank}.json"), "w") as f:
        json.dump(agg, f)
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_over_two_gloo_ranks(tmp_path):
    """bench.py --gpus N = N independent replicas: step time = max over ranks, value = the units all
    ranks processed per that time.  Two CPU processes over gloo on 127.0.0.1."""
    import json
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    mp.spawn(_rank_main, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        agg = json.load(open(tmp_path / f"rank{r}.json"))
        assert agg["ms_per_step"] == 15.0                               # the slower rank decides
        assert abs(agg["value"] - 2 * 1000 / 15e-3) < 1e-6
        assert abs(agg["solves_per_s"] - 2 / 15e-3) < 1e-9


def test_gpus_flag_must_match_world_size(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("WORLD_SIZE", "2")
    with pytest.raises(SystemExit):
        bench.ensure_world(8, [])
    bench.ensure_world(2, [])
    monkeypatch.delenv("WORLD_SIZE")
    bench.ensure_world(1, [])                          # single process, nothing to do
    assert bench.aggregate_over_ranks(4.0, 100, 1)["value"] == 100 / 4e-3


def test_reference_arm_runs_on_rank_zero_only(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")
    bench.run_reference(argparse.Namespace(config=1, steps=1, warmup=0, gpus=2))
    assert capsys.readouterr().out == ""
