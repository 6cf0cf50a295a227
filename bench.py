#!/usr/bin/env python
"""bench.py — nested-grid potential solves on B200 (and the oracle timed beside them).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is ONE whole hot path (steps a1-a8 of DESIGN.md: restriction cascade, the five
pruned FFT passes over every level's (full, hole) pair, prolongation + Eq. 14 sum) over
one seeded synthetic nested density field.  Default workload: BASELINE.json configs[4]
(10 levels x 256^3, the throughput-stress config; the largest one, and it fits one GPU).

Prints ONE JSON line (rank 0).  `value` = cell-updates/s (levels * N^3 * solves / s) summed
over all ranks, inputs resident in HBM; `e2e` = the same metric through cm_potential_host
(pinned HOST buffers, both copies inside the timed region).  Multi-GPU = replicas only
(DESIGN.md §multi-GPU): every rank solves its own independent problem, no data-path
collective; time = max over ranks.

`--impl reference` times the ORACLE (oracle/, plain C on the host cores) on a bounded
sample of the same workload — see run_reference().
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "nested-grid potential cell-updates/s (fp64)"
UNIT = "cell-updates/s"
STAGES = ["restrict", "P1_x_fwd", "P2_y_fwd", "P3_z_conv", "P4_y_inv", "P5_x_inv", "prolong_sum"]


# --------------------------------------------------------------------------- byte models
def algorithmic_bytes(N: int, L: int) -> dict:
    """SURVEY.md §8(d) / DESIGN.md §5: bytes the pruned method itself must move, per LAUNCH
    (one launch of each pass kernel processes all 2L-1 fields).  K-hat is shared by every
    field, so it is counted once per launch."""
    F = 2 * L - 1
    h = (N + 1) * N * N           # half-spectrum pencils x N
    n3 = N ** 3
    return {
        "P1_x_fwd": F * (8 * n3 + 16 * h),
        "P2_y_fwd": F * (16 * h + 32 * h),
        "P3_z_conv": F * (32 * h + 32 * h) + 8 * (N + 1) ** 3,
        "P4_y_inv": F * (32 * h + 16 * h),
        "P5_x_inv": F * (16 * h + 8 * n3),
    }


def implemented_bytes(N: int, L: int) -> dict:
    """What the kernels as written move: one COMPLEX field per level
    (rho_full + i rho_hole), full 2N spectrum per axis, K-hat stored as (2N)^3 reals."""
    n3 = N ** 3
    hole_ring = (L - 1) * (N // 2 + 2) ** 3 * 8
    rc = (L - 1) * (N // 2) ** 3 * 8
    return {
        "P1_x_fwd": L * (8 * n3 + 32 * n3) + rc,
        "P2_y_fwd": L * (32 * n3 + 64 * n3),
        "P3_z_conv": L * (64 * n3 + 64 * n3) + 64 * n3,
        "P4_y_inv": L * (64 * n3 + 32 * n3),
        "P5_x_inv": L * (32 * n3 + 8 * n3) + hole_ring,
    }


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi sampled every 100 ms while the timed region runs (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); smax.append(float(f[1])); pw.append(float(f[2]))
                except ValueError:
                    continue
                for n, v in zip(names, f[3:7]):
                    if v == "Active":
                        reasons.add(n)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(smax), power_w_max=max(pw),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# --------------------------------------------------------------------------- distributed plumbing
def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def ensure_world(gpus: int, argv) -> None:
    """`--gpus N` must mean N ranks.  Under torchrun WORLD_SIZE says so; started as plain
    `python bench.py --gpus N` (N > 1) the script re-launches itself under torch.distributed.run with N ranks on
    127.0.0.1, so a replica run can never report n_gpus = 1.  A WORLD_SIZE that contradicts --gpus is an error."""
    world = int(os.environ.get("WORLD_SIZE", "0") or 0)
    if world == 0:
        if gpus <= 1:
            return
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
        os.execv(sys.executable, cmd)
    if world != max(gpus, 1):
        raise SystemExit(f"bench.py: --gpus {gpus} but WORLD_SIZE={world}: launch with --nproc-per-node {gpus}")


def aggregate_over_ranks(ms_local: float, cells_per_rank: int, world: int, all_reduce_max=None) -> dict:
    """Replicas only: every rank solves its own problem; the job's step time is the MAX over ranks,
    the job's value the units ALL ranks processed per that time.  `all_reduce_max(x) -> max over ranks` is the one
    collective (a timing reduction, not on the data path); None = single process."""
    ms = float(all_reduce_max(ms_local)) if (all_reduce_max is not None and world > 1) else float(ms_local)
    return {"ms_per_step": ms, "value": world * cells_per_rank / (ms * 1e-3), "solves_per_s": world / (ms * 1e-3)}


def load_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return {"hbm_gbs": float(d["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)"}
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)"}



# --------------------------------------------------------------------------- SASS counts and ncu traffic (evidence files)
def count_fp64_sass(kernel_substr: str):
    """fp64 arithmetic instructions (DADD/DMUL/DFMA) in the SASS of the kernel whose mangled name contains
    `kernel_substr`, counted live with cuobjdump from the libcm.so that is loaded (the tile loop is straight-line
    code, so this is the count per thread-tile plus a few set-up instructions).  None if cuobjdump is missing."""
    import shutil
    from paper_2301_06763_b200 import _build
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        return None
    try:
        out = subprocess.run([exe, "-sass", _build.SO], capture_output=True, text=True, timeout=120).stdout
    except Exception:
        return None
    counts, cur = {}, None
    for line in out.splitlines():
        t = line.strip()
        if t.startswith("Function :"):
            cur = t.split(":", 1)[1].strip()
        elif cur and kernel_substr in cur and "*/" in t:
            body = t.split("*/", 1)[1].strip().split()          # "/*0040*/   DADD R4, R2, R6 ;" -> ["DADD", ...]
            if body and body[0].startswith("@"):
                body = body[1:]
            op = body[0].split(".")[0] if body else ""
            if op in ("DADD", "DMUL", "DFMA"):
                c = counts.setdefault(cur, {"DADD": 0, "DMUL": 0, "DFMA": 0})
                c[op] += 1
    if not counts:
        return None
    name = sorted(counts)[0]
    c = counts[name]
    return {"kernel": name, "DADD": c["DADD"], "DMUL": c["DMUL"], "DFMA": c["DFMA"], "total": sum(c.values()),
            "how": "static count in the SASS of the loaded libcm.so (cuobjdump)"}


def ncu_row(config_id: int, kernel_substr: str):
    """The row of the committed ncu capture for this config and kernel, or None — never a hand-typed constant.
    profiles/r02_ncu_raw_config<id>.csv is `ncu -i <report> --page raw --csv --metrics ...` as it came out of ncu
    (first row names, second row units; profiles/r02_ncu_raw.md holds the commands)."""
    import csv
    path = os.path.join(ROOT, "profiles", f"r02_ncu_raw_config{config_id}.csv")
    if not os.path.exists(path):
        return None
    try:
        rows = list(csv.reader(open(path)))
        names, units = rows[0], rows[1]
        for r in rows[2:]:
            d = dict(zip(names, r))
            if kernel_substr in d.get("Kernel Name", ""):
                d["_units"] = dict(zip(names, units))
                return d
    except Exception:
        pass
    return None


_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def ncu_traffic(config_id: int, kernel_substr: str):
    """DRAM bytes (read + write) per launch of the kernel from that capture."""
    r = ncu_row(config_id, kernel_substr)
    if not r:
        return None
    try:
        tot = 0.0
        for k in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            tot += float(r[k].replace(",", "")) * _UNIT[r["_units"][k]]
        return tot
    except Exception:
        return None


# --------------------------------------------------------------------------- oracle timing (CPU)
def oracle_sample(cfg_id: int, rho, steps: int, warmup: int) -> dict:
    """Time the oracle AS IT STANDS on the host cores on a bounded sample of the workload.

    One sample step = ONE field convolution (one (level, full|hole) field of the 2L-1 the
    solve needs: oracle.field_fft, the oracle's own unpruned (2N)^3 FFT) at the workload's
    full N, cycling through the fields; the restriction cascade and the L-1 prolongations are
    timed once and added.  Estimated solve time = (2L-1) * mean field time + aux.
    For N <= 32 a step is the whole solve (oracle.solve, method="fft")."""
    import numpy as np
    import oracle
    import workloads
    L, N = rho.shape[0], rho.shape[1]
    dx0 = 2.0 / N
    cores = oracle.num_threads()
    if N <= 32:
        for _ in range(warmup):
            oracle.solve(rho, dx0, method="fft")
        t0 = time.perf_counter()
        for _ in range(steps):
            oracle.solve(rho, dx0, method="fft")
        t_solve = (time.perf_counter() - t0) / steps
        sample = f"{steps} whole solves (oracle.solve, method=fft) of config {cfg_id}"
        return dict(t_solve=t_solve, cores=cores, sample=sample, steps=steps, estimated=False)
    t0 = time.perf_counter()
    rhobar = oracle.restrict(rho)
    t_restrict = time.perf_counter() - t0
    ghat = oracle.green_hat(N)                       # one-time, like cm_green_precompute: untimed
    fields = [(l, h) for l in range(L) for h in ((False, True) if l < L - 1 else (False,))]
    times = []
    for s in range(warmup + steps):
        l, hole = fields[s % len(fields)]
        t0 = time.perf_counter()
        f = oracle.field_fft(rhobar[l], hole, 1.0, dx0 / (1 << l), ghat)
        dt = time.perf_counter() - t0
        if s >= warmup:
            times.append(dt)
    t0 = time.perf_counter()
    oracle.prolong(f)
    t_prolong = time.perf_counter() - t0
    t_field = sum(times) / len(times)
    t_solve = len(fields) * t_field + t_restrict + (L - 1) * t_prolong
    sample = (f"{steps} of the {len(fields)} field convolutions of one config-{cfg_id} solve at full N={N} "
              f"(oracle.field_fft, mean {t_field:.3f} s each) + restriction + prolongation timed once; "
              f"solve time = {len(fields)} x field + aux")
    return dict(t_solve=t_solve, cores=cores, sample=sample, steps=steps, t_field=t_field, estimated=True)


def run_reference(args) -> None:
    """`--impl reference`: the oracle, unmodified, on the host cores (rank 0 only)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    import workloads
    cfg = workloads.CONFIGS[args.config]
    N, L = cfg["N"], cfg["L"]
    rho = workloads.make_rho(args.config)
    r = oracle_sample(args.config, rho, args.steps, args.warmup)
    value = L * N ** 3 / r["t_solve"]
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * r["t_solve"],
        "estimated": bool(r.get("estimated", False)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "solves_per_s": 1.0 / r["t_solve"],
        "config": {"workload": f"config {args.config}: {cfg['name']}", "N": N, "levels": L,
                   "note": ("value and ms_per_step are ESTIMATES of one whole solve extrapolated from the sampled field "
                            "convolutions (see cpu_baseline.sample)") if r.get("estimated") else "whole solves timed"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
                         "estimated": bool(r.get("estimated", False))},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)



def measure_other_config(pkg, torch, workloads, cfg_id: int, steps: int, dev, stream, peak_gbs: float) -> dict:
    """Configs 3 and 4 (N = 64, 128) in compact form on the same run, so that the ">= 60 % at 64^3 and larger" bar
    is judged on driver-run numbers: whole-solve time through the CUDA graph and per-pass CUDA-event times."""
    cfg = workloads.CONFIGS[cfg_id]
    N, L = cfg["N"], cfg["L"]
    rho = torch.from_numpy(workloads.make_rho(cfg_id)).to(dev)
    phi = torch.empty_like(rho)
    plan = pkg.Plan(N, L, 2.0 / N)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    for _ in range(3):
        flush.fill_(1)
        plan.potential(rho, phi)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        flush.fill_(1)
        a.record(stream)
        plan.potential(rho, phi)
        b.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in evs) / steps
    acc = {k: 0.0 for k in STAGES}
    for _ in range(steps):
        flush.fill_(1)
        for k, v in plan.potential_profile(rho, phi).items():
            acc[k] += v / steps
    alg = algorithmic_bytes(N, L)
    out = {"workload": f"config {cfg_id}: {cfg['name']}", "N": N, "levels": L, "ms_per_step": ms,
           "cell_updates_per_s": L * N ** 3 / (ms * 1e-3), "l2": "256 MB flush buffer written between timed solves",
           "per_pass": {k: {"ms": round(acc[k], 5), "alg_GBs": round(alg[k] / (acc[k] * 1e-3) / 1e9, 1),
                            "frac": round(alg[k] / (acc[k] * 1e-3) / 1e9 / peak_gbs, 3)} for k in alg}}
    plan.close()
    del rho, phi, flush
    return out


# --------------------------------------------------------------------------- the CUDA arm
def run_ours(args) -> None:
    import numpy as np
    import torch
    import workloads
    import paper_2301_06763_b200 as pkg

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    pkg.lib()                                        # raises if libcm.so is not built
    cfg = workloads.CONFIGS[args.config]
    N, L = cfg["N"], cfg["L"]
    dx0 = 2.0 / N
    rho_np = workloads.make_rho(args.config)
    plan = pkg.Plan(N, L, dx0)
    rho = torch.from_numpy(rho_np).to(dev)
    phi = torch.empty_like(rho)
    cells = L * N ** 3
    launches_per_step = plan.kernel_launches
    stream = torch.cuda.current_stream(dev)

    # L2 hygiene: at N >= 128 one solve streams > 10x the 126 MB L2 through every pass, so
    # the inputs themselves evict it; below that, write a 256 MB buffer between timed steps.
    flush = None
    ws = plan.workspace_bytes
    if ws < (1 << 30):
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        if flush is not None:
            flush.fill_(1)
        plan.potential(rho, phi)

    # ---- region 1: K whole solves through cm_potential (CUDA-graph launch), device resident
    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    if flush is None:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        barrier()
        ms_total = e0.elapsed_time(e1)
    else:                                            # time each solve, excluding the flush kernel
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for a, b in evs:
            flush.fill_(1)
            a.record(stream)
            plan.potential(rho, phi)
            b.record(stream)
        barrier()
        ms_total = sum(a.elapsed_time(b) for a, b in evs)
    agg = aggregate_over_ranks(ms_total / args.steps, cells, world, max_over_ranks if dist is not None else None)
    ms_step = agg["ms_per_step"]

    # ---- region 2: the same K solves launched kernel by kernel with CUDA events between the
    # stages (cm_potential_profile) — per-kernel durations for the roofline, measured live.
    acc = {k: 0.0 for k in STAGES}
    for _ in range(args.steps):
        if flush is not None:
            flush.fill_(1)
        for k, v in plan.potential_profile(rho, phi).items():
            acc[k] += v
    stage_ms = {k: v / args.steps for k, v in acc.items()}
    clocks = sampler.stop() if rank == 0 else {}
    barrier()

    # ---- region 3: end to end through cm_potential_host (pinned host buffers, H2D + D2H timed)
    rho_h = torch.from_numpy(rho_np).pin_memory()
    phi_h = torch.empty_like(rho_h).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    plan.potential_host(rho_h, phi_h)
    barrier()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(e2e_steps):
        plan.potential_host(rho_h, phi_h)
    e1.record(stream)
    barrier()
    wall_e2e = (time.perf_counter() - t0) / e2e_steps * 1e3      # the call is synchronous: host clock counts too
    ms_e2e = max_over_ranks(max(e0.elapsed_time(e1) / e2e_steps, wall_e2e))

    # ---- region 4 (rank 0, extra): cm_acceleration on the potentials just computed
    accel = None
    if rank == 0:
        try:
            g = plan.acceleration(phi)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a0.record(stream)
            for _ in range(e2e_steps):
                if flush is not None:
                    flush.fill_(1)
                plan.acceleration(phi, g)
            a1.record(stream)
            torch.cuda.synchronize()
            ms_acc = a0.elapsed_time(a1) / e2e_steps
            if flush is not None:                      # take the flush writes out again
                f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                f0.record(stream)
                for _ in range(e2e_steps):
                    flush.fill_(1)
                f1.record(stream)
                torch.cuda.synchronize()
                ms_acc = max(ms_acc - f0.elapsed_time(f1) / e2e_steps, 1e-6)
            acc_bytes = cells * 32 + (L - 1) * N ** 3 * 9        # Phi read + g written per cell, + child means
            accel = {"ms": ms_acc, "cell_updates_per_s": cells / (ms_acc * 1e-3),
                     "algorithmic_bytes": acc_bytes, "alg_GBs": acc_bytes / (ms_acc * 1e-3) / 1e9,
                     "kernels": 2, "note": "cm_acceleration: six-point stencil with Eq. 3-6 ghosts and child means"}
            del g
        except Exception as e:                          # never lose the main line over the extra
            accel = {"error": str(e)}

    # ---- region 5 (rank 0, extra): the modified (dipole) method, Eq. B.1-B.2, where the doubled grid is supported
    modified = None
    if rank == 0 and N <= 128:
        try:
            pm = plan.potential_modified(rho)
            m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            m0.record(stream)
            for _ in range(e2e_steps):
                plan.potential_modified(rho, pm)
            m1.record(stream)
            torch.cuda.synchronize()
            ms_mod = m0.elapsed_time(m1) / e2e_steps
            modified = {"ms": ms_mod, "ratio_to_original": ms_mod / ms_step, "pairs": L - 1,
                        "note": "cm_potential_modified: one (2N)^3 convolution per pair, pruned to the fine grid's block on the way in and "
                                "decimated to the coarse cells on the way out (cm_expand.cuh), two pairs per complex solve"}

            def _time(fn, reps):
                fn()
                t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                t0.record(stream)
                for _ in range(reps):
                    fn()
                t1.record(stream)
                torch.cuda.synchronize()
                return t0.elapsed_time(t1) / reps

            if L > 2:                   # Eq. B.3-B.6: the quadrupled grid (4N <= 512)
                modified["triplets_ms"] = _time(lambda: plan.potential_modified_triplets(rho, pm), e2e_steps)
                modified["triplets_ratio_to_original"] = modified["triplets_ms"] / ms_step
            if N <= 32 and L > 2:       # Eq. B.7 in place of the quadrupled grid, and on its own (finest -> coarsest)
                modified["triplets_direct_ms"] = _time(lambda: plan.potential_modified_triplets(rho, pm, qdp_direct=True), 3)
                modified["direct_sum_ms"] = _time(lambda: plan.direct_sum(rho, L - 1, 0), 3)
            del pm
        except Exception as e:
            modified = {"error": str(e)}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel
    peaks = load_peaks()
    alg, impl = algorithmic_bytes(N, L), implemented_bytes(N, L)
    dom = max(alg.keys(), key=lambda k: stage_ms[k])
    achieved = alg[dom] / (stage_ms[dom] * 1e-3) / 1e9
    per_pass = {k: {"ms": round(stage_ms[k], 4),
                    "alg_GBs": round(alg[k] / (stage_ms[k] * 1e-3) / 1e9, 1) if stage_ms[k] > 0 else None,
                    "impl_GBs": round(impl[k] / (stage_ms[k] * 1e-3) / 1e9, 1) if stage_ms[k] > 0 else None}
                for k in alg}
    solve_alg_bytes = (2 * L - 1) * (16 * N ** 3 + 192 * (N + 1) * N * N) + 8 * (N + 1) ** 3
    roofline = {
        "bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
        "frac": achieved / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"],
        "algorithmic_bytes_per_launch": alg[dom], "implemented_bytes_per_launch": impl[dom],
        "kernel_ms": stage_ms[dom], "per_pass": per_pass,
        "aux_ms": {"restrict": round(stage_ms["restrict"], 4), "prolong_sum": round(stage_ms["prolong_sum"], 4),
                   "note": "a8 (prolongation + Eq. 14 sum) runs inside P5_x_inv, one launch per level"},
        "stage_sum_ms": sum(stage_ms.values()),
        "whole_solve_alg_GBs": solve_alg_bytes / (ms_step * 1e-3) / 1e9,
        "whole_solve_frac": solve_alg_bytes / (ms_step * 1e-3) / 1e9 / peaks["hbm_gbs"],
    }
    # P3 is bound on chip, not by HBM.  fp64 instructions per thread-tile: counted live in the SASS of
    # the loaded libcm.so; fp64 peak = SMs x 64 lanes/clk x the SM clock sampled DURING this run (64 lanes/clk/SM is
    # what a DFMA/DADD issue probe measured on this part, DESIGN.md §6 — not a data-sheet figure).
    T = N // 16
    kname = "k_z_conv_warp" if N == 128 else "k_z_conv_tma"
    sass = count_fp64_sass(f"{kname}ILi{T}E")
    row = ncu_row(args.config, "k_z_conv")
    if row and row.get("smsp__inst_executed_pipe_fp64.sum"):      # executed count from the ncu capture: exact, preferred
        per_tile = float(row["smsp__inst_executed_pipe_fp64.sum"].replace(",", "")) * 32 / (L * (2 * N) ** 2 * T)
        sass = {"total": per_tile, "how": "smsp__inst_executed_pipe_fp64.sum of the committed ncu capture / thread-tiles",
                "static_sass": sass}
    sm_mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0
    num_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    fp64_peak = num_sms * 64 * sm_mhz * 1e6
    if sass:
        lane_instr = L * (2 * N) ** 2 * T * sass["total"]
        roofline["p3_limits"] = {
            "fp64_instr_per_thread_tile": sass, "fp64_lane_instr_per_launch": lane_instr,
            "fp64_achieved_T_per_s": lane_instr / (stage_ms["P3_z_conv"] * 1e-3) / 1e12,
            "fp64_peak_T_per_s": fp64_peak / 1e12, "fp64_peak_how": f"{num_sms} SMs x 64 lanes/clk x {sm_mhz:.0f} MHz (sampled under load)",
            "fp64_frac": lane_instr / (stage_ms["P3_z_conv"] * 1e-3) / fp64_peak,
            "note": "P3 is co-limited by the fp64 pipe and the shared-memory data pipe (profiles/), both above its HBM time; "
                    "roofline.frac is against HBM as north_star asks"}
    roofline["measured_limiter"] = "fp64 pipe + shared-memory pipe (on chip)" if dom == "P3_z_conv" else "hbm"
    roofline["traffic"] = ncu_traffic(args.config, {"P1_x_fwd": "k_x_fwd", "P2_y_fwd": "k_y_fwd", "P3_z_conv": "k_z_conv",
                                                    "P4_y_inv": "k_y_inv", "P5_x_inv": "k_x_inv"}[dom])
    roofline["traffic_source"] = f"profiles/r02_ncu_raw_config{args.config}.csv (ncu --set full capture of this kernel)" if roofline["traffic"] else None

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        r = oracle_sample(args.config, rho_np, 2 if N > 32 else 3, 0)
        cpu = {"value": cells / r["t_solve"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
               "estimated": bool(r.get("estimated", False))}

    value = agg["value"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "solves_per_s": world / (ms_step * 1e-3),
        "config": {"workload": f"config {args.config}: {cfg['name']}", "N": N, "levels": L, "fields": 2 * L - 1,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": ("inputs larger than L2 (workspace %.1f GB streamed per solve)" % (ws / 1e9)) if flush is None
                         else "256 MB flush buffer written between timed solves",
                   "launch": "cm_potential -> cudaGraphLaunch of %d kernels" % launches_per_step},
        "clocks": clocks,
        "e2e": {"value": world * cells / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e,
                "h2d_bytes_per_step": rho_h.numel() * 8, "d2h_bytes_per_step": phi_h.numel() * 8,
                "api": "cm_potential_host (pinned host rho -> device -> solve -> pinned host phi; level pipeline for N >= 128)"},
        "gpu_launches": args.steps * launches_per_step,
        "roofline": roofline,
        "cpu_baseline": cpu,
        "acceleration": accel,
        "modified_method": modified,
    }
    if world == 1 and args.config == 5 and not args.no_other_configs:
        line["other_configs"] = {}
        for c in (3, 4):
            try:
                line["other_configs"][f"config{c}"] = measure_other_config(pkg, torch, workloads, c, 20, dev, stream, peaks["hbm_gbs"])
            except Exception as e:
                line["other_configs"][f"config{c}"] = {"error": str(e)}
    if args.cufft_ref and world == 1:
        plan.close()
        del rho, phi
        torch.cuda.empty_cache()
        line["cufft_dense_reference"] = cufft_dense_reference(N, L, torch)
    print(json.dumps(line), flush=True)
    plan.close()
    if dist is not None:
        dist.destroy_process_group()


def run_sharded(args) -> None:
    """`--shard-levels`: ONE solve of the config spread over the N ranks by levels (paper_2301_06763_b200/sharded.py,
    SURVEY.md §8e) — strong scaling, against the default mode's replicas.  Each rank holds and solves its own levels;
    the two neighbour exchanges (NCCL send/recv) are inside the timed region.  With N = 1 it times the three shard
    calls (no CUDA graph) against cm_potential.  Untested on more than one GPU in this repository's runs."""
    import torch
    import workloads
    import paper_2301_06763_b200 as pkg

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    else:                                            # a one-rank group so that the same code runs on one GPU
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1)
    cfg = workloads.CONFIGS[args.config]
    N, L = cfg["N"], cfg["L"]
    solver = pkg.ShardedSolver(N, L, 2.0 / N)
    lo, hi = solver.lo, solver.hi
    rho_own = torch.from_numpy(workloads.make_rho(args.config)[lo:hi].copy()).to(dev)
    phi_own = torch.empty_like(rho_own)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        solver.solve(rho_own, phi_own)
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        solver.solve(rho_own, phi_own)
    e1.record(stream)
    barrier()
    t = torch.tensor([e0.elapsed_time(e1) / args.steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item())
    clocks = sampler.stop() if rank == 0 else {}
    # kernels of this rank's solve: k_restrict per own level >= 1, P1..P4, one P5 per level, k_ring_box per neighbour
    launches = 0 if hi == lo else max(0, hi - max(lo, 1)) + 4 + (hi - lo) + int(lo > 0) + int(hi < L)
    if rank == 0:
        H, B = N // 2, N // 2 + 2
        print(json.dumps({
            "metric": METRIC, "value": L * N ** 3 / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "solves_per_s": 1.0 / (ms_step * 1e-3),
            "config": {"workload": f"config {args.config}: {cfg['name']}", "N": N, "levels": L, "fields": 2 * L - 1,
                       "parallelism": f"one solve, levels over {world} rank(s): {pkg.partition_levels(L, world)}",
                       "exchange_bytes_per_boundary": {"fine_to_coarse": 8 * H ** 3, "coarse_to_fine": 8 * B ** 3},
                       "l2": "inputs larger than L2" if N >= 128 else "not flushed (sharded mode is a scaling probe)",
                       "launch": "cm_shard_restrict / cm_shard_forward / cm_shard_finish, kernel by kernel"},
            "clocks": clocks, "e2e": None, "gpu_launches": args.steps * int(launches), "roofline": None, "cpu_baseline": None,
        }), flush=True)
    solver.close()
    dist.destroy_process_group()


def cufft_dense_reference(N: int, L: int, torch) -> dict:
    """Context only (--cufft-ref): the paper's own GPU scheme on this GPU — per field a dense
    zero-padded (2N)^3 cuFFT D2Z, a pointwise multiply and a Z2D, here through torch.fft; restriction,
    interpolation and assembly (host-side in the paper) are not included.  Never linked into libcm."""
    n = 2 * N
    rho = torch.rand(N, N, N, dtype=torch.float64, device="cuda")
    khat = torch.rand(n, n, n // 2 + 1, dtype=torch.float64, device="cuda")

    def field():
        pad = torch.zeros(n, n, n, dtype=torch.float64, device="cuda")
        pad[:N, :N, :N] = rho
        f = torch.fft.rfftn(pad)
        f *= khat
        return torch.fft.irfftn(f, s=(n, n, n))[:N, :N, :N]

    for _ in range(2):
        field()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(5):
        field()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 5
    return {"ms_per_field": ms, "ms_per_solve": (2 * L - 1) * ms, "fields": 2 * L - 1,
            "what": "torch.fft rfftn/irfftn (cuFFT) on the dense (2N)^3 + multiply, FFT part of the paper's scheme only"}


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)       # the paper's protocol: 20 full cycles
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the compact config-3 / config-4 lines")
    ap.add_argument("--cufft-ref", action="store_true", help="also time the paper's dense cuFFT scheme (context)")
    ap.add_argument("--shard-levels", action="store_true",
                    help="one solve spread over the ranks by levels (strong scaling) instead of one replica per rank")
    args = ap.parse_args()
    ensure_world(args.gpus, sys.argv[1:])
    if args.impl == "reference":
        run_reference(args)
    elif args.shard_levels:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
