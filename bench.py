#!/usr/bin/env python
"""Benchmark of the NOLSM hot path (arXiv 2205.12182) on B200.

One "step" = one pass of the whole hot path (assemble, gather, Schulz
inverse, spectral scaling, Newton-Schulz sign with fused convergence test, D columns, scatter, energy)
over one synthetic system. Default workload: BASELINE.json configs[2] (32,768 atoms, 13 basis functions
per atom, periodic, r_c = 6 A, FP16 operands / FP32 accumulate), the config the headline metric is
quoted on. Inputs are seeded and synthetic (workloads/synthetic.py); they are >> L2 (8 GB of block-CSR
values), so no L2 flush is needed between timed steps.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--atoms A] [--impl reference]

Prints ONE JSON line (rank 0). `value` is whole-job submatrices/s with inputs resident in HBM; the
tensor TFLOP/s (2 n^3 per executed GEMM) and the roofline fraction of the dominant
kernel are in `tensor_tflops` and `roofline`. `--impl reference` times the FP64 CPU oracle (oracle/)
on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

NOMINAL_FP16_TFLOPS = 2250.0
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {k: float(d[k]) for k in FALLBACK_PEAKS if k in d} | {"source": "measured"}
    return dict(FALLBACK_PEAKS, source="fallback")


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(system, atoms):
    """Times the oracle as it stands on the listed atoms. Returns (seconds, n_submatrices)."""
    from oracle import nolsm_oracle as orc
    from workloads import MAT_H, MAT_S
    need = np.unique(np.concatenate([system.col_idx[system.row_ptr[a]:system.row_ptr[a + 1]] for a in atoms]))
    sub = system.restrict(need)
    Hs, Ss = sub.fill_np(MAT_H), sub.fill_np(MAT_S)
    blk = orc.block_offsets(sub.atom_nb, sub.row_ptr, sub.col_idx)
    local = np.searchsorted(sub.meta["parent_atoms"], atoms)
    t0 = time.perf_counter()
    for la in local:
        orc.atom_result(int(la), sub.atom_nb, sub.row_ptr, sub.col_idx, blk, Hs, Ss, system.mu)
    return time.perf_counter() - t0, len(atoms)


def blas_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return int(max(n)) if n else 1
    except Exception:
        return os.cpu_count() or 1


def max_over_ranks(value: float, world: int, device=None) -> float:
    """The slowest rank's time decides (replicas run side by side): all-reduce MAX over the process group."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replicas_value(units_per_rank: int, world: int, seconds: float) -> float:
    """Whole-job throughput of `world` independent replicas that each process `units_per_rank` units (weak scaling)."""
    return world * units_per_rank / seconds


def workload_label(name, n_atoms):
    return name if n_atoms is None else f"{name}@{n_atoms}"


def run_reference(args, system):
    """--impl reference: the oracle, unmodified, on the host cores; each step = a bounded sample."""
    rng = np.random.default_rng(1234)
    per_step = args.ref_sample
    times = []
    for it in range(args.warmup + args.steps):
        atoms = np.sort(rng.choice(system.n_atoms, per_step, replace=False))
        dt, n = oracle_sample(system, atoms)
        if it >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    val = per_step / (ms * 1e-3)
    line = {"impl": "reference", "metric": "submatrices_per_s", "value": val, "unit": "submatrices/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_label(args.workload, args.atoms), "atoms": system.n_atoms,
                       "sample": f"{per_step} seeded-random submatrices per step"},
            "cpu_baseline": {"value": val, "unit": "submatrices/s", "cores": blas_threads(), "kind": "oracle",
                             "sample": f"{per_step} seeded-random submatrices per step, {args.steps} steps"},
            "e2e": {"value": val, "unit": "submatrices/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="nolsm", choices=["nolsm", "reference"])
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--atoms", type=int, default=None, help="override the atom count (same density/basis)")
    ap.add_argument("--profile-every", type=int, default=16)
    ap.add_argument("--cpu-sample", type=int, default=12, help="submatrices for the cpu_baseline leg (0 = skip)")
    ap.add_argument("--ref-sample", type=int, default=4)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--combine", type=int, default=0, choices=[0, 1, 2],
                    help="submatrix combination of the timed path (0 = one submatrix per atom, BASELINE.json's configs)")
    ap.add_argument("--no-combine-leg", action="store_true", help="skip the extra combine = 1 / 2 measurements")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from workloads import MAT_H, MAT_S, make_system
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, make_system(args.workload, n_atoms=args.atoms))
        return

    import torch
    import torch.distributed as dist
    from paper_2205_12182_b200 import Nolsm

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    # ---- synthetic inputs, resident in HBM (replicas: every rank evaluates its own copy of the system;
    #      the path has no exchange step -- DESIGN.md "Multi-GPU") ----
    system = make_system(args.workload, n_atoms=args.atoms)
    Hv = system.fill_torch(MAT_H, dev)
    Sv = system.fill_torch(MAT_S, dev)
    nb = torch.from_numpy(system.atom_nb).to(dev)
    rp = torch.from_numpy(system.row_ptr).to(dev)
    ci = torch.from_numpy(system.col_idx).to(dev)
    D = torch.empty_like(Hv)
    stream = torch.cuda.current_stream().cuda_stream
    ctx = Nolsm(local_rank, profile_every=args.profile_every, combine=args.combine)

    def step():
        ctx.assemble(nb, rp, ci, Hv, Sv, stream=stream)
        ctx.density_matrix(system.mu, D, stream=stream)
        return ctx.energy(strict=False)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    prof_acc = None
    ctr_acc = None
    e0.record()
    for _ in range(args.steps):
        E = step()
        pr = ctx.profile()
        prof_acc = pr if prof_acc is None else {k: prof_acc[k] + pr[k] for k in pr}
        ct = ctx.engine_counters()
        if ctr_acc is None:
            ctr_acc = ct
        else:
            for k in ("kernel_ms", "tiles", "sched_idle_ms", "sched_busy_ms", "overshoots"):
                ctr_acc[k] += ct[k]
            for kind, v in ct["side"].items():
                acc = ctr_acc["side"].setdefault(kind, {"busy_ms": 0.0, "bytes": 0.0, "tasks": 0.0})
                for kk in v:
                    acc[kk] += v[kk]
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_step = max_over_ranks(e0.elapsed_time(e1), world, dev) / args.steps
    stats = ctx.stats()

    # ---- the same workload with submatrix combination (Eq. 9 / Eq. 10): fewer, larger
    #      submatrices serve the same atoms; reported beside the headline, which stays one submatrix per atom ----
    combined = None
    if not args.no_combine_leg and args.combine == 0:
        combined = {}
        for mode in (1, 2):
            cx = Nolsm(local_rank, combine=mode)

            def step_c():
                cx.assemble(nb, rp, ci, Hv, Sv, stream=stream)
                cx.density_matrix(system.mu, D, stream=stream)
                return cx.energy(strict=False)
            step_c()
            barrier()
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record()
            Ec = step_c()
            c1.record()
            barrier()
            ms_c = max_over_ranks(c0.elapsed_time(c1), world, dev)
            sc, pc = cx.stats(), cx.profile()
            combined["eq9" if mode == 1 else "eq10"] = {
                "atoms_per_s": replicas_value(system.n_atoms, world, ms_c * 1e-3), "ms_per_step": ms_c,
                "submatrices": sc["n_units"], "dim_mean": sc["dim_mean"], "dim_max": sc["dim_max"],
                "gemms_per_submatrix": sc["gemms_executed"] / max(sc["n_units"], 1),
                "flops_useful_per_step": sc["flops_useful"], "kernel_ms": pc["gemm_ms"],
                "kernel_tflops_useful": pc["gemm_flops_useful"] / max(pc["gemm_ms"], 1e-9) / 1e9,
                "kernel_tflops_padded": pc["gemm_flops_padded"] / max(pc["gemm_ms"], 1e-9) / 1e9,
                "e_elec": Ec, "n_notspd": sc["n_notspd"], "n_noconv": sc["n_noconv"]}
            cx.destroy()

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of the inputs and D2H of D inside ----
    e2e = None
    if not args.no_e2e:
        hH, hS = Hv.cpu().pin_memory(), Sv.cpu().pin_memory()
        hD = torch.empty(Hv.shape[0], dtype=torch.float64).pin_memory()
        h_nb, h_rp, h_ci = system.atom_nb, system.row_ptr, system.col_idx
        ctx2 = Nolsm(local_rank)
        k_e2e = max(1, min(args.steps, 2))

        def step_host():
            ctx2.assemble(h_nb, h_rp, h_ci, hH, hS, stream=stream)
            ctx2.density_matrix(system.mu, hD, stream=stream)
            return ctx2.energy(strict=False)
        step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            step_host()
        torch.cuda.synchronize()
        dt_e2e = max_over_ranks((time.perf_counter() - t0) / k_e2e, world, dev)
        h2d = hH.numel() * 8 * 2 + h_nb.nbytes + h_rp.nbytes + h_ci.nbytes
        d2h = hD.numel() * 8 + 8
        e2e = {"value": replicas_value(system.n_atoms, world, dt_e2e), "unit": "submatrices/s",
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * dt_e2e}
        ctx2.destroy()
        del hH, hS, hD

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    value = replicas_value(system.n_atoms, world, ms_step * 1e-3)
    tflops = world * stats["flops_useful"] / (ms_step * 1e-3) / 1e12
    # dominant kernel. Persistent engine: ONE launch of nolsm_persist_kernel per step runs a1-a7; its duration
    # comes from CUDA events recorded on the launching stream (nolsm_get_profile). Round engine: the grouped
    # GEMM launches of the sampled rounds.
    persistent = bool(ctr_acc and ctr_acc["persistent"])
    gemm_tf = prof_acc["gemm_flops_useful"] / max(prof_acc["gemm_ms"], 1e-9) / 1e9
    gemm_tf_padded = prof_acc["gemm_flops_padded"] / max(prof_acc["gemm_ms"], 1e-9) / 1e9
    sampled_ms = prof_acc["gemm_ms"] + prof_acc["gather_ms"] + prof_acc["dcols_ms"] + prof_acc["other_ms"]
    # DRAM traffic of the kernel from the committed ncu --set full capture (profiles/): measured per submatrix on a
    # 1024-submatrix launch of the same workload, scaled to the submatrices of one launch here
    traffic, traffic_note = None, None
    tp = os.path.join(ROOT, "profiles", "gemm_traffic.json")
    if os.path.exists(tp) and args.workload == "cfg2":
        with open(tp) as f:
            tj = json.load(f)
        traffic = tj.get("dram_bytes_per_submatrix", 0.0) * system.n_atoms or None
        traffic_note = tj.get("capture")
    roofline = {"bound": "tensor", "kernel": "nolsm_persist_kernel" if persistent else "gemm2_round_kernel",
                "achieved": gemm_tf, "peak": peaks["bf16_tflops_sustained"],
                "unit": "TFLOP/s", "frac": gemm_tf / peaks["bf16_tflops_sustained"], "traffic": traffic,
                "peak_source": peaks["source"] + " bf16_tflops_sustained (kernel timed inside a long step)",
                "achieved_padded": gemm_tf_padded, "avg_launch_us": 1e3 * prof_acc["gemm_ms"] / max(prof_acc["gemm_launches"], 1),
                "frac_of_burst": gemm_tf / peaks["bf16_tflops"], "frac_of_nominal_2250": gemm_tf / NOMINAL_FP16_TFLOPS,
                "traffic_source": traffic_note}
    if persistent:
        # share of the step spent inside the kernel (the rest is assemble: host index logic + uploads)
        roofline["share_of_step_time"] = prof_acc["gemm_ms"] / (ms_step * args.steps)
        groups = 2 * ctr_acc["pairs"]                     # one side group (4 warps) per CTA
        side = ctr_acc["side"]
        g, d = side.get("gather", {}), side.get("dcols", {})
        # gather / scatter run as side tasks of the same launch, concurrently with the GEMM pipeline: the rate is
        # algorithmic bytes / (busy time summed over the side groups / #groups), i.e. what the side groups would
        # sustain together if they all ran that task (HBM-bound work, reported against the measured copy bandwidth)
        hbm = {"gather_gbs": g.get("bytes", 0) / max(g.get("busy_ms", 0) / groups, 1e-9) / 1e6,
               "scatter_gbs": d.get("bytes", 0) / max(d.get("busy_ms", 0) / groups, 1e-9) / 1e6,
               "gather_busy_frac_of_side_groups": g.get("busy_ms", 0) / max(groups * prof_acc["gemm_ms"], 1e-9),
               "scatter_busy_frac_of_side_groups": d.get("busy_ms", 0) / max(groups * prof_acc["gemm_ms"], 1e-9),
               "how": "side tasks inside nolsm_persist_kernel; bytes / (sum of side-group busy time / side groups)",
               "peak_gbs": peaks["hbm_gbs"], "peak_source": peaks["source"]}
        engine = {"tiles": ctr_acc["tiles"], "sched_idle_frac": ctr_acc["sched_idle_ms"] / max(ctr_acc["pairs"] * prof_acc["gemm_ms"], 1e-9),
                  "slots": ctr_acc["slots"], "pairs": ctr_acc["pairs"]}
    else:
        roofline["share_of_sampled_kernel_time"] = prof_acc["gemm_ms"] / max(sampled_ms, 1e-9)
        hbm = {"gather_gbs": prof_acc["gather_bytes"] / max(prof_acc["gather_ms"], 1e-9) / 1e6,
               "scatter_gbs": prof_acc["dcols_bytes"] / max(prof_acc["dcols_ms"], 1e-9) / 1e6,
               "peak_gbs": peaks["hbm_gbs"], "peak_source": peaks["source"]}
        engine = None
    hbm["gather_frac"] = hbm["gather_gbs"] / peaks["hbm_gbs"]
    hbm["scatter_frac"] = hbm["scatter_gbs"] / peaks["hbm_gbs"]

    cpu = None
    if args.cpu_sample > 0:
        atoms = np.sort(np.random.default_rng(99).choice(system.n_atoms, args.cpu_sample, replace=False))
        dt, n = oracle_sample(system, atoms)
        cpu = {"value": n / dt, "unit": "submatrices/s", "cores": blas_threads(), "kind": "oracle",
               "sample": f"{n} seeded-random submatrices of {workload_label(args.workload, args.atoms)} in {dt:.1f} s",
               "host_cpu_count": os.cpu_count()}

    line = {"metric": "submatrices_per_s", "value": value, "unit": "submatrices/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16", "data": "synthetic",
            "config": {"workload": workload_label(args.workload, args.atoms), "atoms": system.n_atoms,
                       "basis_per_atom": sorted(set(int(x) for x in np.unique(system.atom_nb))), "n_basis": int(system.atom_nb.sum()),
                       "dim_mean": stats["dim_mean"], "dim_min": stats["dim_min"], "dim_max": stats["dim_max"],
                       "precision": "fp16 operands / fp32 accumulate", "gamma_S": system.gamma,
                       "parallelism": "replicas" if world > 1 else "single",
                       "combine": args.combine,
                       "value_counts": "atoms served per second (one submatrix per atom when combine = 0)",
                       "l2": "inputs (8 GB block-CSR) and workspace >> 126 MB L2; no flush needed"},
            "tensor_tflops": tflops, "pct_of_dense_fp16_peak": {"nominal_2250": 100 * tflops / NOMINAL_FP16_TFLOPS / world,
                                                                 "measured_burst": 100 * tflops / peaks["bf16_tflops"] / world,
                                                                 "measured_sustained": 100 * tflops / peaks["bf16_tflops_sustained"] / world},
            "flops_useful_per_step": stats["flops_useful"], "flops_padded_per_step": stats["flops_padded"],
            "gemms_per_submatrix": stats["gemms_executed"] / max(stats["n_units"], 1), "submatrices": stats["n_units"], "e_elec": E,
            "n_notspd": stats["n_notspd"], "n_noconv": stats["n_noconv"],
            "roofline": roofline, "hbm_kernels": hbm, "engine": engine, "combined": combined, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
            "gpu_launches": int(prof_acc["kernel_launches"]),
            "paper_context": "1.1 EFLOP/s FP16/FP32 on 4400 A100 (~257 TFLOP/s per GPU, ~80% of 312), other hardware"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
