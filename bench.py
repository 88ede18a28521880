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
                "power_w_max": max(pw) if pw else None, "power_w_median": float(np.median(pw)) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


_ORC = {}          # state shared with forked workers (copy-on-write): restricted system and its values


def _oracle_worker(chunk):
    """Oracle on a chunk of (restricted-system) atoms, one BLAS thread."""
    from oracle import nolsm_oracle as orc
    try:
        from threadpoolctl import threadpool_limits
        ctx = threadpool_limits(limits=1)
    except Exception:
        ctx = None
    t0 = time.perf_counter()
    for la in chunk:
        orc.atom_result(int(la), _ORC["nb"], _ORC["rp"], _ORC["ci"], _ORC["blk"], _ORC["H"], _ORC["S"], _ORC["mu"])
    if ctx is not None:
        ctx.restore_original_limits()
    return time.perf_counter() - t0


def oracle_sample(system, atoms, workers=None):
    """Times the oracle as it stands on the listed atoms: one worker process per host core, one BLAS thread each (the two
    symmetric eigendecompositions scale poorly with threads). Returns (wall seconds, n_submatrices, workers)."""
    import multiprocessing as mp
    from oracle import nolsm_oracle as orc
    from workloads import MAT_H, MAT_S
    workers = max(1, min(workers or (os.cpu_count() or 1), len(atoms)))
    need = np.unique(np.concatenate([system.col_idx[system.row_ptr[a]:system.row_ptr[a + 1]] for a in atoms]))
    sub = system.restrict(need)
    _ORC.update(nb=sub.atom_nb, rp=sub.row_ptr, ci=sub.col_idx, H=sub.fill_np(MAT_H), S=sub.fill_np(MAT_S), mu=system.mu)
    _ORC["blk"] = orc.block_offsets(sub.atom_nb, sub.row_ptr, sub.col_idx)
    local = np.searchsorted(sub.meta["parent_atoms"], atoms)
    chunks = [local[w::workers] for w in range(workers)]
    t0 = time.perf_counter()
    if workers == 1:
        _oracle_worker(chunks[0])
    else:
        with mp.get_context("fork").Pool(workers) as pool:
            pool.map(_oracle_worker, chunks)
    dt = time.perf_counter() - t0
    _ORC.clear()
    return dt, len(atoms), workers


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
    workers = os.cpu_count() or 1
    per_step = max(args.ref_sample, workers)
    times = []
    for it in range(args.warmup + args.steps):
        atoms = np.sort(rng.choice(system.n_atoms, per_step, replace=False))
        dt, n, workers = oracle_sample(system, atoms)
        if it >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    val = per_step / (ms * 1e-3)
    sample = f"{per_step} seeded-random submatrices per step, one single-threaded worker per core"
    line = {"impl": "reference", "metric": "submatrices_per_s", "value": val, "unit": "submatrices/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_label(args.workload, args.atoms), "atoms": system.n_atoms, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "submatrices/s", "cores": workers, "kind": "oracle",
                             "sample": f"{sample}, {args.steps} steps", "host_cpu_count": os.cpu_count()},
            "e2e": {"value": val, "unit": "submatrices/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def load_perf_table():
    """p(n) of Eq. 10 measured on B200 (`python bench.py --pn-sweep --out workloads/pn_b200.json`)."""
    p = os.path.join(ROOT, "workloads", "pn_b200.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        t = json.load(f)
    return [int(r["n"]) for r in t["table"]], [float(r["tflops"]) for r in t["table"]]


PN_SIZES = [("pn-5-5.0", 2048), ("pn-7-5.0", 2048), ("pn-6-6.0", 2048), ("pn-7-6.0", 2048), ("pn-8-6.0", 2048), ("pn-10-6.0", 2048),
            ("pn-11-6.0", 2048), ("pn-13-6.0", 2048), ("pn-16-6.0", 2048), ("pn-12-7.0", 2048), ("pn-14-7.0", 2048),
            ("pn-16-7.0", 1024), ("pn-13-8.0", 1024), ("pn-16-8.0", 1024), ("pn-14-8.5", 1024)]


def run_pn_sweep(args):
    """The multiplication rate of the engine against the matrix dimension: one periodic system per size, all
    of its submatrices of (nearly) one dimension; rate = 2 n^3 x GEMMs / kernel time with every product counted in full
    (what predicts the runtime of the matrix function on a submatrix of dimension n)."""
    import torch
    from paper_2205_12182_b200 import Nolsm
    from workloads import MAT_H, MAT_S, make_system
    dev = torch.device("cuda", 0)
    rows = []
    for name, n_atoms in PN_SIZES:
        system = make_system(name, n_atoms=n_atoms)
        Hv, Sv = system.fill_torch(MAT_H, dev), system.fill_torch(MAT_S, dev)
        nb, rp, ci = (torch.from_numpy(x).to(dev) for x in (system.atom_nb, system.row_ptr, system.col_idx))
        D = torch.empty_like(Hv)
        ctx = Nolsm(0)
        kms, fl, fu = 0.0, 0.0, 0.0
        for it in range(1 + args.steps):
            ctx.assemble(nb, rp, ci, Hv, Sv)
            ctx.density_matrix(system.mu, D)
            ctx.energy(strict=False)
            if it:
                st, pr = ctx.stats(), ctx.profile()
                kms += pr["gemm_ms"]; fl += st["flops_paper"]; fu += st["flops_useful"]
        rows.append({"workload": name, "atoms": system.n_atoms, "n": int(round(st["dim_mean"])), "dim_min": st["dim_min"], "dim_max": st["dim_max"],
                     "tflops": round(fl / kms / 1e9, 1), "tflops_executed": round(fu / kms / 1e9, 1),
                     "gemms_per_submatrix": round(st["gemms_executed"] / st["n_units"], 2), "kernel_ms": round(kms / args.steps, 2),
                     "n_noconv": st["n_noconv"], "n_notspd": st["n_notspd"]})
        print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
        ctx.destroy()
        del Hv, Sv, D
    rows.sort(key=lambda r: r["n"])
    out = {"what": "multiplication rate of the NOLSM engine on B200 against the submatrix dimension: p(n) of Eq. 10 (PAPER.md:L89-91)",
           "command": "python bench.py --pn-sweep --steps %d --out workloads/pn_b200.json" % args.steps,
           "rate": "2 n^3 x executed GEMMs (each counted in full) / kernel time, TFLOP/s; default options",
           "gpu": torch.cuda.get_device_name(0), "table": rows}
    text = json.dumps(out, indent=1)
    if args.out:
        with open(args.out, "w") as f:
            f.write(text + "\n")
    print(text)


def measure(ctx, arrays, system, D, stream, world, dev, steps=1, warm=1):
    """`warm` untimed and `steps` timed passes (assemble + density_matrix + energy) of one context; returns a summary."""
    import torch
    nb, rp, ci, Hv, Sv = arrays

    def step():
        ctx.assemble(nb, rp, ci, Hv, Sv, stream=stream)
        ctx.density_matrix(system.mu, D, stream=stream)
        return ctx.energy(strict=False)
    for _ in range(warm):
        step()
    torch.cuda.synchronize()
    c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kms = 0.0
    c0.record()
    for _ in range(steps):
        E = step()
        kms += ctx.profile()["gemm_ms"]
    c1.record()
    torch.cuda.synchronize()
    ms = max_over_ranks(c0.elapsed_time(c1), world, dev) / steps
    kms /= steps
    st = ctx.stats()
    peaks = load_peaks()
    tf = st["flops_useful"] / max(kms, 1e-9) / 1e9
    return {"atoms_per_s": replicas_value(system.n_atoms, world, ms * 1e-3), "ms_per_step": ms, "submatrices": st["n_units"],
            "dim_mean": st["dim_mean"], "dim_max": st["dim_max"], "gemms_per_submatrix": st["gemms_executed"] / max(st["n_units"], 1),
            "symmetric_gemms_per_submatrix": st["gemms_symmetric"] / max(st["n_units"], 1),
            "flops_useful_per_step": st["flops_useful"], "kernel_ms": kms, "kernel_tflops_useful": tf,
            "kernel_tflops_padded": st["flops_padded"] / max(kms, 1e-9) / 1e9,
            "kernel_tflops_paper_convention": st["flops_paper"] / max(kms, 1e-9) / 1e9,
            "frac_of_sustained_peak": tf / peaks["bf16_tflops_sustained"],
            "e_elec": E, "n_notspd": st["n_notspd"], "n_noconv": st["n_noconv"]}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="nolsm", choices=["nolsm", "reference"])
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--atoms", type=int, default=None, help="override the atom count (same density/basis)")
    ap.add_argument("--profile-every", type=int, default=16)
    ap.add_argument("--cpu-sample", type=int, default=-1, help="submatrices for the cpu_baseline leg (0 = skip, -1 = three per host core)")
    ap.add_argument("--ref-sample", type=int, default=4)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--combine", type=int, default=0, choices=[0, 1, 2],
                    help="submatrix combination of the timed path (0 = one submatrix per atom, BASELINE.json's configs)")
    ap.add_argument("--iteration", type=int, default=0, choices=[0, 1], help="0 = Eq. 6 as printed, 1 = symmetric (Loewdin) form")
    ap.add_argument("--symmetric-tiles", type=int, default=0, choices=[0, -1])
    ap.add_argument("--transposed-tiles", type=int, default=0, choices=[0, -1])
    ap.add_argument("--heavy-slots", type=int, default=0)
    ap.add_argument("--claim-lead", type=int, default=0)
    ap.add_argument("--no-extra-legs", "--no-combine-leg", action="store_true", dest="no_extra",
                    help="skip the variants / combination / other-config / side-task measurements")
    ap.add_argument("--pn-sweep", action="store_true", help="measure p(n) of Eq. 10 and print / write the table")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from workloads import MAT_H, MAT_S, make_system
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, make_system(args.workload, n_atoms=args.atoms))
        return
    if args.pn_sweep:
        if rank == 0:
            run_pn_sweep(args)
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
    arrays = (nb, rp, ci, Hv, Sv)
    D = torch.empty_like(Hv)
    stream = torch.cuda.current_stream().cuda_stream
    head_opts = dict(profile_every=args.profile_every, combine=args.combine, iteration=args.iteration,
                     symmetric_tiles=args.symmetric_tiles, heavy_slots=args.heavy_slots, claim_lead=args.claim_lead,
                     transposed_tiles=args.transposed_tiles)
    ctx = Nolsm(local_rank, **head_opts)
    perf_table = load_perf_table()
    if perf_table and args.combine == 2:
        ctx.set_perf_table(*perf_table)

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
            for k in ("kernel_ms", "tiles", "sched_idle_ms", "sched_busy_ms", "overshoots", "mma_wait_record_ms",
                      "mma_wait_accumulator_ms", "mma_kloop_ms", "sched_wait_ring_ms", "sched_wait_claim_point_ms", "power_steps_extra"):
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

    # ---- the HBM-bound side tasks timed alone: the same device code as inside the persistent kernel ----
    side_alone = None
    if not args.no_extra and args.combine == 0:
        try:
            g_ms, g_b = ctx.side_task_bandwidth(0, reps=2)
            s_ms, s_b = ctx.side_task_bandwidth(1, reps=2)
            side_alone = {"gather_gbs": g_b / g_ms / 1e6, "gather_ms": g_ms, "gather_bytes": g_b,
                          "scatter_gbs": s_b / s_ms / 1e6, "scatter_ms": s_ms, "scatter_bytes": s_b,
                          "how": "nolsm_side_task_bandwidth: k_side_gather / k_side_dcols over every submatrix of the workload, "
                                 "one 128-thread side group per CTA, CUDA events; algorithmic bytes / time"}
        except Exception as ex:                                   # diagnostics must not take the bench line down
            side_alone = {"error": str(ex)}
    ctx.destroy()

    # ---- the same workload with the other iteration form / tile mode, and with submatrix combination (Eq. 9 /
    #      Eq. 10): reported beside the headline, which stays one submatrix per atom with the default options ----
    variants, combined, others = None, None, None
    if not args.no_extra and args.combine == 0 and args.iteration == 0 and args.symmetric_tiles == 0:
        variants = {}
        for key, kw in (("eq6_every_tile_multiplied", dict(symmetric_tiles=-1)), ("lowdin_symmetric_form", dict(iteration=1))):
            cx = Nolsm(local_rank, **kw)
            variants[key] = measure(cx, arrays, system, D, stream, world, dev)
            cx.destroy()
        combined = {}
        for mode in (1, 2):
            cx = Nolsm(local_rank, combine=mode)
            if mode == 2 and perf_table:
                cx.set_perf_table(*perf_table)
            combined["eq9" if mode == 1 else "eq10"] = measure(cx, arrays, system, D, stream, world, dev)
            if mode == 2:
                combined["eq10"]["p_of_n"] = "workloads/pn_b200.json (measured, interpolated)" if perf_table else "tile-step model (no table)"
            cx.destroy()

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of the inputs and D2H of D inside ----
    e2e = None
    if not args.no_e2e:
        hH, hS = Hv.cpu().pin_memory(), Sv.cpu().pin_memory()
        hD = torch.empty(Hv.shape[0], dtype=torch.float64).pin_memory()
        h_nb, h_rp, h_ci = system.atom_nb, system.row_ptr, system.col_idx
        ctx2 = Nolsm(local_rank, **head_opts)
        if perf_table and args.combine == 2:
            ctx2.set_perf_table(*perf_table)
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

    # ---- the other BASELINE.json configs at full size, one timed step each (cfg4 streamed in four atom batches) ----
    if not args.no_extra and args.workload == "cfg2" and args.atoms is None and args.combine == 0:
        del Hv, Sv, D, arrays
        torch.cuda.empty_cache()
        others = {}
        for name in ("cfg1", "cfg3", "cfg4"):
            try:
                so = make_system(name)
                Ho, So = so.fill_torch(MAT_H, dev), so.fill_torch(MAT_S, dev)
                ao = tuple(torch.from_numpy(x).to(dev) for x in (so.atom_nb, so.row_ptr, so.col_idx)) + (Ho, So)
                Do = torch.empty_like(Ho)
                cx = Nolsm(local_rank)
                if name != "cfg4":
                    others[name] = measure(cx, ao, so, Do, stream, world, dev, steps=2 if name == "cfg1" else 1)
                    if name == "cfg1":
                        # chemical-potential search for half filling: trial mu per pass on the resident
                        # S_sub^-1 and A0 (nolsm_electron_counts) against one trial per pass
                        target = 0.5 * float(so.atom_nb.sum())
                        mu_search = {"target_electrons": target, "bracket": [-2.0, 2.0], "tol_n": 0.5}
                        for k in (1, 3, 7):
                            cm = Nolsm(local_rank, mu_trials=k)
                            cm.assemble(*ao, stream=stream)
                            torch.cuda.synchronize()
                            t0 = time.perf_counter()
                            mu_f, n_f, ev = cm.find_mu(target, -2.0, 2.0, Do, tol_n=0.5, tol_mu=1e-5, stream=stream)
                            torch.cuda.synchronize()
                            mu_search[f"trials_per_pass_{k}"] = {"mu": mu_f, "electrons": n_f, "trial_mu_evaluated": ev,
                                                                 "seconds": time.perf_counter() - t0}
                            cm.destroy()
                        others["cfg1"]["mu_search"] = mu_search
                else:
                    nbatch = 4
                    edges = [so.n_atoms * b // nbatch for b in range(nbatch + 1)]
                    cx.assemble(*ao, stream=stream)
                    cx.density_matrix_range(so.mu, edges[0], edges[1], Do, want_energy=True, stream=stream)    # warm
                    torch.cuda.synchronize()
                    c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    kms, fl, gem, Eo, ncv = 0.0, 0.0, 0, 0.0, 0
                    c0.record()
                    cx.assemble(*ao, stream=stream)
                    for b in range(nbatch):
                        Eo += cx.density_matrix_range(so.mu, edges[b], edges[b + 1], Do, want_energy=True, stream=stream)
                        stb = cx.stats()
                        kms += cx.profile()["gemm_ms"]; fl += stb["flops_useful"]; gem += stb["gemms_executed"]; ncv += stb["n_noconv"]
                    c1.record()
                    torch.cuda.synchronize()
                    ms = max_over_ranks(c0.elapsed_time(c1), world, dev)
                    tf = fl / max(kms, 1e-9) / 1e9
                    others[name] = {"atoms_per_s": replicas_value(so.n_atoms, world, ms * 1e-3), "ms_per_step": ms, "submatrices": so.n_atoms,
                                    "batches": nbatch, "dim_mean": stb["dim_mean"], "gemms_per_submatrix": gem / so.n_atoms,
                                    "flops_useful_per_step": fl, "kernel_ms": kms, "kernel_tflops_useful": tf,
                                    "frac_of_sustained_peak": tf / load_peaks()["bf16_tflops_sustained"], "e_elec": Eo, "n_noconv": ncv}
                cx.destroy()
                del Ho, So, Do, ao
                torch.cuda.empty_cache()
            except Exception as ex:
                others[name] = {"error": str(ex)}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    value = replicas_value(system.n_atoms, world, ms_step * 1e-3)
    tflops = world * stats["flops_useful"] / (ms_step * 1e-3) / 1e12
    # dominant kernel. Persistent engine: ONE launch of nolsm_persist_kernel per step runs a1-a7; its duration
    # comes from CUDA events recorded on the launching stream (nolsm_get_profile).
    persistent = bool(ctr_acc and ctr_acc["persistent"])
    gemm_tf = prof_acc["gemm_flops_useful"] / max(prof_acc["gemm_ms"], 1e-9) / 1e9
    gemm_tf_padded = prof_acc["gemm_flops_padded"] / max(prof_acc["gemm_ms"], 1e-9) / 1e9
    gemm_tf_paper = args.steps * stats["flops_paper"] / max(prof_acc["gemm_ms"], 1e-9) / 1e9
    sampled_ms = prof_acc["gemm_ms"] + prof_acc["gather_ms"] + prof_acc["dcols_ms"] + prof_acc["other_ms"]
    # DRAM traffic of the kernel: NOT measured in this run. It is the figure of the committed ncu --set full capture
    # (profiles/gemm_traffic.csv: per submatrix on a 1024-submatrix launch of the same workload), scaled to one launch here.
    traffic, traffic_note = None, None
    tp = os.path.join(ROOT, "profiles", "gemm_traffic.csv")
    if os.path.exists(tp) and args.workload == "cfg2":
        import csv
        with open(tp, newline="") as f:
            tj = {r[0]: r[1] for r in csv.reader(f) if len(r) == 2}
        traffic = float(tj.get("dram_bytes_per_submatrix", 0.0)) * system.n_atoms or None
        traffic_note = tj.get("capture")
    roofline = {"bound": "tensor", "kernel": "nolsm_persist_kernel" if persistent else "k_gemm_simt",
                "achieved": gemm_tf, "peak": peaks["bf16_tflops_sustained"],
                "unit": "TFLOP/s", "frac": gemm_tf / peaks["bf16_tflops_sustained"], "traffic": traffic,
                "traffic_measured_in_run": False, "traffic_source": traffic_note,
                "peak_source": peaks["source"] + " bf16_tflops_sustained (kernel timed inside a long step)",
                "achieved_counts": "FLOP of the tiles executed on true dimensions: 2 n^3 per full GEMM, the executed share (ntm + 1) / (2 ntm) "
                                   "of it for a symmetric product that multiplied the upper triangle of tiles only",
                "achieved_padded": gemm_tf_padded, "achieved_paper_convention_2n3_per_gemm": gemm_tf_paper,
                "avg_launch_us": 1e3 * prof_acc["gemm_ms"] / max(prof_acc["gemm_launches"], 1),
                "frac_of_burst": gemm_tf / peaks["bf16_tflops"], "frac_of_nominal_2250": gemm_tf / NOMINAL_FP16_TFLOPS}
    if persistent:
        # share of the step spent inside the kernel (the rest is assemble: host index logic + uploads)
        roofline["share_of_step_time"] = prof_acc["gemm_ms"] / (ms_step * args.steps)
        groups = 2 * ctr_acc["pairs"]                     # one side group (4 warps) per CTA
        side = ctr_acc["side"]
        g, d = side.get("gather", {}), side.get("dcols", {})
        # gather / scatter run as side tasks of the same launch, concurrently with the GEMM pipeline: the in-kernel figure is
        # algorithmic bytes / (busy time summed over the side groups / #groups); `alone` is the same code launched alone
        hbm = {"in_kernel_busy_time_gather_gbs": g.get("bytes", 0) / max(g.get("busy_ms", 0) / groups, 1e-9) / 1e6,
               "in_kernel_busy_time_scatter_gbs": d.get("bytes", 0) / max(d.get("busy_ms", 0) / groups, 1e-9) / 1e6,
               "gather_busy_frac_of_side_groups": g.get("busy_ms", 0) / max(groups * prof_acc["gemm_ms"], 1e-9),
               "scatter_busy_frac_of_side_groups": d.get("busy_ms", 0) / max(groups * prof_acc["gemm_ms"], 1e-9),
               "in_kernel_how": "side tasks inside nolsm_persist_kernel; bytes / (sum of side-group busy time / side groups)",
               "alone": side_alone, "peak_gbs": peaks["hbm_gbs"], "peak_source": peaks["source"]}
        if side_alone and "gather_gbs" in side_alone:
            hbm["gather_gbs"], hbm["scatter_gbs"] = side_alone["gather_gbs"], side_alone["scatter_gbs"]
        else:
            hbm["gather_gbs"], hbm["scatter_gbs"] = hbm["in_kernel_busy_time_gather_gbs"], hbm["in_kernel_busy_time_scatter_gbs"]
        pair_ms = max(ctr_acc["pairs"] * prof_acc["gemm_ms"], 1e-9)       # kernel time summed over the CTA pairs
        engine = {"tiles": ctr_acc["tiles"], "sched_idle_frac": ctr_acc["sched_idle_ms"] / pair_ms,
                  "slots": ctr_acc["slots"], "pairs": ctr_acc["pairs"],
                  # where the MMA-issuing warp of every pair spends the kernel (nolsm_get_engine_counters out[33..35])
                  "mma_warp_frac": {"tile_record_wait": ctr_acc["mma_wait_record_ms"] / pair_ms,
                                    "accumulator_wait": ctr_acc["mma_wait_accumulator_ms"] / pair_ms,
                                    "k_loops": ctr_acc["mma_kloop_ms"] / pair_ms},
                  "sched_frac": {"ring_wait": ctr_acc["sched_wait_ring_ms"] / pair_ms,
                                 "claim_point_wait": ctr_acc["sched_wait_claim_point_ms"] / pair_ms},
                  "power_steps_extra_per_submatrix": ctr_acc["power_steps_extra"] / max(stats["n_units"] * args.steps, 1)}
    else:
        roofline["share_of_sampled_kernel_time"] = prof_acc["gemm_ms"] / max(sampled_ms, 1e-9)
        hbm = {"gather_gbs": prof_acc["gather_bytes"] / max(prof_acc["gather_ms"], 1e-9) / 1e6,
               "scatter_gbs": prof_acc["dcols_bytes"] / max(prof_acc["dcols_ms"], 1e-9) / 1e6,
               "peak_gbs": peaks["hbm_gbs"], "peak_source": peaks["source"]}
        engine = None
    if clocks.get("power_w_median") and roofline.get("achieved"):
        # energy per FLOP of the headline run as a driver-visible number: median board power over the timed region / executed rate
        clocks["watts_per_tflops_executed"] = clocks["power_w_median"] / roofline["achieved"]
    hbm["gather_frac"] = hbm["gather_gbs"] / peaks["hbm_gbs"]
    hbm["scatter_frac"] = hbm["scatter_gbs"] / peaks["hbm_gbs"]

    cpu = None
    if args.cpu_sample != 0:
        ncpu = os.cpu_count() or 1
        nsamp = 3 * ncpu if args.cpu_sample < 0 else args.cpu_sample
        atoms = np.sort(np.random.default_rng(99).choice(system.n_atoms, min(nsamp, system.n_atoms), replace=False))
        dt, n, workers = oracle_sample(system, atoms)
        cpu = {"value": n / dt, "unit": "submatrices/s", "cores": workers, "kind": "oracle",
               "sample": f"{n} seeded-random submatrices of {workload_label(args.workload, args.atoms)} in {dt:.1f} s, "
                         f"{workers} worker processes with one BLAS thread each",
               "host_cpu_count": ncpu}

    line = {"metric": "submatrices_per_s", "value": value, "unit": "submatrices/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16", "data": "synthetic",
            "config": {"workload": workload_label(args.workload, args.atoms), "atoms": system.n_atoms,
                       "basis_per_atom": sorted(set(int(x) for x in np.unique(system.atom_nb))), "n_basis": int(system.atom_nb.sum()),
                       "dim_mean": stats["dim_mean"], "dim_min": stats["dim_min"], "dim_max": stats["dim_max"],
                       "precision": "fp16 operands / fp32 accumulate", "gamma_S": system.gamma,
                       "parallelism": "replicas" if world > 1 else "single",
                       "combine": args.combine, "iteration": "lowdin" if args.iteration else "eq6",
                       "symmetric_tiles": args.symmetric_tiles == 0,
                       "transposed_tiles": args.transposed_tiles == 0,
                       "value_counts": "atoms served per second (one submatrix per atom when combine = 0)",
                       "l2": "inputs (8 GB block-CSR) and workspace >> 126 MB L2; no flush needed"},
            "tensor_tflops": tflops, "pct_of_dense_fp16_peak": {"nominal_2250": 100 * tflops / NOMINAL_FP16_TFLOPS / world,
                                                                 "measured_burst": 100 * tflops / peaks["bf16_tflops"] / world,
                                                                 "measured_sustained": 100 * tflops / peaks["bf16_tflops_sustained"] / world},
            "flops_useful_per_step": stats["flops_useful"], "flops_padded_per_step": stats["flops_padded"],
            "flops_paper_convention_per_step": stats["flops_paper"],
            "gemms_per_submatrix": stats["gemms_executed"] / max(stats["n_units"], 1),
            "symmetric_gemms_per_submatrix": stats["gemms_symmetric"] / max(stats["n_units"], 1), "submatrices": stats["n_units"], "e_elec": E,
            "n_notspd": stats["n_notspd"], "n_noconv": stats["n_noconv"],
            "roofline": roofline, "hbm_kernels": hbm, "engine": engine, "variants": variants, "combined": combined,
            "other_configs": others, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
            "gpu_launches": int(prof_acc["kernel_launches"]),
            "paper_context": "1.1 EFLOP/s FP16/FP32 on 4400 A100 (~257 TFLOP/s per GPU, ~80% of 312), other hardware"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
