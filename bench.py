#!/usr/bin/env python
"""bench.py -- H psi throughput on the synthetic molecule-shaped meshes (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--block 16] [--sweep]
    python bench.py --impl reference ...          # the CPU oracle on the host cores, same metric

A "step" is one pass of the whole hot path over one batch: for every block of B orbitals,
rs_block_pack -> rs_hamiltonian_apply -> rs_block_unpack (steps a4-a7 of DESIGN.md); the mesh tables
(a1-a3) are built once per geometry before the timed region and their wall time is reported.
`value` = nst * np * (2*(6n+1)+2) flops / step time with all inputs resident in HBM; `e2e` is the same
metric through rs_hamiltonian_apply_states_host with pinned HOST buffers (H2D + D2H inside).
Prints ONE JSON line on rank 0.  See DESIGN.md "Measurement" for the byte accounting.
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

import synthetic  # noqa: E402

METRIC = "Hpsi fp64 GFLOP/s"
UNIT = "GFLOP/s"


def flops_per_output(n: int) -> int:
    return 2 * (6 * n + 1) + 2          # BASELINE.json: flops = nst*np*(2*(6*order+1)+2) for real


def algorithmic_bytes(npts: int, ncol: int, table_bytes: int) -> int:
    """Compulsory HBM traffic of one apply launch: psi read once, H psi written once, V once, the
    neighbour structure actually used once."""
    return npts * (2 * 8 * ncol + 8) + table_bytes


def fd_coeffs(n: int) -> np.ndarray:
    """Input of the C ABI (textbook central weights, reading S1); neither side's arithmetic."""
    from math import factorial

    c = np.zeros(n + 1)
    for m in range(1, n + 1):
        c[m] = 2.0 * (-1) ** (m + 1) * factorial(n) ** 2 / (m * m * factorial(n - m) * factorial(n + m))
    c[0] = -2.0 * c[1:].sum()
    return c


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peak_hbm() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------------------------------------
def cpu_oracle_leg(cfg, n: int, seconds_budget: float = 20.0, steps: int = 1, warmup: int = 0) -> dict:
    """The oracle as it stands, on the host cores, on a bounded sample of the workload: whole
    orbitals of the same mesh and potential (cost is exactly linear in the orbital count)."""
    import oracle

    cores = len(os.sched_getaffinity(0))
    om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    v = synthetic.vloc_at(om.xyz(), cfg.centers, cfg.charges)
    c = oracle.fd_coeffs(n)
    probe = synthetic.orbitals(cfg.seed, 0, 1, om.npoints, cfg.is_complex)
    t = time.perf_counter()
    oracle.hpsi(om, n, c, v, probe, nthreads=1)
    t_one = time.perf_counter() - t
    nsample = int(max(cores, min(cfg.nst, cores * max(1.0, seconds_budget / max(t_one, 1e-3)) // max(1, steps + warmup))))
    nsample = max(cores, (nsample // cores) * cores)
    nsample = min(nsample, max(cores, cfg.nst))
    psi = synthetic.orbitals(cfg.seed, 0, nsample, om.npoints, cfg.is_complex)
    times = []
    for it in range(warmup + steps):
        t = time.perf_counter()
        oracle.hpsi(om, n, c, v, psi, nthreads=cores)
        if it >= warmup:
            times.append(time.perf_counter() - t)
    dt = float(np.mean(times))
    lanes = 4 if cfg.is_complex else 1         # the metric's convention for complex (BASELINE.json)
    gf = nsample * om.npoints * flops_per_output(n) * lanes / dt / 1e9
    return {"value": gf, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{nsample} of {cfg.nst} orbitals of config {cfg.index} (np={om.npoints}, fd_order={n}), "
                      f"{cores} OpenMP threads over orbitals, {dt:.2f} s/step",
            "ms_per_step": dt * 1e3, "npoints": om.npoints, "nsample": nsample}


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = synthetic.config(args.config)
    n = args.fd_order or cfg.fd_orders[0]
    leg = cpu_oracle_leg(cfg, n, seconds_budget=40.0, steps=args.steps, warmup=args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": leg["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": leg["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128" if cfg.is_complex else "f64", "data": "synthetic",
            "config": workload_config(cfg, n, args.block, leg["npoints"]),
            "cpu_baseline": {k: leg[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": leg["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(cfg, n, B, npts) -> dict:
    return {"workload": f"configs[{cfg.index}] {cfg.name}: {cfg.centers.shape[0]} centres, R={cfg.radius}, "
                        f"h={cfg.spacing}, np={npts}, nst={cfg.nst} {'complex' if cfg.is_complex else 'real'} fp64",
            "fd_order": n, "block_size": B, "npoints": int(npts), "nst": cfg.nst,
            "l2": "inputs larger than L2 (per-orbital states + blocks >> 126 MB); no explicit flush"}


# ------------------------------------------------------------------------------------------------
def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--block", type=int, default=16)
    ap.add_argument("--fd-order", type=int, default=0)
    ap.add_argument("--nst", type=int, default=0, help="override the orbital count (debugging only; invalidates the number)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "gather", "sweep"])
    ap.add_argument("--sweep", action="store_true", help="also time apply alone for every block size of the config")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-autotune", action="store_true", help="skip rs_hamiltonian_autotune (work dealt by the built-in cost model)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import torch.distributed as dist

    import paper_1306_2953_b200 as rs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = synthetic.config(args.config)
    n = args.fd_order or cfg.fd_orders[0]
    B = args.block
    nst = args.nst or cfg.nst
    kern = {"auto": rs.RS_KERNEL_AUTO, "gather": rs.RS_KERNEL_GATHER, "sweep": rs.RS_KERNEL_SWEEP}[args.kernel]
    coeffs = fd_coeffs(n)
    is_c = cfg.is_complex
    rsdt = rs.RS_COMPLEX128 if is_c else rs.RS_REAL64
    tdt = torch.complex128 if is_c else torch.float64
    lanes = 2 if is_c else 1

    # ---- once per geometry: mesh tables (a1-a3), potential, inputs --------------------------------
    t = time.perf_counter()
    mesh = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, max(cfg.fd_orders))
    t_mesh = time.perf_counter() - t
    npts = mesh.npoints
    ijk = mesh.points()
    v_mesh = synthetic.vloc_at(ijk.astype(np.float64) * cfg.spacing, cfg.centers, cfg.charges)
    rank_of = synthetic.canonical_rank(ijk)
    # weak scaling: every rank owns its own nst orbitals (orbital ids rank*nst ...), same mesh and V
    host_states = torch.empty((nst, npts), dtype=tdt).pin_memory()
    hs = host_states.numpy()
    for j in range(nst):
        hs[j] = synthetic.orbital(cfg.seed, rank * nst + j, npts, is_c)[rank_of]
    host_out = torch.empty((nst, npts), dtype=tdt).pin_memory()
    host_v = torch.from_numpy(v_mesh).pin_memory()

    states = host_states.to(dev)
    out = torch.empty_like(states)
    v = host_v.to(dev)
    blk = torch.empty((npts + 1, B), dtype=tdt, device=dev)
    hblk = torch.empty((npts + 1, B), dtype=tdt, device=dev)
    nblocks = (nst + B - 1) // B

    apply_events = []

    def step(record: bool):
        for ist0 in range(0, nst, B):
            nb = min(B, nst - ist0)
            rs.rs_block_pack(mesh, states, ist0, nb, B, blk)
            if record:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
            rs.rs_hamiltonian_apply(mesh, n, coeffs, v, blk, hblk, B, kernel=kern)
            if record:
                e1.record()
                apply_events.append((e0, e1))
            rs.rs_block_unpack(mesh, hblk, B, nb, out, ist0)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # once per geometry, like the mesh tables: let the library measure its own per-plane costs and re-deal the work
    t = time.perf_counter()
    if not args.no_autotune and args.kernel != "gather":
        rs.rs_block_pack(mesh, states, 0, min(B, nst), B, blk)
        rs.rs_hamiltonian_autotune(mesh, n, coeffs, v, blk, hblk, B)
    t_tune = time.perf_counter() - t
    kname = rs.rs_kernel_name(mesh, n, B, rsdt, kern)
    table_bytes = rs.rs_kernel_table_bytes(mesh, n, B, rsdt, kern)     # of the tables in use (after the re-deal)
    for _ in range(args.warmup):
        step(False)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    t0w = time.time()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        step(True)
    ev1.record()
    barrier()
    t1w = time.time()
    ms_total = ev0.elapsed_time(ev1)
    if world > 1:
        tt = torch.tensor([ms_total], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_total = float(tt.item())
    clocks = sampler.stop(t0w, t1w) if rank == 0 else None
    ms_step = ms_total / args.steps
    fl_step = nst * npts * flops_per_output(n) * (4 if is_c else 1)     # metric convention: 4x for complex
    value = world * fl_step / (ms_step * 1e-3) / 1e9

    apply_ms = float(np.mean([a.elapsed_time(b) for a, b in apply_events]))
    alg_bytes = algorithmic_bytes(npts, B * lanes, table_bytes)
    achieved = alg_bytes / (apply_ms * 1e-3) / 1e9
    peak, peak_src = measured_peak_hbm()
    roofline = {"bound": "hbm", "kernel": f"rs_hamiltonian_apply[{kname}] B={B} n={n}", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "frac_of_8TBs": achieved / 8000.0,
                "peak_source": peak_src, "traffic": None, "algorithmic_bytes_per_launch": alg_bytes,
                "apply_ms_per_launch": apply_ms, "apply_share_of_step": apply_ms * nblocks / ms_step,
                "apply_gflops": B * npts * flops_per_output(n) * (4 if is_c else 1) / (apply_ms * 1e-3) / 1e9}
    traffic_file = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(traffic_file):      # dram bytes per launch from the committed ncu --set full capture
        import csv
        key = f"config{cfg.index}_B{B}_n{n}_{kname}"
        for row in csv.DictReader(open(traffic_file)):
            if row["key"] == key:
                roofline["traffic"] = int(row["dram_bytes_per_launch"])

    # ---- block-size sweep of the apply kernel alone (the metric is "vs orbital block size") -------
    sweep = None
    if args.sweep and rank == 0:
        sweep = []
        for Bs in cfg.block_sizes:
            b1 = torch.empty((npts + 1, Bs), dtype=tdt, device=dev)
            b2 = torch.empty((npts + 1, Bs), dtype=tdt, device=dev)
            rs.rs_block_pack(mesh, states, 0, min(Bs, nst), Bs, b1)
            reps = max(3, min(50, int(nst // Bs)))
            if not args.no_autotune and args.kernel != "gather":
                rs.rs_hamiltonian_autotune(mesh, n, coeffs, v, b1, b2, Bs)
            for _ in range(3):
                rs.rs_hamiltonian_apply(mesh, n, coeffs, v, b1, b2, Bs, kernel=kern)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                rs.rs_hamiltonian_apply(mesh, n, coeffs, v, b1, b2, Bs, kernel=kern)
            b.record()
            torch.cuda.synchronize()
            ms = a.elapsed_time(b) / reps
            ab = algorithmic_bytes(npts, Bs * lanes, rs.rs_kernel_table_bytes(mesh, n, Bs, rsdt, kern))
            sweep.append({"block": Bs, "kernel": rs.rs_kernel_name(mesh, n, Bs, rsdt, kern), "apply_ms": ms,
                          "gflops": Bs * npts * flops_per_output(n) * (4 if is_c else 1) / ms / 1e6,
                          "alg_gbs": ab / ms / 1e6, "frac_measured": ab / ms / 1e6 / peak,
                          "note": "block working set may fit L2" if 2 * b1.numel() * b1.element_size() < 126e6 else ""})
            del b1, b2

    # ---- end to end through the host-buffer entry point ------------------------------------------
    e2e = None
    if not args.no_e2e:
        del states, out, blk, hblk
        torch.cuda.empty_cache()
        for _ in range(1):
            rs.rs_hamiltonian_apply_states_host(mesh, n, coeffs, host_v, host_states, host_out, B)
        barrier()
        k = max(1, min(args.steps, 3))
        t = time.perf_counter()
        for _ in range(k):
            rs.rs_hamiltonian_apply_states_host(mesh, n, coeffs, host_v, host_states, host_out, B)
        barrier()
        dt = (time.perf_counter() - t) / k
        if world > 1:
            tt = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dt = float(tt.item())
        sbytes = host_states.numel() * host_states.element_size()
        e2e = {"value": world * fl_step / dt / 1e9, "unit": UNIT, "h2d_bytes_per_step": sbytes + npts * 8,
               "d2h_bytes_per_step": sbytes, "ms_per_step": dt * 1e3, "steps": k,
               "api": "rs_hamiltonian_apply_states_host (pinned host buffers)"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "c128" if is_c else "f64", "data": "synthetic",
                "config": {**workload_config(cfg, n, B, npts), "kernel": kname, "parallelism": f"orbital-blocks x{world}",
                           "mesh_build_s": t_mesh, "autotune_s": t_tune, "autotuned": not args.no_autotune, "nbricks": mesh.nbricks},
                "roofline": roofline, "clocks": clocks, "gpu_launches": 3 * nblocks * args.steps}
        if e2e:
            line["e2e"] = e2e
        if sweep:
            line["sweep"] = sweep
        if not args.no_cpu_baseline and world == 1:
            leg = cpu_oracle_leg(cfg, n, seconds_budget=15.0)
            line["cpu_baseline"] = {k: leg[k] for k in ("value", "unit", "cores", "kind", "sample")}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
