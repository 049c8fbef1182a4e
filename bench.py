#!/usr/bin/env python
"""bench.py -- H psi throughput on the synthetic molecule-shaped meshes (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--block 16] [--no-sweep]
    python bench.py --impl reference ...          # the CPU oracle on the host cores, same metric

A "step" is one pass of the whole hot path over one batch: for every block of B orbitals,
rs_block_pack -> rs_hamiltonian_apply -> rs_block_unpack (steps a4-a7 of DESIGN.md); the mesh tables
(a1-a3) are built once per geometry before the timed region and their wall time is reported.
`value` = nst * np * (2*(6n+1)+2) flops / step time with all inputs resident in HBM; `e2e` is the same
metric through rs_hamiltonian_apply_states_stream with pinned HOST buffers (H2D + D2H inside); its output
is compared with the oracle on sampled orbitals.  The line also carries the apply-alone block-size sweep
(the metric's axis), the tuned and un-tuned kernel times, and the oracle on 1 core and on all cores.
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
    t_one = time.perf_counter() - t          # one orbital on ONE core: the 1-core baseline (cost is linear in orbitals)
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
            "one_core": {"value": om.npoints * flops_per_output(n) * lanes / t_one / 1e9, "unit": UNIT, "cores": 1,
                         "sample": f"1 orbital of config {cfg.index}, single thread, {t_one:.2f} s"},
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
            "cpu_baseline": {k: leg[k] for k in ("value", "unit", "cores", "kind", "sample", "one_core")},
            "e2e": {"value": leg["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(cfg, n, B, npts, nst=None) -> dict:
    nst = cfg.nst if nst is None else nst
    note = "" if nst == cfg.nst else f" (REDUCED from the config's {cfg.nst} by --nst: not the named workload)"
    return {"workload": f"configs[{cfg.index}] {cfg.name}: {cfg.centers.shape[0]} centres, R={cfg.radius}, "
                        f"h={cfg.spacing}, np={npts}, nst={nst} {'complex' if cfg.is_complex else 'real'} fp64{note}",
            "fd_order": n, "block_size": B, "npoints": int(npts), "nst": nst,
            "l2": "inputs larger than L2 (per-orbital states + blocks >> 126 MB); no explicit flush"}


# ------------------------------------------------------------------------------------------------
def time_apply(rs, torch, mesh, n, coeffs, v, b1, b2, Bs, kern, reps):
    """Mean duration (ms) of `reps` back-to-back apply launches, CUDA events on torch's current stream."""
    for _ in range(3):
        rs.rs_hamiltonian_apply(mesh, n, coeffs, v, b1, b2, Bs, kernel=kern)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        rs.rs_hamiltonian_apply(mesh, n, coeffs, v, b1, b2, Bs, kernel=kern)
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def traffic_rows() -> dict:
    """DRAM bytes per launch from the committed `ncu --set full` captures (profiles/traffic.csv): NOT measured by this
    run (a number taken under a profiler is never a bench value); each row names its capture and commit."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return {}
    return {row["key"]: row for row in csv.DictReader(open(path))}


def run_streamed(args) -> None:
    """BASELINE.json configs[4] at its stated size: the whole orbital set streamed through HBM block by block from HOST memory
    (rs_hamiltonian_apply_states_stream, 3-window workspace).  Orbitals are generated chunk by chunk into one pinned buffer, so
    neither side ever holds the set (31 GB for config 4); generation time is not timed; one seeded orbital per chunk is compared
    with the oracle.  Prints one JSON line (an e2e-only record, not the driver's bench line)."""
    import torch

    import oracle
    import paper_1306_2953_b200 as rs

    cfg = synthetic.config(args.config)
    n = args.fd_order or cfg.fd_orders[0]
    B, chunk = args.block, args.stream_chunk
    nst = args.nst or cfg.nst
    is_c = cfg.is_complex
    tdt = torch.complex128 if is_c else torch.float64
    rsdt = rs.RS_COMPLEX128 if is_c else rs.RS_REAL64
    torch.cuda.set_device(0)
    mesh = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, max(cfg.fd_orders))
    npts = mesh.npoints
    ijk = mesh.points()
    rank_of = synthetic.canonical_rank(ijk)
    om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    vc = synthetic.vloc_at(om.xyz(), cfg.centers, cfg.charges)
    host_v = torch.from_numpy(np.ascontiguousarray(vc[rank_of])).pin_memory()
    host_in = torch.empty((chunk, npts), dtype=tdt).pin_memory()
    host_out = torch.empty((chunk, npts), dtype=tdt).pin_memory()
    coeffs = fd_coeffs(n)
    ws = rs.rs_workspace_create(mesh, B, rsdt, npts)
    rng = np.random.default_rng(args.config)
    total, worst, checked = 0.0, 0.0, []
    for ist0 in range(0, nst, chunk):
        nb = min(chunk, nst - ist0)
        hin = host_in.numpy()
        for j in range(nb):
            hin[j] = synthetic.orbital(cfg.seed, ist0 + j, npts, is_c)[rank_of]
        if ist0 == 0:   # warm-up (tables, first touch of the pinned buffers), not timed
            rs.rs_hamiltonian_apply_states_stream(ws, n, coeffs, host_v, host_in[:nb], host_out[:nb])
        torch.cuda.synchronize()
        t = time.perf_counter()
        rs.rs_hamiltonian_apply_states_stream(ws, n, coeffs, host_v, host_in[:nb], host_out[:nb])
        total += time.perf_counter() - t
        j = int(rng.integers(0, nb))
        psi = synthetic.orbital(cfg.seed, ist0 + j, npts, is_c)[None, :]
        o = oracle.hpsi(om, n, oracle.fd_coeffs(n), vc, psi, nthreads=len(os.sched_getaffinity(0)))
        g = np.empty_like(o)
        g[:, rank_of] = host_out.numpy()[j:j + 1]
        err = float(np.abs(g - o).max() / np.abs(o).max())
        worst = err if not (err <= worst) else worst          # a NaN must not hide behind max()
        checked.append(ist0 + j)
    esz = 16 if is_c else 8
    fl = nst * npts * flops_per_output(n) * (4 if is_c else 1)
    print(json.dumps({"metric": METRIC, "impl": "ours-streamed", "value": fl / total / 1e9, "unit": UNIT, "seconds": total,
                      "config": workload_config(cfg, n, B, npts, nst), "chunk_orbitals": chunk,
                      "h2d_bytes": nst * npts * esz + (nst + chunk - 1) // chunk * npts * 8, "d2h_bytes": nst * npts * esz,
                      "gbs_per_direction": nst * npts * esz / total / 1e9, "workspace_bytes": ws.nbytes,
                      "device_resident_states_bytes": 0, "max_normwise_err": worst, "checked_orbitals": checked,
                      "api": "rs_hamiltonian_apply_states_stream, one call per chunk, pinned host buffers"}))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--block", type=int, default=16)
    ap.add_argument("--fd-order", type=int, default=0)
    ap.add_argument("--nst", type=int, default=0, help="override the orbital count (debugging only; the line says so)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "gather", "sweep"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the apply-alone block-size sweep (the metric's axis)")
    ap.add_argument("--sweep", action="store_true", help="(default now; kept for old command lines)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-autotune", action="store_true", help="skip rs_hamiltonian_autotune (work dealt by the built-in cost model)")
    ap.add_argument("--ordering", default="lex", choices=["lex", "brick", "tile"],
                    help="point enumeration of the mesh (ordering study; brick / tile are served by the gather kernel)")
    ap.add_argument("--planes-tuned", type=int, default=0,
                    help="x-slab thickness of the plane-sweep work pieces after autotune (0: library default = whole tile columns)")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the timings of the f1-f3 operations (SURVEY.md 8(f))")
    ap.add_argument("--stream-chunk", type=int, default=0,
                    help="e2e only, for orbital sets too large to keep resident: stream the config's orbitals from host memory in "
                         "chunks of this many, generated on the fly (configs[4]: 1024 orbitals)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.stream_chunk:
        run_streamed(args)
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
    conv = 4 if is_c else 1          # the metric's flop convention for complex (BASELINE.json); executed arithmetic is 2x real (S12)
    tune = not args.no_autotune and args.kernel != "gather"

    # ---- once per geometry: mesh tables (a1-a3), potential, inputs --------------------------------
    t = time.perf_counter()
    ordering = {"lex": rs.RS_ORDER_LEX, "brick": rs.RS_ORDER_BRICK, "tile": rs.RS_ORDER_TILE}[args.ordering]
    mesh = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, max(cfg.fd_orders), ordering)
    t_mesh = time.perf_counter() - t
    if args.planes_tuned:
        rs.rs_mesh_set_sweep_options(mesh, planes_tuned=args.planes_tuned)
    npts = mesh.npoints
    ijk = mesh.points()
    v_mesh = synthetic.vloc_at(ijk.astype(np.float64) * cfg.spacing, cfg.centers, cfg.charges)
    rank_of = synthetic.canonical_rank(ijk)
    # weak scaling: every rank owns its own nst orbitals (orbital ids rank*nst ...), same mesh and V
    host_states = torch.empty((nst, npts), dtype=tdt).pin_memory()
    hs = host_states.numpy()
    for j, ist in enumerate(synthetic.rank_orbital_ids(rank, nst)):
        hs[j] = synthetic.orbital(cfg.seed, ist, npts, is_c)[rank_of]
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

    # once per geometry, like the mesh tables: build the neighbour structure, then let the library measure its own
    # per-plane costs and re-deal the work (rs_hamiltonian_autotune); the un-tuned time is reported beside the tuned one
    t = time.perf_counter()
    rs.rs_hamiltonian_prepare(mesh, n, B, rsdt)
    t_prepare = time.perf_counter() - t
    rs.rs_block_pack(mesh, states, 0, min(B, nst), B, blk)
    untuned_ms = time_apply(rs, torch, mesh, n, coeffs, v, blk, hblk, B, kern, 20)
    t = time.perf_counter()
    if tune:
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
    fl_step = nst * npts * flops_per_output(n) * conv                   # metric convention: 4x for complex
    value = world * fl_step / (ms_step * 1e-3) / 1e9

    apply_ms = float(np.mean([a.elapsed_time(b) for a, b in apply_events]))
    alg_bytes = algorithmic_bytes(npts, B * lanes, table_bytes)
    achieved = alg_bytes / (apply_ms * 1e-3) / 1e9
    peak, peak_src = measured_peak_hbm()
    roofline = {"bound": "hbm", "kernel": f"rs_hamiltonian_apply[{kname}] B={B} n={n}", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "frac_of_8TBs": achieved / 8000.0,
                "peak_source": peak_src, "traffic": None, "algorithmic_bytes_per_launch": alg_bytes,
                "apply_ms_per_launch": apply_ms, "apply_ms_per_launch_untuned": untuned_ms,
                "apply_share_of_step": apply_ms * nblocks / ms_step,
                "apply_gflops": B * npts * flops_per_output(n) * conv / (apply_ms * 1e-3) / 1e9,
                "apply_gflops_executed": B * npts * flops_per_output(n) * lanes / (apply_ms * 1e-3) / 1e9}
    # second bound of the same kernel: plain fp64 arithmetic (DFMA issues at one warp instruction
    # per 2 clocks per scheduler = 64 lanes per SM; peak = SMs x 64 x 2 flops x the SM clock sampled during this run)
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_mhz = float((clocks or {}).get("sm_mhz") or 0.0) or 1965.0
    alu_peak = sm_count * 64 * 2 * sm_mhz * 1e6 / 1e12
    roofline["alu"] = {"bound": "alu", "achieved": roofline["apply_gflops_executed"] / 1e3, "peak": alu_peak, "unit": "TFLOP/s",
                       "frac": roofline["apply_gflops_executed"] / 1e3 / alu_peak,
                       "note": "useful flops only (2(6n+1)+2 per output); the kernel also spends fp64 issue slots on points of "
                               "partly filled tiles and on the 2n centre-only planes around every work piece"}
    traffic = traffic_rows()
    row = traffic.get(f"config{cfg.index}_B{B}_n{n}_{kname}")
    if row:    # from a committed ncu capture of this kernel, not from this run
        roofline.update({"traffic": int(row["dram_read_bytes"]) + int(row["dram_write_bytes"]),
                         "traffic_read": int(row["dram_read_bytes"]), "traffic_write": int(row["dram_write_bytes"]),
                         "traffic_compulsory_read": npts * (8 * B * lanes + 8) + table_bytes,
                         "traffic_compulsory_write": npts * 8 * B * lanes,
                         "traffic_source": f"{row['capture']} (ncu --set full, commit {row['commit']}); not measured by this run"})

    # ---- the caller that keeps psi in the block layout (the paper's storage format): apply alone over all blocks
    blocked = None
    if rank == 0:
        for _ in range(2):
            for _k in range(nblocks):
                rs.rs_hamiltonian_apply(mesh, n, coeffs, v, blk, hblk, B, kernel=kern)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            for _k in range(nblocks):
                rs.rs_hamiltonian_apply(mesh, n, coeffs, v, blk, hblk, B, kernel=kern)
        b.record()
        torch.cuda.synchronize()
        msb = a.elapsed_time(b) / args.steps
        blocked = {"value": fl_step / (msb * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": msb,
                   "note": "apply over all blocks, psi kept blocked (no pack / unpack); one block buffer pair reused: "
                           f"{2 * blk.numel() * blk.element_size() / 1e6:.0f} MB per launch vs 126 MB L2"}

    # ---- block-size sweep of the apply kernel alone (the metric is "vs orbital block size") -------
    sweep = None
    if not args.no_sweep and rank == 0:
        sweep = []
        for Bs in cfg.block_sizes:
            b1 = torch.empty((npts + 1, Bs), dtype=tdt, device=dev)
            b2 = torch.empty((npts + 1, Bs), dtype=tdt, device=dev)
            rs.rs_block_pack(mesh, states, 0, min(Bs, nst), Bs, b1)
            reps = max(3, min(50, int(nst // Bs)))
            rs.rs_hamiltonian_prepare(mesh, n, Bs, rsdt)
            ms_untuned = time_apply(rs, torch, mesh, n, coeffs, v, b1, b2, Bs, kern, reps) if Bs != B else untuned_ms
            if tune and Bs != B:
                rs.rs_hamiltonian_autotune(mesh, n, coeffs, v, b1, b2, Bs)
            ms = time_apply(rs, torch, mesh, n, coeffs, v, b1, b2, Bs, kern, reps)
            kn = rs.rs_kernel_name(mesh, n, Bs, rsdt, kern)
            ab = algorithmic_bytes(npts, Bs * lanes, rs.rs_kernel_table_bytes(mesh, n, Bs, rsdt, kern))
            row = traffic.get(f"config{cfg.index}_B{Bs}_n{n}_{kn}")
            sweep.append({"block": Bs, "kernel": kn, "apply_ms": ms, "apply_ms_untuned": ms_untuned,
                          "gflops": Bs * npts * flops_per_output(n) * conv / ms / 1e6,
                          "gflops_executed": Bs * npts * flops_per_output(n) * lanes / ms / 1e6,
                          "alg_gbs": ab / ms / 1e6, "frac_measured": ab / ms / 1e6 / peak, "frac_of_8TBs": ab / ms / 1e6 / 8000.0,
                          "traffic": (int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])) if row else None,
                          "note": "block working set may fit L2" if 2 * b1.numel() * b1.element_size() < 126e6 else ""})
            if kn.startswith("sweep[") and Bs * lanes < 16 and kern == rs.RS_KERNEL_AUTO:
                # 8 columns run as half a 16-column slice of the plane-sweep kernel (it does the work of 16 columns, and its
                # compact records make the algorithmic byte count smaller than the gather kernel's): the alternative beside it
                msg = time_apply(rs, torch, mesh, n, coeffs, v, b1, b2, Bs, rs.RS_KERNEL_GATHER, reps)
                abg = algorithmic_bytes(npts, Bs * lanes, rs.rs_kernel_table_bytes(mesh, n, Bs, rsdt, rs.RS_KERNEL_GATHER))
                sweep[-1].update({"gather_apply_ms": msg, "gather_alg_gbs": abg / msg / 1e6, "gather_frac_measured": abg / msg / 1e6 / peak,
                                  "note": "half slice of the sweep kernel: faster than the gather kernel, fewer algorithmic bytes"})
            del b1, b2

    # ---- the operations around H psi on the same block: time and algorithmic rates -------
    next_rows = None
    if not args.no_next_rows and rank == 0:
        def timed(fn, reps=20):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / reps
        rs.rs_block_pack(mesh, states, 0, min(B, nst), B, blk)
        rs.rs_hamiltonian_apply(mesh, n, coeffs, v, blk, hblk, B, kernel=kern)
        blk_bytes = npts * B * 8 * lanes
        sums = torch.empty((3, B), dtype=torch.float64, device=dev)
        eps_d = torch.zeros(B, dtype=torch.float64, device=dev)
        Mm = torch.empty((B, B), dtype=tdt, device=dev)
        alpha = torch.ones(B, dtype=tdt, device=dev)
        ms_exp = timed(lambda: rs.rs_block_expectation(mesh, blk, hblk, eps_d, B, sums))
        ms_ex = timed(lambda: rs.rs_hamiltonian_apply_ex(mesh, n, coeffs, v, blk, hblk, B, eps_d, sums))
        ms_ovl = timed(lambda: rs.rs_block_overlap(mesh, blk, hblk, B, Mm))
        ms_axpy = timed(lambda: rs.rs_block_axpy(mesh, alpha, blk, hblk, B))
        rs.rs_hamiltonian_apply(mesh, n, coeffs, v, blk, hblk, B, kernel=kern)
        rc_nl, lmax = 2.0, 1
        nl = rs.rs_nonlocal_create(mesh, cfg.centers, rc_nl, (lmax + 1) ** 2)
        nsph = 0
        for A in range(cfg.centers.shape[0]):
            idx = nl.sphere(A)
            nsph += idx.size
            nl.set_projectors(A, synthetic.projector_values(ijk[idx].astype(np.float64) * cfg.spacing - cfg.centers[A], lmax, 0.7))
        nl.prepare()
        ms_nl = timed(lambda: rs.rs_nonlocal_apply(nl, blk, hblk, B))
        nlm = (lmax + 1) ** 2
        next_rows = {
            "f1_expectation": {"ms": ms_exp, "alg_gbs": 2 * blk_bytes / ms_exp / 1e6, "frac_measured": 2 * blk_bytes / ms_exp / 1e6 / peak},
            "f1_apply_ex": {"ms": ms_ex, "extra_over_apply": ms_ex / apply_ms - 1.0,
                            "note": "apply + streaming reduction kernel (a fused consumer epilogue was measured slower, DESIGN.md)"},
            "f1_axpy": {"ms": ms_axpy, "alg_gbs": 3 * blk_bytes / ms_axpy / 1e6, "frac_measured": 3 * blk_bytes / ms_axpy / 1e6 / peak},
            "f2_overlap": {"ms": ms_ovl, "alg_gbs": 2 * blk_bytes / ms_ovl / 1e6, "frac_measured": 2 * blk_bytes / ms_ovl / 1e6 / peak,
                           "tflops_executed": 2.0 * npts * (B * lanes) ** 2 / ms_ovl / 1e9, "kernel": "overlap_kernel (fp64 DMMA m8n8k4)"},
            "f3_nonlocal": {"ms": ms_nl, "atoms": int(cfg.centers.shape[0]), "rc": rc_nl, "nlm": nlm, "sphere_points": int(nsph),
                            "colors": nl.ncolors, "gflops_executed": 4.0 * nsph * B * lanes * nlm / ms_nl / 1e6,
                            "alg_gbs": nsph * (3 * B * lanes * 8 + 2 * nlm * 8 + 4) / ms_nl / 1e6},
        }
        del nl

    # ---- end to end through the host-buffer entry point (a7 workspace, created once) ---------------
    e2e = None
    if not args.no_e2e:
        del states, out, blk, hblk
        torch.cuda.empty_cache()
        ws = rs.rs_workspace_create(mesh, B, rsdt, npts)
        rs.rs_hamiltonian_apply_states_stream(ws, n, coeffs, host_v, host_states, host_out)      # warm-up
        barrier()
        k = max(1, min(args.steps, 3))
        t = time.perf_counter()
        for _ in range(k):
            rs.rs_hamiltonian_apply_states_stream(ws, n, coeffs, host_v, host_states, host_out)
        barrier()
        dt = (time.perf_counter() - t) / k
        if world > 1:
            tt = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dt = float(tt.item())
        sbytes = host_states.numel() * host_states.element_size()
        e2e = {"value": world * fl_step / dt / 1e9, "unit": UNIT, "h2d_bytes_per_step": sbytes + npts * 8,
               "d2h_bytes_per_step": sbytes, "ms_per_step": dt * 1e3, "steps": k,
               "workspace_bytes": ws.nbytes,
               "api": "rs_hamiltonian_apply_states_stream (pinned host buffers, 3-window workspace created once)"}
        if rank == 0 and not args.no_cpu_baseline:
            # the end-to-end OUTPUT is compared with the oracle on a seeded sample of orbitals (first / last block and two between)
            import oracle
            om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
            assert om.npoints == npts
            vc = synthetic.vloc_at(om.xyz(), cfg.centers, cfg.charges)
            pick = sorted({0, nst - 1, *np.random.default_rng(12).integers(0, nst, 2).tolist()})
            psi = np.stack([synthetic.orbital(cfg.seed, rank * nst + j, npts, is_c) for j in pick])
            o = oracle.hpsi(om, n, oracle.fd_coeffs(n), vc, psi, nthreads=len(os.sched_getaffinity(0)))
            g = np.empty_like(o)
            g[:, rank_of] = host_out.numpy()[pick]
            e2e["max_normwise_err"] = float(np.abs(g - o).max() / np.abs(o).max())
            e2e["checked_orbitals"] = pick
        del ws

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "c128" if is_c else "f64", "data": "synthetic",
                "config": {**workload_config(cfg, n, B, npts, nst), "kernel": kname, "parallelism": f"orbital-blocks x{world}",
                           "mesh_build_s": t_mesh, "prepare_s": t_prepare, "autotune_s": t_tune, "autotuned": tune,
                           "nbricks": mesh.nbricks, "ordering": args.ordering, "planes_tuned": args.planes_tuned or "whole columns"},
                "value_executed_flops": world * nst * npts * flops_per_output(n) * lanes / (ms_step * 1e-3) / 1e9,
                "flop_convention": "BASELINE.json: nst*np*(2*(6n+1)+2), x4 for complex; *_executed counts the arithmetic "
                                   "actually done (complex = 2 real lanes, reading S12)",
                "roofline": roofline, "clocks": clocks, "gpu_launches": 3 * nblocks * args.steps}
        if blocked:
            line["blocked_resident"] = blocked
        if next_rows:
            line["next_rows"] = next_rows
        if e2e:
            line["e2e"] = e2e
        if sweep:
            line["sweep"] = sweep
        if not args.no_cpu_baseline and world == 1:
            leg = cpu_oracle_leg(cfg, n, seconds_budget=15.0)
            line["cpu_baseline"] = {k: leg[k] for k in ("value", "unit", "cores", "kind", "sample", "one_core")}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
