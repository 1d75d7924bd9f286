#!/usr/bin/env python
"""bench.py -- headline benchmark of the multishift solver hot path (contract: see DESIGN.md).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one complete CG-M solve (every iteration runs rows A1-A7 of SURVEY.md 8(a)) of the
workload BASELINE.json's target is quoted on: the 32^3x64 SU(3) lattice (configs[3]), complex128,
3x3-block BSR, 16 shifts, tol 1e-10.  `value` = solver iterations/s with inputs resident in HBM;
`ms_per_step` = time to solution; `e2e` = the same through msolve_solve_host with HOST b and x
(H2D/D2H inside the timed region); `roofline` = the dominant kernel (fused multishift update)
against the measured HBM copy bandwidth; `cpu_baseline` = the CPU oracle on this box's cores.
N > 1: independent replicas (one problem per GPU, different right-hand sides), no collective on
the data path ("replicas only"); value = all ranks' iterations / max-over-ranks time.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1102_2143_b200 import workloads as W  # noqa: E402

DTYPE_NAME = {np.complex128: "c128", np.complex64: "c64", np.float64: "f64", np.float32: "f32"}
METRIC = "multishift_solver_iterations_per_s"
UNIT = "iterations/s"


# ----------------------------------------------------------------------------------- workloads
def make_workload(name: str, rank: int, want_csr: bool, extents=None):
    """Returns (workload, dtype, format).  Right-hand side differs per rank (replicas).
    extents: config 4's operator on another lattice (size sweeps; config4_c128_bsr3 / _lat only)."""
    if extents is not None:
        if name not in ("config4_c128_bsr3", "config4_c128_lat"):
            raise SystemExit("--extents goes with --workload config4_c128_bsr3 or config4_c128_lat")
        w, dt, fmt = W.config4(extents=tuple(extents), want_csr=want_csr), np.complex128, name.rsplit("_", 1)[1]
    elif name == "config4_c128_bsr3":
        w, dt, fmt = W.config4(want_csr=want_csr), np.complex128, "bsr3"
    elif name == "config4_c64_bsr3":
        w, dt, fmt = W.config4(want_csr=want_csr, tol=1e-5), np.complex64, "bsr3"
    elif name == "config4_c128_lat":                   # matrix-free operator from the link field
        w, dt, fmt = W.config4(want_csr=want_csr), np.complex128, "lat"
    elif name == "config4_c64_lat":
        w, dt, fmt = W.config4(want_csr=want_csr, tol=1e-5), np.complex64, "lat"
    elif name == "config4_small_c128_lat":
        w, dt, fmt = W.config4(extents=(32, 8, 8, 8), want_csr=want_csr), np.complex128, "lat"
    elif name == "config3_c128_lat":
        w, dt, fmt = W.config3(), np.complex128, "lat"
    elif name == "config2_c128_lat":
        w, dt, fmt = W.config2(), np.complex128, "lat"
    elif name == "config4_c128_csr":
        w, dt, fmt = W.config4(want_csr=True), np.complex128, "csr"
    elif name == "config4_c64_csr":
        w, dt, fmt = W.config4(want_csr=True, tol=1e-5), np.complex64, "csr"
    elif name == "config3_c128_csr":
        w, dt, fmt = W.config3(), np.complex128, "csr"
    elif name == "config2_c128_csr":
        w, dt, fmt = W.config2(), np.complex128, "csr"
    elif name == "config1_c128_csr":                 # BASELINE configs[0]: 8x8 U(1) lattice, N = 64
        w, dt, fmt = W.config1(), np.complex128, "csr"
    elif name == "config4_small_c128_bsr3":          # quick functional check of the bench itself
        w, dt, fmt = W.config4(extents=(8, 8, 8, 16), want_csr=want_csr), np.complex128, "bsr3"
    elif name == "config2_c128_bsr3":
        w, dt, fmt = W.config2(), np.complex128, "bsr3"
    elif name == "config3_c128_bsr3":
        w, dt, fmt = W.config3(), np.complex128, "bsr3"
    elif name == "config3x_c128_bsr3":               # config 3's non-Hermitian operator on config 4's lattice:
        w, dt, fmt = W.config3(extents=(32, 32, 32, 64)), np.complex128, "bsr3"   # BiCGStab-M kernels at HBM-bound size
    elif name == "config3x_c128_lat":
        w, dt, fmt = W.config3(extents=(32, 32, 32, 64)), np.complex128, "lat"
    elif name == "config5_c128_csr":
        w, dt, fmt = W.config5(), np.complex128, "csr"
    elif name == "config5_c64_csr":
        w, dt, fmt = W.config5(tol=1e-5), np.complex64, "csr"
    elif name in ("poisson1000_f64_csr", "poisson1000_f32_csr"):   # the paper's own Table 1 run
        dt = np.float64 if "f64" in name else np.float32
        w, fmt = W.poisson_workload(1000, 1000, nshifts=15, tol=1e-5, real=True), "csr"
        w.max_iter = 2000                                          # default_monitor(b, 2000, 1e-5)
    elif name == "config5_small_c128_csr":
        w, dt, fmt = W.config5(n=1 << 16), np.complex128, "csr"
    else:
        raise SystemExit("unknown workload %s" % name)
    if rank:
        w.b = (W.real_unit_rhs if np.isrealobj(w.b) else W.unit_rhs)(W.DEFAULT_SEED + rank, w.n)
    return w, dt, fmt


def algorithmic_bytes(w, dtype, fmt, s_active, defer=0, profile_iters=20):
    """bytes the method must move per kernel launch (x gathered once).
    defer = M > 0 (CG-M, deferred multishift update): `cgm_update` is the r update alone (r, q in, r out) and
    `cgm_flush` is launched in every iteration but moves bytes once per M: the mean over the launches that
    msolve_profile_iteration times (bodies 2 .. profile_iters + 1 of a solve; the first flush of a solve reads M
    residuals and writes S x_k and S p_k, a later one also reads them)."""
    e = np.dtype(dtype).itemsize
    n = w.n
    if fmt == "bsr3":
        nb = w.bcolidx.size
        spmv = nb * (9 * e + 4) + (n // 3 + 1) * 4 + 2 * n * e
    elif fmt == "lat":          # every link once (d blocks of 9 per site), x in, y out; no indices
        spmv = w.links.size * e + 2 * n * e
    else:
        spmv = w.nnz * (e + 4) + (n + 1) * 4 + 2 * n * e
    if w.algorithm == "cgm" and defer > 0:
        flushes = [b for b in range(2, profile_iters + 2) if b % defer == 0]
        fb = sum((defer + (2 if b == defer else 4) * s_active) * n * e for b in flushes) / max(1, profile_iters)
        return {"cgm_pupdate": 3 * n * e, "spmv_dot": spmv, "cgm_update": 3 * n * e, "cgm_flush": fb,
                "cgm_scal1": 0, "cgm_scal2": 0}
    if w.algorithm == "cgm":
        return {"cgm_pupdate": 3 * n * e, "spmv_dot": spmv, "cgm_update": (3 + 4 * s_active) * n * e,
                "cgm_scal1": 0, "cgm_scal2": 0}
    return {"spmv1_dot": spmv + n * e, "spmv2_dots": spmv + 2 * n * e, "bi_supdate": 3 * n * e,
            "bi_update": (7 + 4 * s_active) * n * e, "bi_scal1": 0, "bi_scal2": 0, "bi_scal3": 0}


# The only numbers the paper publishes (Table 1): CG-M, 15 shifts, 2-D
# Poisson 1000x1000, one Tesla T10: 12.9839 ms/iteration fp64, 8.82461 ms/iteration fp32.
PAPER_ITERS_PER_S = {"poisson1000_f64_csr": 1e3 / 12.9839, "poisson1000_f32_csr": 1e3 / 8.82461}


# ----------------------------------------------------------------------------------- clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_bytes(kernel: str, workload: str):
    """(dram read+write bytes per launch, source) of the dominant kernel from the newest committed ncu summary
    that holds a capture of this kernel on this workload -- a STORED figure from one `ncu --set full` capture
    (profiles/*.md names the command and the commit), not something measured in this run -- or (None, None)."""
    for name in ("r02_ncu_dram_traffic.csv", "r01_ncu_dram_traffic.csv"):
        p = os.path.join(ROOT, "profiles", name)
        if not os.path.exists(p):
            continue
        try:
            hit = None
            for ln in open(p):
                f = ln.strip().split(",")
                if len(f) >= 6 and f[0] == kernel and f[5] == workload:
                    hit = f                      # the last row of a kernel is its newest capture
            if hit:
                commit = hit[6] if len(hit) > 6 else "round 1 (see profiles/r01_ncu_dram_traffic.md)"
                return float(hit[1]), "profiles/%s: stored ncu --set full capture taken at commit %s; not re-measured in this run" % (name, commit)
        except Exception:
            continue
    return None, None


# ----------------------------------------------------------------------------------- ranks
def aggregate_over_ranks(times_ms, counts, device, world):
    """Whole-job numbers from per-rank ones: elapsed times -> MAX over ranks, counts -> SUM.
    (device = "cuda" under NCCL, "cpu" under gloo in the CPU test.)"""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return t.tolist(), c.tolist()


def shard_shifts(shifts, rank, world):
    """--shard shifts: rank r solves shifts r, r+world, ... of the same system (same A, same b).  Every
    shift's x_k, conv_iter and residual depend on the base Krylov sequence only, never on the other
    shifts (eq. (2)-(4)), so the union of the ranks' outputs IS the full solve and the
    data path needs no collective.  Interleaved so that every rank gets small and large shifts."""
    return np.ascontiguousarray(np.asarray(shifts)[rank::world])


def throughput(total_iterations, max_ms):
    return total_iterations / (max_ms * 1e-3)


# ----------------------------------------------------------------------------------- oracle legs
def oracle_sample(w, dtype, iters, omp):
    """The CPU oracle, as it stands, on the first `iters` iterations of the same workload (tol = 0: every shift
    stays active).  omp=False: the single-threaded parity build; omp=True: the same source built with -fopenmp,
    loops over rows / elements on all host cores.  The time includes the oracle's own allocation and
    x_k <- 0, p_k <- b initialisation (2 S vectors), which is why a sample is not shorter than ~14 iterations."""
    import oracle
    (oracle.build_omp if omp else oracle.build)()
    fn = oracle.cgm if w.algorithm == "cgm" else oracle.bicgstabm
    t0 = time.perf_counter()
    res = fn(w.rowptr, w.colidx, w.val.astype(dtype, copy=False), w.b.astype(dtype), w.shifts, 0.0, iters, omp=omp)
    dt = time.perf_counter() - t0
    return res.iterations / dt, dt, res.iterations


def host_threads():
    try:
        return int(os.environ.get("OMP_NUM_THREADS", "")) or os.cpu_count()
    except ValueError:
        return os.cpu_count()


def config_dict(args, w, dtype, fmt, world, S, shifts_total):
    """`config` of the JSON line: a function of the workload and the command line only, so that the GPU arm and
    the --impl reference arm print the same keys and values for the same command."""
    e = np.dtype(dtype).itemsize
    if fmt == "bsr3":
        units, spmv = int(w.bcolidx.size), w.bcolidx.size * (9 * e + 4) + (w.n // 3 + 1) * 4 + 2 * w.n * e
    elif fmt == "lat":
        units, spmv = int(w.links.size // 9), w.links.size * e + 2 * w.n * e
    else:
        units, spmv = int(w.nnz), w.nnz * (e + 4) + (w.n + 1) * 4 + 2 * w.n * e
    footprint_mb = (spmv + (4 + 2 * S) * w.n * e) / 1e6
    l2_note = ("inputs larger than L2 (matrix + %d vectors = %.0f MB >> 126 MB), no flush" % (4 + 2 * S, footprint_mb)
               if footprint_mb > 252 else
               "working set %.0f MB (matrix + %d vectors) is not larger than 2 x L2 (126 MB) and is NOT flushed between "
               "iterations: a solve re-reads its own vectors every iteration by construction" % (footprint_mb, 4 + 2 * S))
    return {"workload": args.workload, "extents": args.extents, "algorithm": w.algorithm, "n": w.n, "format": fmt, "nnz_or_blocks": units,
            "shifts": S, "tol": w.tol,
            "parallelism": ("shifts split over %d ranks (%d of %d per rank)" % (world, S, shifts_total)) if args.shard == "shifts" else "replicas x%d" % world,
            "loop_mode": args.loop_mode, "spmv": args.spmv, "update_kernel": args.update_kernel, "defer_update": (32 if args.defer < 0 else args.defer) if args.update_kernel == "regs" else 0, "lattice_kernel": args.lattice_kernel, "x_window": bool(args.x_window), "matrix_l2": args.matrix_l2, "matrix_l2_keep_percent": args.matrix_l2_keep, "iter_path": args.iter_path, "fused_ctas": args.fused_ctas, "l2": l2_note}


def run_reference(args, rank):
    """--impl reference: the oracle on the host cores (all of them: the -fopenmp build of the same source).  Each
    step = the same bounded sample the cpu_baseline leg of the GPU arm times (--cpu-iters iterations, tol = 0)."""
    if rank != 0:
        return
    w, dtype, fmt = make_workload(args.workload, 0, want_csr=True, extents=args.extents)
    per_step = max(args.cpu_iters, 1)
    for _ in range(args.warmup):
        oracle_sample(w, dtype, per_step, True)
    t_tot, it_tot = 0.0, 0
    for _ in range(args.steps):
        _, dt, it = oracle_sample(w, dtype, per_step, True)
        t_tot += dt
        it_tot += it
    value = it_tot / t_tot
    S = int(w.shifts.size)
    sample = ("first %d iterations of %s per step (tol=0), all %d shifts active, OpenMP build of the oracle on %d threads"
              % (per_step, w.name, S, host_threads()))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
            "higher_is_better": True, "scaling": "strong" if args.shard == "shifts" else "weak", "vs_baseline": None,
            "dtype": DTYPE_NAME[dtype], "data": "synthetic",
            "config": config_dict(args, w, dtype, fmt, int(os.environ.get("WORLD_SIZE", "1")), S, S),
            "oracle_reads": "the same operator assembled as CSR (rowptr/colidx/val), whatever `format` the GPU arm takes",
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": host_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_slabs(args, ms, torch, w, dtype, fmt):
    """--slabs P: the same solves through P row slabs on one device (no per-kernel table, no e2e leg)."""
    if fmt == "lat":
        raise SystemExit("--slabs takes the assembled forms (bsr3 / csr)")
    tdt = {np.complex128: torch.complex128, np.complex64: torch.complex64, np.float64: torch.float64, np.float32: torch.float32}[dtype]
    t0 = time.perf_counter()
    if fmt == "bsr3":
        S_ = ms.msolve_slabs_create_bsr3(w.browptr, w.bcolidx, w.blocks.astype(dtype, copy=False), args.slabs)
    else:
        S_ = ms.msolve_slabs_create_csr(w.rowptr, w.colidx, w.val.astype(dtype, copy=False), args.slabs)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t0
    solve = ms.msolve_slabs_cgm if w.algorithm == "cgm" else ms.msolve_slabs_bicgstabm
    b_dev = torch.from_numpy(w.b.astype(dtype)).cuda()
    nS = int(w.shifts.size)
    x_dev = torch.empty((nS, w.n), dtype=tdt, device="cuda")
    for _ in range(args.warmup):
        res = solve(S_, b_dev, w.shifts, w.tol, w.max_iter, x=x_dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    iters, launches = 0, 0
    ev0.record()
    for _ in range(args.steps):
        res = solve(S_, b_dev, w.shifts, w.tol, w.max_iter, x=x_dev)
        iters += res.iterations
        launches += ms.msolve_slabs_last_launch_count(S_)
    ev1.record()
    torch.cuda.synchronize()
    ms_total = ev0.elapsed_time(ev1)
    halo = ms.msolve_slabs_halo_elements(S_)
    cfg = config_dict(args, w, dtype, fmt, 1, nS, nS)
    cfg["parallelism"] = "%d row slabs on one device (halo exchange + summed dot products, csrc/slab.cu)" % args.slabs
    line = {"metric": METRIC, "value": throughput(iters, ms_total), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": DTYPE_NAME[dtype], "data": "synthetic", "config": cfg,
            "iterations_per_solve": iters / args.steps, "status": res.status, "create_ms": 1e3 * t_create,
            "halo_elements_per_slab": halo, "halo_bytes_per_exchange": int(sum(halo)) * np.dtype(dtype).itemsize,
            "gpu_launches": int(launches)}
    print(json.dumps(line))
    ms.msolve_slabs_destroy(S_)


# ----------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4_c128_bsr3")
    ap.add_argument("--profile-iters", type=int, default=20)
    ap.add_argument("--cpu-iters", type=int, default=14, help="oracle iterations timed per cpu_baseline sample / per --impl reference step (0 = skip)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--spmv", default="auto", choices=["auto", "vector", "merge", "tile"],
                    help="SpMV kernel for CSR workloads (BSR3: auto = TMA tile kernel, vector = row kernel)")
    ap.add_argument("--lattice-kernel", type=int, default=0, choices=[0, 1, 2, 3, 4],
                    help="tile kernel of the lattice operator (MSOLVE_CFG_LATTICE_KERNEL; 0 = default per element type)")
    ap.add_argument("--extents", type=lambda t: [int(v) for v in t.split(",")], default=None,
                    help="config4_c128_bsr3 / config4_c128_lat on another lattice, e.g. 16,16,16,16 (size sweeps)")
    ap.add_argument("--defer", type=int, default=-1,
                    help="CG-M: chunk length of the deferred multishift update (MSOLVE_CFG_DEFER_UPDATE; 0 = update "
                         "every x_k, p_k in every iteration; -1 = the library's default, 32)")
    ap.add_argument("--update-kernel", default="regs", choices=["regs", "tma"],
                    help="CG-M fused multishift update: register kernel (default) or the TMA-staged kernel")
    ap.add_argument("--x-window", action="store_true",
                    help="vector-CSR kernel: L2 access-policy window over the gathered vector (MSOLVE_CFG_X_WINDOW)")
    ap.add_argument("--iter-path", default="auto", choices=["auto", "graph", "fused", "resident"],
                    help="graph: iteration as a CUDA graph of kernels; fused: whole solve in one cooperative kernel "
                         "(L2-resident systems); resident: one kernel, matrix and vectors in shared memory (CG-M, a few "
                         "MB); auto: by footprint (MSOLVE_CFG_ITER_PATH)")
    ap.add_argument("--fused-ctas", type=int, default=0, help="CTAs of the one-kernel path (0 = by problem size)")
    ap.add_argument("--matrix-l2", default="auto", choices=["auto", "stream", "keep"],
                    help="L2 policy of the matrix stream (MSOLVE_CFG_MATRIX_L2)")
    ap.add_argument("--phase-clock", action="store_true",
                    help="one-kernel path: also report the microseconds per iteration CTA 0 spends in every phase "
                         "(msolve_set_phase_clock; extra solves after the timed region)")
    ap.add_argument("--matrix-l2-keep", type=int, default=0,
                    help="percent of the matrix stream loaded evict-last (MSOLVE_CFG_MATRIX_L2_KEEP_PERCENT)")
    ap.add_argument("--slabs", type=int, default=0,
                    help="row partition on ONE device (msolve_slabs_*, SURVEY 8(f)-3): P slabs with halo exchange and "
                         "summed dot products; measures what the partition costs against the unpartitioned solve")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "shifts"],
                    help="N > 1: replicas = every rank solves the whole family for its own right-hand side (weak "
                         "scaling, default); shifts = the ranks split the shifts of ONE system (strong scaling)")
    ap.add_argument("--loop-mode", default="while", choices=["while", "chunk"],
                    help="while: device WHILE graph node (default). chunk: unrolled graph relaunched by the host; "
                         "same kernels, used for ncu (kernel nodes of conditional graphs cannot be profiled)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                      # timing rule: W >= 3
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_1102_2143_b200 import binding as ms, build as _build

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        if local_rank == 0:
            _build.build()                                   # one compile per node, the other ranks wait
        dist.barrier()
    else:
        _build.build()
    ms.load_library()

    need_csr = args.workload.endswith("_csr") or (rank == 0 and world == 1 and args.cpu_iters > 0)
    w, dtype, fmt = make_workload(args.workload, 0 if args.shard == "shifts" else rank, want_csr=need_csr, extents=args.extents)
    shifts_total = int(w.shifts.size)
    if args.shard == "shifts":
        if world > shifts_total:
            raise SystemExit("--shard shifts needs at least one shift per rank")
        w.shifts = shard_shifts(w.shifts, rank, world)
    tdt = {np.complex128: torch.complex128, np.complex64: torch.complex64,
           np.float64: torch.float64, np.float32: torch.float32}[dtype]
    alg = ms.MSOLVE_ALG_CGM if w.algorithm == "cgm" else ms.MSOLVE_ALG_BICGSTABM
    solve = ms.msolve_cgm if w.algorithm == "cgm" else ms.msolve_bicgstabm

    def dev(a):
        return torch.from_numpy(np.ascontiguousarray(a)).cuda()

    if args.slabs > 0:
        run_slabs(args, ms, torch, w, dtype, fmt)
        return
    t_create = time.perf_counter()
    flags = {"auto": ms.MSOLVE_SPMV_AUTO, "vector": ms.MSOLVE_SPMV_VECTOR, "merge": ms.MSOLVE_SPMV_MERGE, "tile": ms.MSOLVE_SPMV_TILE}[args.spmv]
    if fmt == "bsr3":
        A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks.astype(dtype, copy=False)), flags)
    elif fmt == "lat":
        m = w.meta
        A = ms.msolve_create_lattice_su3(m["extents"], dev(w.links.astype(dtype, copy=False)), m["diag"], m["c_f"],
                                         m["c_b"], flags)
    else:
        A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype, copy=False)), flags)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t_create
    ms.msolve_config(A, ms.MSOLVE_CFG_LOOP_MODE, 0 if args.loop_mode == "while" else 1)
    ms.msolve_config(A, ms.MSOLVE_CFG_UPDATE_KERNEL, 1 if args.update_kernel == "tma" else 0)
    if args.lattice_kernel:
        ms.msolve_config(A, ms.MSOLVE_CFG_LATTICE_KERNEL, args.lattice_kernel)
    if args.defer >= 0:
        ms.msolve_config(A, ms.MSOLVE_CFG_DEFER_UPDATE, args.defer)
    if args.x_window:
        ms.msolve_config(A, ms.MSOLVE_CFG_X_WINDOW, 1)
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, {"auto": 0, "graph": 1, "fused": 2, "resident": 3}[args.iter_path])
    ms.msolve_config(A, ms.MSOLVE_CFG_FUSED_CTAS, args.fused_ctas)
    ms.msolve_config(A, ms.MSOLVE_CFG_MATRIX_L2, {"auto": 0, "stream": 1, "keep": 2}[args.matrix_l2])
    if args.matrix_l2_keep:
        ms.msolve_config(A, ms.MSOLVE_CFG_MATRIX_L2_KEEP_PERCENT, args.matrix_l2_keep)
    S = int(w.shifts.size)
    b_host = torch.from_numpy(w.b.astype(dtype)).pin_memory()
    b_dev = b_host.cuda()
    x_dev = torch.empty((S, w.n), dtype=tdt, device="cuda")
    ws = torch.empty(ms.msolve_workspace_bytes(A, S, alg), dtype=torch.uint8, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K complete solves
    for _ in range(args.warmup):
        res = solve(A, b_dev, w.shifts, w.tol, w.max_iter, x=x_dev, workspace=ws)
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    iters, launches = 0, 0
    ev0.record()
    for _ in range(args.steps):
        res = solve(A, b_dev, w.shifts, w.tol, w.max_iter, x=x_dev, workspace=ws)
        iters += res.iterations
        launches += ms.msolve_last_launch_count(A)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    status, conv_iter = res.status, res.conv_iter.tolist()
    phases = None
    if args.phase_clock:
        # one-kernel path only: where CTA 0 spends an iteration (msolve_set_phase_clock), over `steps` more solves
        ns = torch.zeros(16, dtype=torch.int64, device="cuda")
        ms.msolve_set_phase_clock(A, ns)
        for _ in range(args.steps):
            solve(A, b_dev, w.shifts, w.tol, w.max_iter, x=x_dev, workspace=ws)
        ms.msolve_set_phase_clock(A, None)
        t = ns.cpu().numpy().astype(np.float64)
        names = (["p_update", "barrier", "spmv_dot", "barrier_sum", "scalars_update", "barrier_sum2"] if alg == ms.MSOLVE_ALG_CGM else
                 ["spmv1_dot", "barrier_sum", "scalars_s_update", "barrier", "spmv2_dots", "barrier_sum5", "scalars_update", "barrier_sum1"])
        if t[15] > 0:
            phases = {k: round(v / t[15] / 1e3, 2) for k, v in zip(names, t)}
            phases["sum"] = round(float(t[:len(names)].sum()) / t[15] / 1e3, 2)
            phases["iterations"] = int(t[15])

    # ---- end to end: host b in, host x out, every step.  The K steps go through ONE call of the public
    # batch interface (msolve_solve_host_batch: K right-hand sides of the same family), which overlaps the
    # D2H copy of step i with the solve of step i+1; every step's H2D and D2H are inside the timed region.
    # e2e_single is the same through K separate msolve_solve_host calls (nothing overlapped).
    e2e = None
    if not args.no_e2e:
        x_hosts = [torch.empty((S, w.n), dtype=tdt, pin_memory=True) for _ in range(2)]
        xs = [x_hosts[i & 1] for i in range(args.steps)]      # results land in two pinned buffers in turn
        bs = [b_host] * args.steps
        ms.msolve_solve_host_batch(A, alg, bs[:2], w.shifts, w.tol, w.max_iter, xs=xs[:2])
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        rs = ms.msolve_solve_host_batch(A, alg, bs, w.shifts, w.tol, w.max_iter, xs=xs)
        e1.record()
        barrier()
        it_e2e = sum(r.iterations for r in rs)
        ms_e2e = e0.elapsed_time(e1)
        for _ in range(2):
            ms.msolve_solve_host(A, alg, b_host, w.shifts, w.tol, w.max_iter, x=x_hosts[0])
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        it_single = 0
        s0.record()
        for _ in range(args.steps):
            it_single += ms.msolve_solve_host(A, alg, b_host, w.shifts, w.tol, w.max_iter, x=x_hosts[0]).iterations
        s1.record()
        barrier()
        ms_single = s0.elapsed_time(s1)
        e2e = (it_e2e, ms_e2e, b_host.numel() * b_host.element_size() + 8 * S,
               x_hosts[0].numel() * x_hosts[0].element_size(), it_single, ms_single)
        del x_hosts, xs

    # ---- per-kernel steady state (all shifts active), CUDA events around every kernel launch
    prof = ms.msolve_profile_iteration(A, alg, b_dev, w.shifts, args.profile_iters, x=x_dev, workspace=ws)
    torch.cuda.synchronize()

    # ---- CG-M with the deferred multishift update (the default): the same solves once more with the update of every
    # x_k, p_k in every iteration (MSOLVE_CFG_DEFER_UPDATE = 0, Alg. 1 l.28-29 step by step), so that the line carries
    # the fused multishift-update kernel and the iteration rate of that form as well (rank 0 reports its own numbers)
    stepwise = None
    defer_now = 0 if (w.algorithm != "cgm" or args.update_kernel != "regs") else (32 if args.defer < 0 else args.defer)
    if defer_now > 0 and args.iter_path in ("auto", "graph") and ms.msolve_last_launch_count(A) > 1:
        ms.msolve_config(A, ms.MSOLVE_CFG_DEFER_UPDATE, 0)
        for _ in range(2):
            solve(A, b_dev, w.shifts, w.tol, w.max_iter, x=x_dev, workspace=ws)
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        it0 = 0
        t0.record()
        for _ in range(args.steps):
            it0 += solve(A, b_dev, w.shifts, w.tol, w.max_iter, x=x_dev, workspace=ws).iterations
        t1.record()
        torch.cuda.synchronize()
        prof0 = ms.msolve_profile_iteration(A, alg, b_dev, w.shifts, args.profile_iters, x=x_dev, workspace=ws)
        torch.cuda.synchronize()
        ms.msolve_config(A, ms.MSOLVE_CFG_DEFER_UPDATE, defer_now)
        stepwise = (it0, t0.elapsed_time(t1), prof0)

    # ---- reduce over ranks
    (ms_total, ms_e2e, ms_single), (iters_all, launches_all, it_e2e_all, it_single_all) = aggregate_over_ranks(
        [ms_total, e2e[1] if e2e else 0.0, e2e[5] if e2e else 0.0],
        [iters, launches, e2e[0] if e2e else 0, e2e[4] if e2e else 0], "cuda", world)
    if args.shard == "shifts" and world > 1:
        # one system: the job's iteration count is that of its slowest shift (MAX over ranks, not SUM)
        (it_max, it_e2e_max, it_single_max), _ = aggregate_over_ranks(
            [float(iters), float(e2e[0] if e2e else 0), float(e2e[4] if e2e else 0)], [0], "cuda", world)
        iters_all, it_e2e_all, it_single_all = it_max, it_e2e_max, it_single_max

    if rank == 0:
        peak, peak_src = measured_peak_gbs()
        defer = 0 if (w.algorithm != "cgm" or args.update_kernel != "regs") else (32 if args.defer < 0 else args.defer)
        ab = algorithmic_bytes(w, dtype, fmt, S, defer, args.profile_iters)
        kernels = {}
        for name, kms in prof.items():
            gbs = ab.get(name, 0) / (kms * 1e-3) / 1e9 if kms > 0 else 0.0
            kernels[name] = {"ms": round(kms, 5), "alg_GB": round(ab.get(name, 0) / 1e9, 4),
                             "GBps": round(gbs, 1), "frac_measured_peak": round(gbs / peak, 4),
                             "frac_8TBps": round(gbs / 8000.0, 4)}
        # the dominant kernel: the one an iteration spends most of its time in (the fused multishift update while it
        # runs in every iteration; the SpMV once the update is deferred)
        dom = max((k for k in kernels if ab.get(k, 0) > 0), key=lambda k: kernels[k]["ms"])
        traffic, traffic_src = ncu_traffic_bytes(dom, args.workload)
        roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["GBps"], "peak": peak,
                    "unit": "GB/s", "frac": round(kernels[dom]["GBps"] / peak, 4), "peak_source": peak_src,
                    "traffic": traffic, "traffic_source": traffic_src, "algorithmic_bytes_per_launch": ab[dom]}
        iter_ms = sum(v["ms"] for v in kernels.values())
        cpu = None
        if args.cpu_iters > 0 and world == 1:
            v, dt, it = oracle_sample(w, dtype, args.cpu_iters, True)
            v1, dt1, it1 = oracle_sample(w, dtype, max(args.cpu_iters // 2, 1), False)
            cpu = {"value": v, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
                   "sample": "first %d iterations of %s (tol=0, all %d shifts active), %.1f s, OpenMP build of the oracle "
                             "(same source, -fopenmp) on %d threads; allocation and p_k/x_k initialisation included"
                             % (it, w.name, S, dt, host_threads()),
                   "single_thread_value": v1,
                   "single_thread_sample": "first %d iterations, %.1f s, the parity build (one thread)" % (it1, dt1)}
        line = {
            "metric": METRIC, "value": throughput(iters_all, ms_total), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_total / args.steps,
            "higher_is_better": True, "scaling": "strong" if args.shard == "shifts" else "weak",
            "vs_baseline": (throughput(iters_all, ms_total) / (1 if args.shard == "shifts" else world) / PAPER_ITERS_PER_S[args.workload]
                            if args.workload in PAPER_ITERS_PER_S else None),
            "dtype": DTYPE_NAME[dtype], "data": "synthetic",
            "config": config_dict(args, w, dtype, fmt, world, S, shifts_total),
            "time_to_solution_ms": ms_total / args.steps, "iterations_per_solve": iters_all / args.steps / (1 if args.shard == "shifts" else world),
            "status": status, "conv_iter": conv_iter, "create_ms": 1e3 * t_create,
            "steady_state_ms_per_iteration": round(iter_ms, 4),
            "steady_state_iterations_per_s": round(1e3 / iter_ms, 2) if iter_ms > 0 else None,
            "kernels": kernels, "roofline": roofline, "cpu_baseline": cpu,
            "e2e": None if e2e is None else {"value": throughput(it_e2e_all, ms_e2e), "unit": UNIT,
                                             "h2d_bytes_per_step": e2e[2], "d2h_bytes_per_step": e2e[3],
                                             "ms_per_step": ms_e2e / args.steps,
                                             "api": "msolve_solve_host_batch, %d right-hand sides (D2H of step i overlaps the solve of step i+1)" % args.steps,
                                             "single_call_value": throughput(it_single_all, ms_single),
                                             "single_call_api": "msolve_solve_host per step, nothing overlapped"},
            "gpu_launches": int(launches_all), "clocks": clocks,
        }
        if stepwise is not None:
            it0, ms0, prof0 = stepwise
            ab0 = algorithmic_bytes(w, dtype, fmt, S, 0, args.profile_iters)
            k0 = {}
            for name, kms in prof0.items():
                gbs = ab0.get(name, 0) / (kms * 1e-3) / 1e9 if kms > 0 else 0.0
                k0[name] = {"ms": round(kms, 5), "alg_GB": round(ab0.get(name, 0) / 1e9, 4), "GBps": round(gbs, 1),
                            "frac_measured_peak": round(gbs / peak, 4), "frac_8TBps": round(gbs / 8000.0, 4)}
            tr0, tr0_src = ncu_traffic_bytes("cgm_update", args.workload)
            line["stepwise_update"] = {
                "what": "the same solves with MSOLVE_CFG_DEFER_UPDATE = 0: every x_k, p_k updated in every iteration (Alg. 1 l.28-29 step by step)",
                "value": throughput(it0, ms0), "unit": UNIT, "ms_per_step": ms0 / args.steps, "kernels": k0,
                "roofline": {"bound": "hbm", "kernel": "cgm_update", "achieved": k0["cgm_update"]["GBps"], "peak": peak, "unit": "GB/s",
                             "frac": round(k0["cgm_update"]["GBps"] / peak, 4), "traffic": tr0, "traffic_source": tr0_src,
                             "algorithmic_bytes_per_launch": ab0["cgm_update"]}}
        if phases is not None:
            line["one_kernel_phases_us_per_iteration"] = phases
        print(json.dumps(line))
    ms.msolve_destroy(A)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
