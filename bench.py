#!/usr/bin/env python
"""bench.py -- time-to-solution of the dense complex-FP64 Hermitian eigensolve on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--nev NEV] [--impl reference]

A "step" is one pass of the whole hot path (eigh_solve: full->band, band->tridiagonal, tridiagonal D&C, both
back-transformations) over one synthetic matrix of BASELINE.json's `configs`.  Default workload = config 4, the
N = 49152 BdG vortex-tangle matrix (the largest single-GPU config and the north_star target).  BASELINE.json lists
two runs for it, "full eigendecomposition and nev = N/2 subset": all eigenpairs are computed when W + K full solves
fit the time budget (--time-budget, default 1500 s: the default W = 3, K = 2 run does), otherwise the nev = N/2 run is
timed (the driver's --steps 20 --warmup 5: 25 x 72.5 s does not fit its 1800 s limit, 25 x 45.5 s does); which one ran is
stated in `config.nev` / `config.nev_rule`.  The rule is a pure function of (config, W, K, budget), so both arms of
the driver's comparison make the same choice.  The matrix is regenerated in place (eigh_assemble_bdg on the device, or
a device copy of a pristine matrix for config 1) OUTSIDE the per-step CUDA-event brackets, because eigh_solve
overwrites A.

One JSON line on stdout (rank 0):  metric = eigh_time_s (seconds per eigensolve, lower is better), plus `phases`
(ms, credited / executed TFLOP/s or GB/s per phase, S3 merge statistics), `roofline` (the dominant kernel against the
FP64 tensor peak), `e2e` (host buffers through eigh_solve_host), `cpu_baseline` (the oracle on a bounded sample) and
`clocks`.

Multi-GPU: the path does not shard ("replicas only"): every rank solves its own replica,
value = max-over-ranks time / n_gpus.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 37.2: 148 SMs x 64 FP64 FMA/clk/SM x 1.965 GHz
CLOCK_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
               "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
               "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
PHASES = ["p1_full_to_band", "p2_band_to_tridiag", "p3_tridiag_dc", "p4a_backtransform_band", "p4b_backtransform_full"]
# seconds per eigh_solve (all eigenpairs) measured on one B200 for the nev rule; source: profiles/r01_summary.md and
# profiles/r02_summary.md.  Only used to decide between the two runs BASELINE.json lists for configs 3 and 4.
FULL_SOLVE_MODEL_S = {0: 0.03, 1: 0.2, 2: 0.6, 3: 13.5, 4: 72.5}
# executed real FP64 tensor flops per credited flop: GEMM engine in the 3M form = 6/8; bt_sweep_kernel: 116 DMMAs of
# 512 flops per compact-WY block of 8 reflectors x 8 columns, credited 2 x 8 x 64 x 8 x 8
EXECUTED_PER_CREDITED = {"p1": 0.75, "p4a": 116 * 512 / 65536.0, "p4b": 0.75}


def credited_work(N: int, nev: int, b: int):
    """Credited algorithmic work per phase (lower-order terms dropped)."""
    steps = 0
    for j in range(0, N - 1):
        steps += -(-(N - 1 - j) // b)
    # per chase step: D lower (b^2/2) + S (b^2) read and written, 16 B each; reflector b written
    bytes_p2 = steps * (2 * (b * b // 2 + b * b) * 16 + b * 16)
    return {
        "p1_flops": 16.0 / 3.0 * N ** 3,
        "p2_flops": 24.0 * b * N * N,
        "p2_bytes": float(bytes_p2),
        "p2_steps": steps,
        "p4a_flops": 8.0 * N * N * nev,
        "p4b_flops": 8.0 * N * N * nev,
    }


def choose_nev(config: int, N: int, nev_runs, warmup: int, steps: int, budget_s: float, nev_arg: int = 0):
    """The run of BASELINE.json's config that is timed: (nev, rule text).  Deterministic in its arguments."""
    if nev_arg > 0:
        return min(nev_arg, N), "--nev given"
    full = (warmup + steps) * FULL_SOLVE_MODEL_S.get(config, 75.0)
    if len(nev_runs) < 2 or full <= budget_s:
        return N, "all eigenpairs: (W + K) x %.1f s = %.0f s fits the %.0f s budget" % (
            FULL_SOLVE_MODEL_S.get(config, 75.0), full, budget_s)
    return int(nev_runs[1]), ("nev = N/2 run of BASELINE.json's config (lowest N/2 pairs): (W + K) x %.1f s = %.0f s of full "
                              "solves exceed the %.0f s budget" % (FULL_SOLVE_MODEL_S.get(config, 75.0), full, budget_s))


def config_dict(w, nev: int, rule: str, b: int = 64):
    """`config` of the JSON line -- the same keys and values in both arms (--impl ours / reference)."""
    return {"workload": w.name, "N": w.N, "nev": nev, "nev_rule": rule, "band_width": b,
            "parallelism": "replicas only",
            "l2": "inputs larger than L2 (matrix %.1f GB)" % (w.N * w.N * 16 / 1e9),
            "input_regeneration": "on the device, outside the timed brackets"}


class ClockSampler:
    def __init__(self, gpu_index: int):
        self.rows = []
        self.proc = None
        self.idx = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={CLOCK_QUERY}", "--format=csv,noheader,nounits", "-lms", "200",
                 "-i", str(self.idx)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, pw, reasons = [], [], [], set()
        for ts, line in self.rows:
            if ts < t0 or ts > t1 + 0.3:
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def max_over_ranks(value_ms: float, dist, device=None) -> float:
    """Timing rule for N > 1: the job's time is the MAX over ranks of the device-timed total (replicas only:
    no collective on the data path, this all-reduce of one scalar happens after the timed region)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value_ms)
    import torch
    t = torch.tensor([value_ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_value_s(ms_per_step: float, world: int) -> float:
    """Whole-job metric for `world` independent replicas: seconds per eigensolve = step time / replicas."""
    return ms_per_step / 1e3 / world


def oracle_sample(w, ns):
    """A bounded sample of the workload for the CPU oracle: the leading ns x ns block of the dense matrix when it is
    affordable (N <= 8192), else the same recipe (fields, mu) restricted to a sub-lattice with 2 nx ny nz <= ns (not
    the same matrix: stated in `sample`).  Returns (matrix, description)."""
    import numpy as np
    if w.problem is None or w.N <= 8192:
        H = np.ascontiguousarray(w.dense()[:ns, :ns])
        return H, f"leading {H.shape[0]} x {H.shape[0]} block of the matrix"
    from paper_2310_03341_b200 import workloads as wl
    p = w.problem
    nx, ny, nz = p.shape
    while 2 * nx * ny * nz > ns:
        if nx >= ny and nx >= nz: nx //= 2
        elif ny >= nz: ny //= 2
        else: nz //= 2
    idx = np.arange(np.prod(p.shape)).reshape(p.shape)[:nx, :ny, :nz].reshape(-1)
    q = wl.BdGProblem(p.name, (nx, ny, nz), p.mu, p.V[idx], p.Delta[idx])
    H = q.dense()
    return H, f"the same recipe (fields, mu) on the {nx}x{ny}x{nz} sub-lattice, order {H.shape[0]}"


def reference_arm(args, wl_mod):
    """--impl reference: the CPU oracle (unmodified, as it stands; all eigenpairs -- it has no subset mode) on a
    bounded sample of the workload, timed per step on the box's host cores and scaled by (N/n_s)^3 (the oracle is a
    23 N^3 level-1/2 method)."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = wl_mod.make_config(args.config)
    N = w.N
    nev, rule = choose_nev(args.config, N, w.nev_runs, args.warmup, args.steps, args.time_budget, args.nev)
    H, what = oracle_sample(w, min(N, args.ref_sample))
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.eigh(H)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
    per = sum(times) / len(times)
    ns = H.shape[0]
    est = per * (N / ns) ** 3
    line = {
        "impl": "reference", "metric": "eigh_time_s", "value": est, "unit": "s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": est * 1e3, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
        "config": config_dict(w, nev, rule),
        "cpu_baseline": {"value": est, "unit": "s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": f"{what}: {per:.3f} s per step measured (all eigenpairs), scaled by (N/{ns})^3",
                         "measured_s": per, "measured_order": ns},
        "e2e": {"value": est, "unit": "s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def kernel_source_sha(name: str) -> str:
    with open(os.path.join(ROOT, "paper_2310_03341_b200", "csrc", name), "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()[:16]


def lookup_traffic(workload: str, nev: int):
    """DRAM bytes (read + write) of one bt_sweep_kernel launch from an ncu capture -- only if the capture recorded in
    profiles/traffic.json was taken on this workload, this nev and THIS source of the kernel (sha of bt_band.cu)."""
    try:
        entries = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    except Exception:
        return None, "no profiles/traffic.json"
    sha = kernel_source_sha("bt_band.cu")
    for e in entries:
        if e.get("workload") == workload and e.get("nev") == nev and e.get("source_sha") == sha:
            return float(e["dram_bytes"]), e.get("capture")
    return None, "no ncu capture of this kernel source (sha %s) on this workload / nev" % sha


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=int(os.environ.get("EIGH_BENCH_CONFIG", "4")))
    ap.add_argument("--nev", type=int, default=0, help="0 = the run chosen by the time budget (all eigenpairs or N/2)")
    ap.add_argument("--time-budget", type=float, default=1500.0,
                    help="seconds available for the W + K solves; decides between the two runs of configs 3 / 4")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--ref-sample", type=int, default=3456, help="order of the oracle sample of --impl reference")
    ap.add_argument("--cpu-sample", type=int, default=3456,
                    help="order of the oracle's sample (about 10-30 s of CPU work on the box's host cores)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--host-buffers", default="pinned", choices=("pinned", "pageable"),
                    help="e2e leg: host buffers page-locked in place (cudaHostRegister; falls back to pageable when the "
                         "registration fails) or plain pageable memory through the handle's 2 x 256 MiB pinned ring")
    ap.add_argument("--no-epilogue", action="store_true")
    ap.add_argument("--context", action="store_true",
                    help="also time library routines on the same matrix as CONTEXT (never the target, never on the hot path): "
                         "torch.linalg.eigh (cuSOLVER) on this GPU and numpy.linalg.eigh (LAPACK) on the CPU sample")
    ap.add_argument("--opt", action="append", default=[], help="solver option key=value (eigh_set_option), repeatable")
    ap.add_argument("--method", type=int, default=2, choices=(1, 2),
                    help="2 = two-stage solver (the hot path, default); 1 = the 1-stage variant of SURVEY.md 8(f)2 "
                         "(PAPER.md:148 steps i-iii; use with --config 0..2)")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1 only, NOT the default (the path is 'replicas only'): strong-scaling run of ONE problem with "
                         "the back-transformations sharded by eigenvector columns (option col_begin; S1-S3 replicated, Z "
                         "left distributed, no collective on the data path) -- SURVEY.md 8(f)3 first slice, DESIGN.md 3.10")
    ap.add_argument("--real", action="store_true",
                    help="real-symmetric FP64 path (needs --method 1 and a real matrix: --config 0)")
    args = ap.parse_args()
    # W >= 3 is the timing rule for a valid bench number; smaller values are accepted for profiler runs only
    # (ncu launch lists), whose printed numbers are never bench values
    if args.warmup < 0:
        args.warmup = 0

    from paper_2310_03341_b200 import workloads as wl_mod
    if args.impl == "reference":
        reference_arm(args, wl_mod)
        return

    import numpy as np
    import torch
    from paper_2310_03341_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    w = wl_mod.make_config(args.config)
    N = w.N
    nev, nev_rule = choose_nev(args.config, N, w.nev_runs, args.warmup, args.steps, args.time_budget, args.nev)
    opts = {}
    if args.method == 1:
        opts["method"] = 1
        if args.real:
            opts["dtype"] = 1
    for kv in args.opt:
        key, val = kv.split("=")
        opts[key] = int(val)
    nev_total = nev
    sharded = args.shard and world > 1
    if sharded:
        from paper_2310_03341_b200 import shard as shard_mod
        c0, c1 = shard_mod.column_shards(nev_total, world)[rank]
        nev = max(c1 - c0, 1)
        opts["col_begin"] = min(c0, N - nev)
    solver = binding.Eigh(N, nev, device=dev, **opts)
    b = solver.band_width                                    # read from the handle (eigh_get_option)
    mat_bytes = N * N * 16
    wdt = solver.dtype                                       # complex128, or float64 on the real-symmetric path
    At = torch.empty((N, N), dtype=wdt, device=dev)          # A column-major (stored as A^T row-major)
    W = torch.empty(N, dtype=torch.float64, device=dev)
    Zt = torch.empty((nev, N), dtype=wdt, device=dev)
    pristine = None
    fields = None
    if args.real:
        tmp = torch.empty((N, N), dtype=torch.complex128, device=dev)
        w.dense_torch(dev, out=tmp)
        assert float(tmp.imag.abs().max().item()) == 0.0, "--real needs a real matrix (config 0)"
        pristine = tmp.real.contiguous()
        del tmp
    elif w.problem is not None:
        # BdG configs: H is re-assembled on the device from its fields by the library's own prologue kernel
        pb = w.problem
        fields = ([torch.from_numpy(wl_mod.kinetic_1d(L)).to(dev) for L in pb.shape],
                  torch.from_numpy(pb.V).to(dev), torch.from_numpy(np.ascontiguousarray(pb.Delta)).to(dev))
    else:
        pristine = torch.empty((N, N), dtype=torch.complex128, device=dev)
        w.dense_torch(dev, out=pristine)

    def regenerate():
        if fields is not None:
            K3, Vd, Dd = fields
            solver.assemble_bdg(w.problem.shape, K3[0], K3[1], K3[2], Vd, Dd, w.problem.mu, At=At)
        else:
            At.copy_(pristine)

    stream = torch.cuda.current_stream()
    ev0 = torch.cuda.Event(enable_timing=True)
    ev1 = torch.cuda.Event(enable_timing=True)

    def one_step():
        regenerate()
        ev0.record(stream)
        solver.solve(At, W, Zt)
        ev1.record(stream)
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1), solver.phase_times_ms() + [solver.kernel_time_ms("bt_sweep_kernel")], solver.launch_count()

    for _ in range(args.warmup):
        one_step()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.time()
    step_ms, phases, launches = [], [], 0
    for _ in range(args.steps):
        ms, ph, ln = one_step()
        step_ms.append(ms)
        phases.append(ph)
        launches += ln
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t1 = time.time()
    total_ms = sum(step_ms)
    total_ms = max_over_ranks(total_ms, dist, dev)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ms_per_step = total_ms / args.steps
    value_s = replica_value_s(ms_per_step, world)        # seconds per eigensolve, whole job (replicas)
    if sharded:
        value_s = ms_per_step / 1e3                      # one problem solved by all ranks together
    dc_flops, dc_kept = solver.dc_stats()                # S3 merge statistics of the last solve

    # ---- quick validity check of the last solve (device side, independent ZGEMM by torch)
    valid = {}
    if rank == 0:
        with torch.no_grad():
            regenerate()
            Hl = At.t()                                          # logical H (all N^2 elements are valid)
            if args.real:
                Hl = Hl.to(torch.complex128)
            ncheck = min(nev, 256)
            cols = torch.linspace(0, nev - 1, ncheck, device=dev).long()
            Zc = Zt[cols].t().to(torch.complex128)              # N x ncheck
            R = Hl @ Zc - Zc * W[cols][None, :]
            hn = float(torch.linalg.norm(Hl).item())
            valid["residual_sampled"] = float(torch.linalg.norm(R).item()) / (hn * (ncheck ** 0.5))
            valid["orth_sampled"] = float((Zc.conj().t() @ Zc - torch.eye(ncheck, device=dev)).abs().max().item())
            valid["trace_err"] = abs(float(W.sum().item()) - float(torch.diagonal(Hl).real.sum().item()))
            del R, Zc

    hbm = None
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        hbm = peaks.get("hbm_gbs")
    except Exception:
        pass

    # ---- SCF epilogue (outside the timed step): eigh_densities on the eigenpairs just computed,
    # Eq. 16a/16d at T = 0.  HBM-bound: algorithmic bytes = the u and v halves of every ACTIVE column of Z read once
    # (16 N bytes per column) + the two output fields; CUDA events on the launching stream.
    epilogue = None
    if rank == 0 and w.problem is not None and N % 2 == 0 and not args.no_epilogue and not args.real:
        try:
            branch = 1 if nev == N else -1                       # lowest N/2 pairs: particle-hole partners (reading 3)
            E = W[:nev].contiguous()
            n_f, nu_f = solver.densities(E, Zt, T=0.0, branch=branch)
            torch.cuda.synchronize()
            ts = []
            for _ in range(5):
                ev0.record(stream)
                solver.densities(E, Zt, T=0.0, branch=branch, n=n_f, nu=nu_f)
                ev1.record(stream)
                torch.cuda.synchronize()
                ts.append(ev0.elapsed_time(ev1))
            active = int((E > 0).sum().item()) if branch == 1 else int((E < 0).sum().item())
            dbytes = 16.0 * N * active + 24.0 * (N // 2)
            dms = sorted(ts)[len(ts) // 2]
            epilogue = {"op": "eigh_densities (Eq. 16a, 16d; T = 0; branch %+d)" % branch, "ms": dms,
                        "active_columns": active, "algorithmic_bytes": dbytes, "bound": "hbm",
                        "achieved_gbs": dbytes / dms / 1e6 if dms else None, "peak_gbs": hbm,
                        "frac": (dbytes / dms / 1e6) / hbm if hbm and dms else None, "launches": 3,
                        "particle_number": float(n_f.sum().item()),
                        "note": "inputs (%.1f GB of active columns) larger than L2" % (16.0 * N * active / 1e9)}
            pb = w.problem
            Dd = [torch.from_numpy(np.ascontiguousarray(wl_mod.derivative_1d(L).T)).to(dev) for L in pb.shape]
            solver.gradient_densities(pb.shape, Dd[0], Dd[1], Dd[2], E, Zt, T=0.0, branch=branch)
            torch.cuda.synchronize()
            ts = []
            for _ in range(3):
                ev0.record(stream)
                solver.gradient_densities(pb.shape, Dd[0], Dd[1], Dd[2], E, Zt, T=0.0, branch=branch)
                ev1.record(stream)
                torch.cuda.synchronize()
                ts.append(ev0.elapsed_time(ev1))
            gms = sorted(ts)[len(ts) // 2]
            gflops = 2.0 * 4.0 * sum(pb.shape) * (N // 2) * active          # 4 L FMAs per point, state and axis
            gbytes = 3.0 * 16.0 * N * active
            epilogue["gradient"] = {"op": "eigh_gradient_densities (Eq. 16b, 16c; T = 0)", "ms": gms, "launches": 5,
                                    "algorithmic_flops": gflops, "algorithmic_bytes": gbytes, "bound": "tensor",
                                    "achieved_tflops": gflops / gms / 1e9 if gms else None, "peak_tflops": FP64_NOMINAL_TFLOPS,
                                    "frac": gflops / gms / 1e9 / FP64_NOMINAL_TFLOPS if gms else None,
                                    "achieved_gbs": gbytes / gms / 1e6 if gms else None,
                                    "hbm_frac": (gbytes / gms / 1e6) / hbm if hbm and gms else None}
            ts = []
            for _ in range(5):
                ev0.record(stream)
                regenerate()
                ev1.record(stream)
                torch.cuda.synchronize()
                ts.append(ev0.elapsed_time(ev1))
            ams = sorted(ts)[len(ts) // 2]
            epilogue["prologue"] = {"op": "eigh_assemble_bdg (Eq. 5/7/8: H from K, V, Delta; all N^2 elements written)",
                                    "ms": ams, "algorithmic_bytes": 16.0 * N * N, "bound": "hbm",
                                    "achieved_gbs": 16.0 * N * N / ams / 1e6 if ams else None, "peak_gbs": hbm,
                                    "frac": (16.0 * N * N / ams / 1e6) / hbm if hbm and ams else None, "launches": 1}
            # second workload: one TDSLDA step (eigh_tdslda_step) for a block of the states just computed.
            # Algorithmic bytes per step and state: 2 evaluations x 8 x 16 N (three kinetic passes) + 2 combines x 7 x 16 N
            # + 2 density passes x 16 N = 512 N bytes; HBM-bound.
            nst = min(nev, 2048)
            Kd = [torch.from_numpy(wl_mod.kinetic_1d(L)).to(dev) for L in pb.shape]
            Vd = torch.from_numpy(pb.V).to(dev)
            Yt = Zt[:nst].clone()
            E0 = E[:nst].contiguous()
            Dl0 = torch.from_numpy(np.ascontiguousarray(pb.Delta)).to(dev)
            Fl = [solver.tdslda_rhs(pb.shape, Kd[0], Kd[1], Kd[2], Vd, Dl0, pb.mu, Yt) for _ in range(5)]
            Ypt = torch.empty_like(Yt)
            n_t = torch.empty(N // 2, dtype=torch.float64, device=dev)
            D_t = torch.empty(N // 2, dtype=torch.complex128, device=dev)
            ts = []
            for it in range(4):
                ev0.record(stream)
                Fl = solver.tdslda_step(pb.shape, Kd[0], Kd[1], Kd[2], Vd, -1.0, pb.mu, E0, 1e-3, Yt, Fl, Ypt, n_t, D_t,
                                        branch=branch)
                ev1.record(stream)
                torch.cuda.synchronize()
                ts.append(ev0.elapsed_time(ev1))
            sms = sorted(ts[1:])[len(ts[1:]) // 2]
            sbytes = 512.0 * N * nst
            epilogue["tdslda_step"] = {"op": "eigh_tdslda_step (Eq. 5, Eq. 8, ABM PECE step; %d states)" % nst, "ms": sms,
                                       "launches": 20, "algorithmic_bytes": sbytes, "bound": "hbm",
                                       "achieved_gbs": sbytes / sms / 1e6 if sms else None, "peak_gbs": hbm,
                                       "frac": (sbytes / sms / 1e6) / hbm if hbm and sms else None,
                                       "minimal_bytes": 320.0 * N * nst,
                                       "frac_minimal": (320.0 * N * nst / sms / 1e6) / hbm if hbm and sms else None,
                                       "note": "algorithmic_bytes = the three-pass kinetic scheme as built (512 N per state and "
                                               "step); minimal_bytes = phi read once and f written once per evaluation (320 N)",
                                       "norm_drift": float((Yt.abs() ** 2).sum(dim=1).sub(1.0).abs().max().item())}
            del Yt, Fl, Ypt
        except Exception as ex:   # reported, never hidden
            epilogue = dict(epilogue or {}, error=str(ex)[:200])

    # ---- e2e: host buffers through eigh_solve_host, H2D of the full matrix and D2H of W and Z inside the timed region
    # (wall clock around the synchronous call, device idle on both sides).  Default: the host buffers are page-locked in
    # place (cudaHostRegister, exact size, outside the timed region) and copied directly in 256 MiB chunks; with
    # --host-buffers pageable (or when the registration fails) they stay pageable and are streamed through the handle's
    # bounded pinned ring (2 x 256 MiB).
    e2e = None
    if not args.no_e2e and rank == 0:
        try:
            regenerate()
            torch.cuda.synchronize()
            Ah = torch.empty((N, N), dtype=wdt)
            Ah.copy_(At)
            Wh = torch.empty(N, dtype=torch.float64)
            Zh = torch.empty((nev, N), dtype=wdt)
            rt = torch.cuda.cudart()
            registered = []
            if args.host_buffers == "pinned":
                for hb in (Ah, Zh, Wh):
                    if int(rt.cudaHostRegister(hb.data_ptr(), hb.numel() * hb.element_size(), 0)) != 0:
                        break
                    registered.append(hb)
                if len(registered) < 3:                 # all or nothing: report what the timed call really saw
                    for hb in registered:
                        rt.cudaHostUnregister(hb.data_ptr())
                    registered = []
            times = []
            for i in range(2 if N <= 8192 else 1):
                torch.cuda.synchronize()
                tt = time.perf_counter()
                solver.solve_host(Ah, Wh, Zh, At, W, Zt)
                torch.cuda.synchronize()
                times.append(time.perf_counter() - tt)
            e2e = {"value": min(times), "unit": "s", "h2d_bytes_per_step": mat_bytes,
                   "d2h_bytes_per_step": N * 8 + N * nev * (8 if args.real else 16),
                   "host_buffers": ("page-locked in place (cudaHostRegister), direct copies in 256 MiB chunks (eigh_solve_host)"
                                    if registered else
                                    "pageable, streamed through a 2 x 256 MiB pinned ring (eigh_solve_host)"),
                   "check_W_max_abs_diff": float((Wh - W.cpu()).abs().max().item())}
            for hb in registered:
                rt.cudaHostUnregister(hb.data_ptr())
            del Ah, Zh
        except Exception as ex:  # host allocation may fail for the largest configs
            e2e = {"value": None, "unit": "s", "error": str(ex)[:200]}

    # ---- cpu baseline: the oracle, as it stands, on a bounded sample (+ the measured, not extrapolated, small configs)
    cpu = None
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        import oracle
        Hs, what = oracle_sample(w, min(N, args.cpu_sample))
        ns = Hs.shape[0]
        tt = time.perf_counter()
        oracle.eigh(Hs)
        dt = time.perf_counter() - tt
        cpu = {"value": dt * (N / ns) ** 3, "unit": "s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{what}: {dt:.3f} s measured (all eigenpairs), scaled by (N/{ns})^3 (23 N^3 flops method)",
               "measured_s": dt, "measured_order": ns}
        try:   # config 0 measured as it is (not extrapolated)
            H0 = wl_mod.make_config(0).dense()
            tt = time.perf_counter()
            oracle.eigh(H0)
            cpu["measured_config0_N1024_s"] = time.perf_counter() - tt
        except Exception as ex:
            cpu["measured_config0_error"] = str(ex)[:100]

    # ---- context rows: library eigensolvers on the same seeded matrix; reported, never the target
    context = None
    if args.context and rank == 0 and world == 1:
        context = {}
        try:
            Wkeep = W.clone()
            del Zt
            torch.cuda.empty_cache()
            regenerate()
            torch.cuda.synchronize()
            ev0.record(stream)
            Wc, Zc = torch.linalg.eigh(At.t())
            ev1.record(stream)
            torch.cuda.synchronize()
            context["torch_linalg_eigh_s"] = ev0.elapsed_time(ev1) / 1e3
            context["torch_linalg_eigh_max_abs_diff_W"] = float((Wc - Wkeep).abs().max().item())
            del Wc, Zc
        except Exception as ex:
            context["torch_linalg_eigh_error"] = str(ex)[:200]
        try:
            Hs, _ = oracle_sample(w, min(N, args.cpu_sample))
            tt = time.perf_counter()
            np.linalg.eigh(Hs)
            context["numpy_linalg_eigh_sample"] = {"n": Hs.shape[0], "s": time.perf_counter() - tt}
        except Exception as ex:
            context["numpy_linalg_eigh_error"] = str(ex)[:200]

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    cw = credited_work(N, nev, b)
    ph = [sum(p[i] for p in phases) / len(phases) for i in range(6)]

    def tf(flops, ms):
        return flops / ms / 1e9 if ms else None

    s3_flops = float(sum(dc_flops))
    phase_report = {
        "p1_full_to_band": {"ms": ph[0], "tflops": tf(cw["p1_flops"], ph[0]),
                            "tflops_executed": tf(cw["p1_flops"] * EXECUTED_PER_CREDITED["p1"], ph[0])},
        "p2_band_to_tridiag": {"ms": ph[1], "gbs_credited": cw["p2_bytes"] / ph[1] / 1e6 if ph[1] else None,
                               "tflops": tf(cw["p2_flops"], ph[1]), "chase_steps": cw["p2_steps"],
                               "us_per_step_per_cta": ph[1] * 1e3 / (cw["p2_steps"] / 148.0) if ph[1] else None},
        "p3_tridiag_dc": {"ms": ph[2], "merge_flops_executed": s3_flops, "tflops_executed": tf(s3_flops, ph[2]),
                          "frac_of_fp64_peak": tf(s3_flops, ph[2]) / FP64_NOMINAL_TFLOPS if ph[2] else None,
                          "kept_frac_per_level": dc_kept, "deflated_frac_per_level": [1.0 - k for k in dc_kept],
                          "merge_flops_per_level": dc_flops,
                          "note": "executed = sum over the merge GEMMs of 2 M N K as launched (real DMMA flops); the "
                                  "phase time also holds the secular / deflation kernels (ALU)"},
        "p4a_backtransform_band": {"ms": ph[3], "tflops": tf(cw["p4a_flops"], ph[3]),
                                   "tflops_executed": tf(cw["p4a_flops"] * EXECUTED_PER_CREDITED["p4a"], ph[3])},
        "p4b_backtransform_full": {"ms": ph[4], "tflops": tf(cw["p4b_flops"], ph[4]),
                                   "tflops_executed": tf(cw["p4b_flops"] * EXECUTED_PER_CREDITED["p4b"], ph[4])},
    }
    # roofline object: the dominant kernel = the one with the largest device time per step.  S4a is ONE persistent launch
    # (bt_sweep_kernel) timed by CUDA events inside the library on the solve's stream; the GEMM families of S1 / S4b are
    # spread over hundreds of launches per phase and each family stays below its phase total (see the launch list in
    # profiles/).  Algorithmic work of the launch = the credited 8 N^2 nev flops of the band back-transformation
    # (WY padding and the T products excluded).
    dominant = max(range(5), key=lambda i: ph[i])
    sweep_ms = ph[5]
    achieved = cw["p4a_flops"] / sweep_ms / 1e9 if sweep_ms else 0.0
    traffic, traffic_note = lookup_traffic(w.name, nev)
    roofline = {
        "bound": "tensor", "kernel": "eigh::bt_sweep_kernel<%d> (FP64 DMMA, 1 launch per solve, all of phase p4a)" % solver.get_option("wy_group"),
        "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP64_NOMINAL_TFLOPS,
        "frac_executed": achieved * EXECUTED_PER_CREDITED["p4a"] / FP64_NOMINAL_TFLOPS,
        "traffic": traffic, "traffic_unit": "bytes per launch (dram read + write, ncu)", "traffic_source": traffic_note,
        "algorithmic_flops_per_launch": cw["p4a_flops"], "kernel_ms": sweep_ms, "launches_per_step": 1,
        "kernel_share_of_step": sweep_ms / ms_per_step if ms_per_step else None,
        "dominant_phase": PHASES[dominant],
        "dominant_kernel_rule": "largest device time of a single kernel family per step: bt_sweep_kernel = all of p4a in one "
                                "launch; the GEMM families of p1 / p4b (HEMM-lower, HER2K-lower, NN, CN instances of zgemm_kernel) "
                                "stay at 12-17 % each (profiles/r02_launches_c4.md)",
        "peak_source": "FP64 tensor (DMMA) 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2 TFLOP/s, equal to the burst DMMA rate "
                       "measured on this pool (profiles/r01_fp64_peaks.md; cuBLAS ZGEMM 36.8); MEASURED_PEAKS.json has "
                       "no FP64 entry.  `frac` divides CREDITED flops (8 per complex multiply-add) by it; `frac_executed` "
                       "the real flops the kernel issues (3-product forms)",
        "tensor_phase_fracs": {"p1": tf(cw["p1_flops"], ph[0]) / FP64_NOMINAL_TFLOPS if ph[0] else None,
                               "p4a": tf(cw["p4a_flops"], ph[3]) / FP64_NOMINAL_TFLOPS if ph[3] else None,
                               "p4b": tf(cw["p4b_flops"], ph[4]) / FP64_NOMINAL_TFLOPS if ph[4] else None},
        "tensor_phase_fracs_executed": {k: (tf(cw[k + "_flops"], ph[i]) * EXECUTED_PER_CREDITED[k] / FP64_NOMINAL_TFLOPS if ph[i] else None)
                                        for k, i in (("p1", 0), ("p4a", 3), ("p4b", 4))},
        "hbm_peak_gbs": hbm,
        "p2_hbm_frac_credited": (cw["p2_bytes"] / ph[1] / 1e6) / hbm if ph[1] and hbm else None,
    }
    cfg = config_dict(w, nev_total, nev_rule, b)
    if sharded:
        cfg["parallelism"] = "column-sharded back-transformations over %d ranks (rank 0: %d of %d columns)" % (world, nev, nev_total)
    if args.method == 1:
        # 1-stage variant.  Dominant kernel = hetrd_panel_kernel (one cooperative launch per 64-column
        # panel, all inside phase 0 together with the HER2K / SYR2K GEMMs): HBM-bound, algorithmic bytes = the lower
        # triangle of the trailing matrix read once per column, sum_c es (N-1-c)(N-c)/2  (~ es N^3 / 6; es = 16 or 8).
        es = 8 if args.real else 16
        tri_bytes = float(sum(es * (N - 1 - c) * (N - c) // 2 for c in range(N - 1)))
        npanels = -(-(N - 1) // 64)
        bt_flops = (2.0 if args.real else 8.0) * N * N * nev
        upd_flops = (2.0 if args.real else 8.0) * N ** 3 / 3.0          # rank-2k updates (HER2K-lower)
        phase_report = {
            "p1_tridiagonalise_direct": {"ms": ph[0], "gbs_lower_triangle": tri_bytes / ph[0] / 1e6 if ph[0] else None,
                                         "her2k_flops": upd_flops, "panels": npanels},
            "p3_tridiag_dc": phase_report["p3_tridiag_dc"],
            "p4_backtransform_direct": {"ms": ph[4], "tflops": tf(bt_flops, ph[4])},
        }
        ach = tri_bytes / ph[0] / 1e6 if ph[0] else 0.0
        roofline = {
            "bound": "hbm", "kernel": "eigh::hetrd_panel_kernel<%s> (%d cooperative launches per solve, phase p1; the phase "
                                      "time also holds the %d rank-2k GEMM updates)" % ("double" if args.real else "c128", npanels, npanels),
            "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm if hbm else None, "traffic": None,
            "traffic_source": "no ncu capture", "algorithmic_bytes_per_step": tri_bytes,
            "algorithmic_bytes_per_launch": tri_bytes / npanels, "kernel_ms": ph[0] / npanels, "launches_per_step": npanels,
            "kernel_share_of_step": ph[0] / ms_per_step if ms_per_step else None,
            "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured); for N below ~4000 the lower triangle fits the 126 MB L2",
        }
        cfg["method"] = "one-stage (PAPER.md:148 steps i-iii)"
        cfg["dtype"] = "f64 real symmetric" if args.real else "c128"
    line = {
        "metric": "eigh_time_s", "value": value_s, "unit": "s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False,
        "scaling": "strong" if sharded else "weak",
        "vs_baseline": None, "dtype": "f64" if args.real else "c128", "data": "synthetic",
        "config": cfg,
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "phases": phase_report, "roofline": roofline,
        "cpu_baseline": cpu, "validity": valid, "epilogue": epilogue, "context": context,
        "total_tflops": (cw["p1_flops"] + cw["p2_flops"] + cw["p4a_flops"] + cw["p4b_flops"]) / ms_per_step / 1e9
        if args.method == 2 else None,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
