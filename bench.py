#!/usr/bin/env python
"""bench.py -- time-to-solution of the dense complex-FP64 Hermitian eigensolve on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--nev NEV] [--impl reference]

A "step" is one pass of the whole hot path (eigh_solve: full->band, band->tridiagonal, tridiagonal
D&C, both back-transformations) over one synthetic matrix of BASELINE.json's `configs` (default
config 3, the N = 27648 vortex-tangle BdG matrix: the largest one whose W + K solves finish within
minutes; --config 4 runs the N = 49152 target, --config 2 the N = 8192 case).  The matrix is regenerated in place
(device-side copy from a resident pristine copy, or the device generator when two copies do not
fit) OUTSIDE the per-step CUDA-event brackets, because eigh_solve overwrites A.

One JSON line on stdout (rank 0):  metric = eigh_time_s (seconds per eigensolve, lower is better),
plus `phases` (ms, credited TFLOP/s or GB/s per phase), `roofline` (dominant phase against the FP64
tensor peak), `e2e` (host buffers through eigh_solve_host), `cpu_baseline` (the oracle on a
bounded sample) and `clocks`.

Multi-GPU: the path does not shard ("replicas only"): every rank solves its own replica,
value = max-over-ranks time / n_gpus.
"""
from __future__ import annotations

import argparse
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


def credited_work(N: int, nev: int, b: int):
    """Credited algorithmic work per phase (lower-order terms dropped)."""
    steps = 0
    bytes_p2 = 0
    for j in range(0, N - 1):
        ks = -(-(N - 1 - j) // b)
        steps += ks
    # per chase step: D lower (b^2/2) + S (b^2) read and written, 16 B each; reflector b written
    bytes_p2 = steps * (2 * (b * b // 2 + b * b) * 16 + b * 16)
    return {
        "p1_flops": 16.0 / 3.0 * N ** 3,
        "p2_flops": 24.0 * b * N * N,
        "p2_bytes": float(bytes_p2),
        "p3_flops_max": 8.0 / 3.0 * N ** 3,       # dense merges without deflation (as executed: no block structure)
        "p4a_flops": 8.0 * N * N * nev,
        "p4b_flops": 8.0 * N * N * nev,
    }


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


def reference_arm(args, wl_mod):
    """--impl reference: the CPU oracle (unmodified, as it stands) on a bounded sample of the workload:
    the leading principal n_s x n_s submatrix, timed per step and scaled by (N/n_s)^3 (the oracle is a
    23 N^3 level-1/2 method)."""
    import numpy as np
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = wl_mod.make_config(args.config)
    N = w.N
    ns = min(N, args.ref_sample)
    if w.problem is not None:
        H = _leading_block_bdg(w, ns)
    else:
        H = w.dense()[:ns, :ns]
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.eigh(H)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
    per = sum(times) / len(times)
    ns = H.shape[0]                       # the BdG sub-lattice sample may be smaller than requested
    est = per * (N / ns) ** 3
    line = {
        "impl": "reference", "metric": "eigh_time_s", "value": est, "unit": "s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": est * 1e3, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "nev": N},
        "cpu_baseline": {"value": est, "unit": "s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": f"{ns}x{ns} sample (leading block, or the same recipe on a sub-lattice) solved in {per:.3f} s "
                                   f"per step, scaled by (N/{ns})^3"},
        "e2e": {"value": est, "unit": "s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def _leading_block_bdg(w, ns):
    """Leading ns x ns block of a BdG config without materialising the full matrix: solve the same
    generator on a smaller lattice slab is NOT the same matrix, so take the block of the dense matrix
    when it is affordable, else a sub-lattice of the same recipe (stated in `sample`)."""
    import numpy as np
    if w.N <= 8192:
        return np.ascontiguousarray(w.dense()[:ns, :ns])
    from paper_2310_03341_b200 import workloads as wl
    # same recipe (fields, mu) restricted to a sub-lattice with 2*nx*ny*nz ~ ns
    p = w.problem
    nx, ny, nz = p.shape
    while 2 * nx * ny * nz > ns:
        if nx >= ny and nx >= nz: nx //= 2
        elif ny >= nz: ny //= 2
        else: nz //= 2
    idx = np.arange(np.prod(p.shape)).reshape(p.shape)[:nx, :ny, :nz].reshape(-1)
    q = wl.BdGProblem(p.name, (nx, ny, nz), p.mu, p.V[idx], p.Delta[idx])
    return q.dense()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=int(os.environ.get("EIGH_BENCH_CONFIG", "3")))
    ap.add_argument("--nev", type=int, default=0, help="0 = all eigenpairs")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--ref-sample", type=int, default=3456, help="order of the oracle sample of --impl reference")
    ap.add_argument("--cpu-sample", type=int, default=3456,
                    help="order of the oracle's sample (about 10-30 s of CPU work on the box's host cores)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--context", action="store_true",
                    help="also time library routines on the same matrix as CONTEXT (never the target, never on the hot path): "
                         "torch.linalg.eigh (cuSOLVER) on this GPU and numpy.linalg.eigh (LAPACK) on the CPU sample")
    ap.add_argument("--wy-group", type=int, default=0)
    ap.add_argument("--opt", action="append", default=[], help="solver option key=value (eigh_set_option), repeatable")
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
    nev = args.nev if args.nev > 0 else N
    opts = {}
    if args.wy_group:
        opts["wy_group"] = args.wy_group
    for kv in args.opt:
        key, val = kv.split("=")
        opts[key] = int(val)
    solver = binding.Eigh(N, nev, device=dev, **opts)
    b = 64
    mat_bytes = N * N * 16
    free_b, total_b = torch.cuda.mem_get_info()
    keep_pristine = free_b > 3 * mat_bytes + (2 << 30)
    At = torch.empty((N, N), dtype=torch.complex128, device=dev)       # A column-major (stored as A^T row-major)
    W = torch.empty(N, dtype=torch.float64, device=dev)
    Zt = torch.empty((nev, N), dtype=torch.complex128, device=dev)
    pristine = None
    if keep_pristine:
        pristine = torch.empty((N, N), dtype=torch.complex128, device=dev)
        w.dense_torch(dev, out=pristine)

    def regenerate():
        if pristine is not None:
            At.copy_(pristine)
        else:
            w.dense_torch(dev, out=At)

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

    # ---- quick validity check of the last solve (device side, independent ZGEMM by torch)
    valid = {}
    if rank == 0:
        with torch.no_grad():
            Hd = pristine if pristine is not None else w.dense_torch(dev, out=At)
            Hl = Hd.t() if pristine is not None else Hd
            ncheck = min(nev, 256)
            cols = torch.linspace(0, nev - 1, ncheck, device=dev).long()
            Zc = Zt[cols].t()                                   # N x ncheck
            R = Hl @ Zc - Zc * W[cols][None, :]
            hn = float(torch.linalg.norm(Hl).item())
            valid["residual_sampled"] = float(torch.linalg.norm(R).item()) / (hn * (ncheck ** 0.5))
            valid["orth_sampled"] = float((Zc.conj().t() @ Zc - torch.eye(ncheck, device=dev)).abs().max().item())
            valid["trace_err"] = abs(float(W.sum().item()) - float(torch.diagonal(Hl).real.sum().item()))

    # ---- SCF epilogue (outside the timed step): eigh_densities on the eigenpairs just computed,
    # Eq. 16a/16d at T = 0.  HBM-bound: algorithmic bytes = the u and v halves of every ACTIVE column of Z read once
    # (16 N bytes per column with 0 < E < Ec) + the two output fields; CUDA events on the launching stream.
    epilogue = None
    if rank == 0 and w.problem is not None and N % 2 == 0:
        try:
            n_f, nu_f = solver.densities(W, Zt, T=0.0)
            torch.cuda.synchronize()
            ts = []
            for _ in range(5):
                ev0.record(stream)
                solver.densities(W, Zt, T=0.0, n=n_f, nu=nu_f)
                ev1.record(stream)
                torch.cuda.synchronize()
                ts.append(ev0.elapsed_time(ev1))
            active = int(((W[:nev] > 0)).sum().item())
            dbytes = 16.0 * N * active + 24.0 * (N // 2)
            dms = sorted(ts)[len(ts) // 2]
            hbm = None
            try:
                hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs")
            except Exception:
                pass
            epilogue = {"op": "eigh_densities (Eq. 16a, 16d; T = 0; all columns with E > 0)", "ms": dms,
                        "active_columns": active, "algorithmic_bytes": dbytes, "bound": "hbm",
                        "achieved_gbs": dbytes / dms / 1e6 if dms else None, "peak_gbs": hbm,
                        "frac": (dbytes / dms / 1e6) / hbm if hbm and dms else None, "launches": 3,
                        "particle_number": float(n_f.sum().item()),
                        "note": "inputs (%.1f GB of active columns) larger than L2" % (16.0 * N * active / 1e9)}
            # Eq. 16b/16c: eigh_gradient_densities (three launches, one per axis; FP64 tensor cores + HBM: 4 L FMAs and 32
            # bytes per grid point, state and axis -- at L = 24..32 the two rooflines nearly coincide, both are reported)
            pb = w.problem
            Dd = [torch.from_numpy(np.ascontiguousarray(wl_mod.derivative_1d(L).T)).to(dev) for L in pb.shape]
            solver.gradient_densities(pb.shape, Dd[0], Dd[1], Dd[2], W, Zt, T=0.0)
            torch.cuda.synchronize()
            ts = []
            for _ in range(3):
                ev0.record(stream)
                solver.gradient_densities(pb.shape, Dd[0], Dd[1], Dd[2], W, Zt, T=0.0)
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
            # prologue: eigh_assemble_bdg writes all N^2 elements of H from (K, V, Delta): HBM-write-bound, 16 N^2 bytes
            Kd = [torch.from_numpy(wl_mod.kinetic_1d(L)).to(dev) for L in pb.shape]
            Vd = torch.from_numpy(pb.V).to(dev)
            Dd = torch.from_numpy(np.ascontiguousarray(pb.Delta)).to(dev)
            solver.assemble_bdg(pb.shape, Kd[0], Kd[1], Kd[2], Vd, Dd, pb.mu, At=At)
            torch.cuda.synchronize()
            ts = []
            for _ in range(5):
                ev0.record(stream)
                solver.assemble_bdg(pb.shape, Kd[0], Kd[1], Kd[2], Vd, Dd, pb.mu, At=At)
                ev1.record(stream)
                torch.cuda.synchronize()
                ts.append(ev0.elapsed_time(ev1))
            ams = sorted(ts)[len(ts) // 2]
            epilogue["prologue"] = {"op": "eigh_assemble_bdg (Eq. 5/7/8: H from K, V, Delta; all N^2 elements written)",
                                    "ms": ams, "algorithmic_bytes": 16.0 * N * N, "bound": "hbm",
                                    "achieved_gbs": 16.0 * N * N / ams / 1e6 if ams else None, "peak_gbs": hbm,
                                    "frac": (16.0 * N * N / ams / 1e6) / hbm if hbm and ams else None, "launches": 1}
        except Exception as ex:   # reported, never hidden
            epilogue = {"error": str(ex)[:200]}

    # ---- e2e: host buffers through eigh_solve_host (H2D of A, D2H of W and Z inside the timed region)
    e2e = None
    if not args.no_e2e and rank == 0:
        try:
            src = pristine if pristine is not None else w.dense_torch(dev, out=At)
            Ah = torch.empty((N, N), dtype=torch.complex128, pin_memory=True)
            Ah.copy_(src if pristine is not None else At)
            Wh = torch.empty(N, dtype=torch.float64, pin_memory=True)
            Zh = torch.empty((nev, N), dtype=torch.complex128, pin_memory=True)
            times = []
            for i in range(2 if N <= 8192 else 1):
                torch.cuda.synchronize()
                ev0.record(stream)
                solver.solve_host(Ah, Wh, Zh, At, W, Zt)
                ev1.record(stream)
                torch.cuda.synchronize()
                times.append(ev0.elapsed_time(ev1))
            e2e = {"value": min(times) / 1e3, "unit": "s", "h2d_bytes_per_step": mat_bytes,
                   "d2h_bytes_per_step": N * 8 + N * nev * 16}
            del Ah, Zh
        except Exception as ex:  # pinned allocation may fail for the largest configs
            e2e = {"value": None, "unit": "s", "error": str(ex)[:200]}

    # ---- cpu baseline: the oracle, as it stands, on a bounded sample
    cpu = None
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        import oracle
        ns = min(N, args.cpu_sample)
        Hs = _leading_block_bdg(w, ns) if w.problem is not None else w.dense()[:ns, :ns]
        ns = Hs.shape[0]                  # the BdG sub-lattice sample may be smaller than requested
        tt = time.perf_counter()
        oracle.eigh(Hs)
        dt = time.perf_counter() - tt
        cpu = {"value": dt * (N / ns) ** 3, "unit": "s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{ns}x{ns} sample (leading block of the matrix, or for N > 8192 the same recipe on a sub-lattice): "
                         f"{dt:.3f} s measured, scaled by (N/{ns})^3 (23 N^3 flops method)"}

    # ---- context rows: library eigensolvers on the same seeded matrix; reported, never the target
    context = None
    if args.context and rank == 0 and world == 1:
        context = {}
        try:
            del Zt
            torch.cuda.empty_cache()
            Hc = w.dense_torch(dev, out=At)                   # logical H (column-major storage in At)
            torch.cuda.synchronize()
            ev0.record(stream)
            Wc, Zc = torch.linalg.eigh(Hc)
            ev1.record(stream)
            torch.cuda.synchronize()
            context["torch_linalg_eigh_s"] = ev0.elapsed_time(ev1) / 1e3
            context["torch_linalg_eigh_max_abs_diff_W"] = float((Wc - W).abs().max().item())
            del Wc, Zc
        except Exception as ex:
            context["torch_linalg_eigh_error"] = str(ex)[:200]
        try:
            ns = min(N, args.cpu_sample)
            Hs = _leading_block_bdg(w, ns) if w.problem is not None else w.dense()[:ns, :ns]
            tt = time.perf_counter()
            np.linalg.eigh(Hs)
            context["numpy_linalg_eigh_sample"] = {"n": ns, "s": time.perf_counter() - tt}
        except Exception as ex:
            context["numpy_linalg_eigh_error"] = str(ex)[:200]

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    cw = credited_work(N, nev, b)
    ph = [sum(p[i] for p in phases) / len(phases) for i in range(6)]
    phase_report = {
        "p1_full_to_band": {"ms": ph[0], "tflops": cw["p1_flops"] / ph[0] / 1e9 if ph[0] else None},
        "p2_band_to_tridiag": {"ms": ph[1], "gbs_credited": cw["p2_bytes"] / ph[1] / 1e6 if ph[1] else None,
                               "tflops": cw["p2_flops"] / ph[1] / 1e9 if ph[1] else None},
        "p3_tridiag_dc": {"ms": ph[2], "tflops_if_no_deflation": cw["p3_flops_max"] / ph[2] / 1e9 if ph[2] else None},
        "p4a_backtransform_band": {"ms": ph[3], "tflops": cw["p4a_flops"] / ph[3] / 1e9 if ph[3] else None},
        "p4b_backtransform_full": {"ms": ph[4], "tflops": cw["p4b_flops"] / ph[4] / 1e9 if ph[4] else None},
    }
    # roofline object: the dominant kernel.  S4a is one persistent launch (bt_sweep_kernel) whose duration is
    # measured by CUDA events inside the library on the solve's stream; its algorithmic work is the credited
    # 8 N^2 nev flops of the band back-transformation (WY padding and the T products excluded).
    dominant = max(range(5), key=lambda i: ph[i])
    sweep_ms = ph[5]
    achieved = cw["p4a_flops"] / sweep_ms / 1e9 if sweep_ms else 0.0
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    # DRAM bytes (read + write) of one bt_sweep_kernel launch from the committed ncu capture of this workload
    # (profiles/r01_bt_sweep_c3_traffic.csv, command in profiles/r01_ncu_kernels.md); null for other workloads
    traffic = None
    if w.index == 3 and nev == N:
        try:
            import csv
            tot = 0.0
            with open(os.path.join(ROOT, "profiles", "r01_bt_sweep_c3_traffic.csv")) as f:
                for row in csv.reader(l for l in f if not l.startswith("==")):
                    if len(row) > 3 and row[-3] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                        tot += float(row[-1].replace(",", ""))
            traffic = tot if tot > 0 else None
        except Exception:
            traffic = None
    roofline = {
        "bound": "tensor", "kernel": "eigh::bt_sweep_kernel<8> (FP64 DMMA, 1 launch per solve, phase p4a)",
        "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP64_NOMINAL_TFLOPS,
        "traffic": traffic, "traffic_unit": "bytes per launch (dram read + write, ncu)",
        "algorithmic_flops_per_launch": cw["p4a_flops"], "kernel_ms": sweep_ms, "launches_per_step": 1,
        "dominant_phase": ["p1_full_to_band", "p2_band_to_tridiag", "p3_tridiag_dc", "p4a_backtransform_band",
                           "p4b_backtransform_full"][dominant],
        "peak_source": "FP64 tensor (DMMA) 148 SM x 64 FMA/clk x 1.965 GHz = 37.2 TFLOP/s, equal to the burst DMMA rate "
                       "measured on this pool (profiles/r01_fp64_peaks.md; cuBLAS ZGEMM 36.8); MEASURED_PEAKS.json has "
                       "no FP64 entry",
        "tensor_phase_fracs": {"p1": cw["p1_flops"] / ph[0] / 1e9 / FP64_NOMINAL_TFLOPS if ph[0] else None,
                               "p4a": cw["p4a_flops"] / ph[3] / 1e9 / FP64_NOMINAL_TFLOPS if ph[3] else None,
                               "p4b": cw["p4b_flops"] / ph[4] / 1e9 / FP64_NOMINAL_TFLOPS if ph[4] else None},
        "hbm_peak_gbs": peaks.get("hbm_gbs"),
        "p2_hbm_frac_credited": (cw["p2_bytes"] / ph[1] / 1e6) / peaks["hbm_gbs"] if ph[1] and peaks.get("hbm_gbs") else None,
    }
    line = {
        "metric": "eigh_time_s", "value": value_s, "unit": "s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "c128", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "nev": nev, "band_width": b, "parallelism": "replicas only",
                   "l2": "inputs larger than L2 (matrix %.1f GB)" % (mat_bytes / 1e9),
                   "input_regeneration": "device copy outside the timed brackets"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "phases": phase_report, "roofline": roofline,
        "cpu_baseline": cpu, "validity": valid, "epilogue": epilogue, "context": context,
        "total_tflops": (cw["p1_flops"] + cw["p2_flops"] + cw["p4a_flops"] + cw["p4b_flops"]) / ms_per_step / 1e9,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
