#!/usr/bin/env python
"""Benchmark of the Chebyshev-filter hot path (BASELINE.json metric) on B200.

A "step" is one `chfsi_cheb_filter` call -- residual S0, m-1 recurrence steps, recover S7, i.e. every row of
SURVEY.md 8(a) -- over one block of synthetic vectors.  Default workload: BASELINE.json configs[3], the largest
single-GPU configuration: 12x12x12 periodic cells, side 32 Bohr, p = 8 (96^3 nodes, 1.77M complex DoF), Bloch k-point
(0.25,0,0) 2 pi/L, 216 atoms x 8 projectors, 1024 complex128 vectors processed in chunks of 256, Chebyshev degree 30,
FP64 throughout (the paper's reference arithmetic), the residual-based recurrence (eq. 11).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--prec fp64|fp32|fp32s]

The JSON line also carries `all_configs`: one compact row per BASELINE config / precision (c0 latency; c1, c2, c3, the c4
sweep: cell-kernel ms, its roofline fraction, whole-call fraction), measured in the same run (`--no-table` skips it).
N > 1 (under torchrun): the filter shards over columns with no exchange (the paper's band partitioning in its n_r = 1
limit): every rank filters its own block of the same mesh, value = all ranks' units / max-over-ranks
time, scaling "weak".  `--impl reference` times the CPU oracle (oracle/fe_oracle.py, as it stands) on a bounded sample.
Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2605_30128_b200 import inputs as inp  # noqa: E402

METRIC = "chebyshev_filter_throughput"
UNIT = "complex_DoF*vectors*degree/s"
FALLBACK_HBM_GBS = 6650.0        # /opt/skills/guides/B200_PROFILING.md fallback
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_cell_kernel_traffic.csv")
DTYPE = {"fp64": "f64", "fp64m": "f64 (cell contractions on mma.sync.m8n8k4.f64)",
         "fp32": "f32 product / f64 storage and recurrence",
         "fp32s": "f32 multivectors / f64 residual and Lambda_k",
         "tf32": "f32 multivectors, tf32 tensor-core cell contractions / f64 residual and Lambda_k",
         "tf32x3": "f32 multivectors, 3xtf32 tensor-core cell contractions / f64 residual and Lambda_k"}


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(config, prec, nvec_launch):
    """dram__bytes_read.sum + dram__bytes_write.sum per cell-kernel launch from the committed `ncu --set full` captures
    (profiles/r2_cell_kernel_traffic.csv, written from the .ncu-rep files by the command in the .md beside it), keyed by
    (config, precision, vectors per launch); None where no capture exists."""
    try:
        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(f):
                if int(row["config"]) == config and row["prec"] == prec and int(row["nvec_per_launch"]) == nvec_launch:
                    return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nm, val in zip(names, r[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def aggregate_over_ranks(ms_local, units_per_rank, world, dist=None, device="cpu"):
    """N > 1: every rank filtered its own block of `units_per_rank` units in `ms_local` ms; no data-path collective -- the
    only cross-rank step is this MAX of the device-timed durations.  Returns (max ms over ranks, whole-job units per second)."""
    ms = float(ms_local)
    if dist is not None and world > 1:
        import torch
        t = torch.tensor([ms], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms, world * units_per_rank / (ms * 1e-3)


def units_per_step(cfg, nvec):
    return 2.0 * cfg.nnodes * nvec * cfg.degree


def alg_bytes_per_unit(prec, recur="residual"):
    """Algorithmic HBM bytes per unit of a recurrence step: eq. 11 reads Z_k and R and
    read-modify-writes Z_{k-1} -> Z_{k+1}.  complex128: 16 + 16 + 32 = 64 B; complex64 iterates with R in FP64
    ("only R and Lambda_k in FP64"): 8 + 16 + 16 = 40 B.  eq. 10: no R, 48 B."""
    if recur != "residual":
        return 48.0
    return 40.0 if prec in ("fp32s", "tf32", "tf32x3") else 64.0


# --------------------------------------------------------------------------------------------
def cpu_oracle_rate(cfg, ncols, repeat=1):
    """Oracle (eq. 11, FP64, as it stands) on `ncols` sampled columns of the workload; units/s."""
    from oracle import fe_oracle as fo
    mesh = fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    ham = fo.Hamiltonian(mesh, hi.V, hi.Bx, hi.By, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj, hi.P, hi.D)
    X = inp.make_vectors(cfg.nnodes, list(range(ncols)))
    lam = np.zeros(ncols)
    b = 1.5 * (np.pi * cfg.p * cfg.ncell / cfg.L) ** 2 + 50.0    # crude, safe upper bound; timing only
    a0, a = -3.0, 5.0
    best, cpu_used = None, 1.0
    for _ in range(repeat):
        t0, c0 = time.perf_counter(), time.process_time()
        fo.cheb_filter_residual(ham, X, lam, cfg.degree, a, b, a0)
        dt, dc = time.perf_counter() - t0, time.process_time() - c0
        if best is None or dt < best:
            best, cpu_used = dt, dc / dt
    return units_per_step(cfg, ncols) / best, best, max(1, int(round(cpu_used)))


def _oracle_worker(cfg, cols, barrier, q):
    """One host process of the all-cores CPU baseline: the oracle, as it stands, on its own columns (columns are independent)."""
    os.environ["OMP_NUM_THREADS"] = os.environ["OPENBLAS_NUM_THREADS"] = os.environ["MKL_NUM_THREADS"] = "1"
    from oracle import fe_oracle as fo
    mesh = fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    ham = fo.Hamiltonian(mesh, hi.V, hi.Bx, hi.By, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj, hi.P, hi.D)
    X = inp.make_vectors(cfg.nnodes, cols)
    b = 1.5 * (np.pi * cfg.p * cfg.ncell / cfg.L) ** 2 + 50.0
    barrier.wait()                                   # every process has built its operator: the timed region starts
    t0 = time.perf_counter()
    fo.cheb_filter_residual(ham, X, np.zeros(len(cols)), cfg.degree, 5.0, b, -3.0)
    q.put(time.perf_counter() - t0)


def cpu_oracle_rate_all_cores(cfg, cols_per_proc=1, nproc=None):
    """The same oracle on every host core at once: one process per core (spawned: no CUDA state is inherited), each filtering
    its own `cols_per_proc` columns; rate = all columns' units / the slowest process's time."""
    import multiprocessing as mp
    nproc = nproc or os.cpu_count() or 1
    ctx = mp.get_context("spawn")
    barrier, q = ctx.Barrier(nproc), ctx.Queue()
    procs = [ctx.Process(target=_oracle_worker, args=(cfg, list(range(i * cols_per_proc, (i + 1) * cols_per_proc)), barrier, q))
             for i in range(nproc)]
    for pr in procs:
        pr.start()
    times = []
    deadline = time.time() + 1800
    while len(times) < nproc:
        try:
            times.append(q.get(timeout=2))
        except Exception:
            dead = [pr for pr in procs if pr.exitcode not in (None, 0)]
            if dead or time.time() > deadline:                       # a worker died (or hung): do not wait for it
                for pr in procs:
                    if pr.is_alive():
                        pr.terminate()
                raise RuntimeError("cpu baseline: an oracle worker process failed")
    for pr in procs:
        pr.join()
    dt = max(times)
    return units_per_step(cfg, nproc * cols_per_proc) / dt, dt, nproc


def workload_name(args, cfg, nvec, chunk):
    return (f"BASELINE configs[{args.config}] ({cfg.name}): {cfg.ncell}^3 cells, side {cfg.L} Bohr, p={cfg.p}, "
            f"{2 * cfg.nnodes} complex DoF, kfrac {tuple(cfg.kfrac)}, {nvec} complex128 vectors in chunks of {chunk or nvec}, "
            f"{cfg.natoms} atoms x {cfg.nproj} projectors, degree {cfg.degree}, recurrence {args.recur}, prec {args.prec}")


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    ncols = max(1, args.ref_cols // 2)      # each of the K + W steps is a bounded sample: the run ends within minutes
    times, cores = [], 1
    for i in range(args.warmup + args.steps):
        rate, dt, cores = cpu_oracle_rate(cfg, ncols)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = units_per_step(cfg, ncols) / (ms * 1e-3)
    sample = f"{ncols} of {cfg.nvec} columns of {cfg.name}, full degree {cfg.degree}, eq. 11 FP64 (columns are independent)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args, cfg, cfg.nvec, cfg.chunk), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle (numpy, single process)", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------
class Workload:
    """One mesh + Hamiltonian + device block, with the timing helpers used for the headline and for the table."""

    def __init__(self, torch, B, cfg, prec_name, recur_name, nvec, device, seed, pb=None):
        from paper_2605_30128_b200.harness import GpuProblem
        self.torch, self.B, self.cfg = torch, B, cfg
        self.prec = B.PREC["fp64" if prec_name == "fp64m" else prec_name]
        self.mma64 = prec_name == "fp64m"        # FP64 on the tensor-core cell kernel (chfsi_mesh_set_cell_kernel)
        self.recur = B.RECUR_RESIDUAL if recur_name == "residual" else B.RECUR_STANDARD
        self.nvec = nvec
        self.chunk = cfg.chunk if (cfg.chunk and cfg.chunk < nvec) else (256 if nvec > 512 else 0)
        self.own_pb = pb is None
        self.pb = pb if pb is not None else GpuProblem(cfg, seed=0, device=device)
        dev = f"cuda:{device}"
        g = torch.Generator(device=dev); g.manual_seed(seed)
        self.X = torch.empty((cfg.nnodes, 2, nvec), dtype=torch.complex128, device=dev)
        Xr = torch.view_as_real(self.X)
        for j0 in range(0, nvec, 64):                      # filled in slabs: no full-size temporaries
            j1 = min(nvec, j0 + 64)
            Xr[:, :, j0:j1, :] = torch.rand((cfg.nnodes, 2, j1 - j0, 2), generator=g, device=dev, dtype=torch.float64) * 2 - 1
        self.Y = torch.empty_like(self.X)
        self.a0, self.b = self.pb.lanczos_bounds(10)
        self.a = self.a0 + 0.1 * (self.b - self.a0)
        self.lam = self.pb.rayleigh_quotients(self.X) if self.recur == B.RECUR_RESIDUAL else None
        self.work = self.pb.work(self.prec, self.recur, self.chunk if self.chunk else nvec)
        self.stream = torch.cuda.current_stream()

    def step(self):
        if self.mma64 != getattr(self.pb, "_mma64", False):
            self.B.chfsi_mesh_set_cell_kernel(self.pb.mesh, self.B.FP64, self.B.CELL_MMA if self.mma64 else self.B.CELL_DEFAULT)
            self.pb._mma64 = self.mma64
        self.B.chfsi_cheb_filter(self.pb.mesh, self.prec, self.recur, self.cfg.degree, self.a, self.b, self.a0, self.X,
                                 self.lam, self.Y, self.work, chunk=self.chunk, stream=self.stream)

    def time_steps(self, steps, warmup, barrier=None):
        torch = self.torch
        for _ in range(warmup):
            self.step()
        (barrier or torch.cuda.synchronize)()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        ev[0].record(self.stream)
        for i in range(steps):
            self.step()
            ev[i + 1].record(self.stream)
        (barrier or torch.cuda.synchronize)()
        per = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
        return ev[0].elapsed_time(ev[steps]), per

    def cell_profile(self, nsteps):
        """Cell-kernel launches of `nsteps` filter calls, timed with CUDA events on the launching stream by the library
        (the nonlocal kernels then run on the same stream instead of the forked side stream)."""
        B = self.B
        B.chfsi_profile_enable(self.pb.mesh, True)
        for _ in range(nsteps):
            self.step()
        cell_ms, cell_n, cell_bytes = B.chfsi_profile_read(self.pb.mesh)
        B.chfsi_profile_enable(self.pb.mesh, False)
        return cell_ms, cell_n, cell_bytes

    def close(self):
        self.X = self.Y = self.work = None
        self.pb._work = {}
        if self.own_pb:
            self.pb.close()
        self.torch.cuda.empty_cache()


def config_row(torch, B, cfg_id, prec, nvec, device, peak, steps=2, warmup=1, pb=None):
    """One row of the all-config table."""
    cfg = inp.CONFIGS[cfg_id]
    w = Workload(torch, B, cfg, prec, "residual", nvec, device, 4321, pb=pb)
    try:
        ms_total, _ = w.time_steps(steps, warmup)
        ms_step = ms_total / steps
        cell_ms, cell_n, cell_bytes = w.cell_profile(1)
        bpu = alg_bytes_per_unit(prec)
        ups = units_per_step(cfg, nvec) / (ms_step * 1e-3)
        return {"config": cfg_id, "prec": prec, "nvec": nvec, "chunk": w.chunk or nvec, "filter_ms": round(ms_step, 4),
                "units_per_s": float(f"{ups:.4g}"), "cell_ms": round(cell_ms / cell_n, 5),
                "cell_frac": round(cell_bytes / (cell_ms * 1e-3) / 1e9 / peak, 4),
                "whole_frac": round(ups * bpu / (peak * 1e9), 4), "alg_bytes_per_unit": bpu}
    finally:
        w.close()


def eigen_check(torch, B, device):
    """configs[4] asks for the converged eigenvalue error per precision: Algorithm 1 (harness: Rayleigh-Ritz in FP64, bounds from
    Lanczos) on configs[4]'s mesh and Hamiltonian with a 64-vector block, once per filter precision; reported: passes to a residual
    of 3e-6 on the lowest 32 states and the largest difference of those eigenvalues from the FP64-filter run (Ha)."""
    from paper_2605_30128_b200.harness import GpuProblem
    cfg = inp.CONFIGS[4]
    pb = GpuProblem(cfg, seed=0, device=device)
    out = {}
    try:
        _, b = pb.lanczos_bounds(10)
        X0 = torch.from_numpy(inp.make_vectors(cfg.nnodes, 64, seed=0)).to(f"cuda:{device}")
        ref = None
        for name in ("fp64", "fp32", "fp32s", "tf32x3", "tf32"):
            _, lam, hist = pb.subspace_iteration(X0, cfg.degree, b, 60, tol=3e-6, n_check=32, prec=B.PREC[name])
            if ref is None:
                ref = lam
            out[name] = {"passes": len(hist), "residual": float(f"{hist[-1]:.3g}"),
                         "max_abs_diff_vs_fp64_Ha": float(f"{np.max(np.abs(lam[:32] - ref[:32])):.3g}")}
    finally:
        pb.close()
        torch.cuda.empty_cache()
    return out


def all_configs_table(torch, B, device, peak):
    """c0 (latency, also through a CUDA graph), c1, c3 (one chunk) and the c4 sweep (c2 = its 512-vector rows) in every
    built precision."""
    from paper_2605_30128_b200.harness import GpuProblem
    rows = []
    # c0: launch / latency bound -- time only, plain launch and graph replay
    cfg0 = inp.CONFIGS[0]
    w = Workload(torch, B, cfg0, "fp64", "residual", cfg0.nvec, device, 4321)
    try:
        ms_total, _ = w.time_steps(20, 5)
        row = {"config": 0, "prec": "fp64", "nvec": cfg0.nvec, "filter_ms": round(ms_total / 20, 4),
               "note": "launch/latency bound: time only"}
        try:
            s = torch.cuda.Stream()
            s.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(s):
                w.stream = s
                w.step(); s.synchronize()
                gr = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gr, stream=s):
                    w.step()
                for _ in range(3):
                    gr.replay()
                s.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(s)
                for _ in range(20):
                    gr.replay()
                e1.record(s); s.synchronize()
                row["filter_ms_cuda_graph"] = round(e0.elapsed_time(e1) / 20, 4)
        except Exception as ex:                                   # graph capture is a convenience of the harness
            row["filter_ms_cuda_graph"] = None
            row["graph_error"] = str(ex)[:160]
        rows.append(row)
    finally:
        w.close()
    ALLP = ["fp64", "fp64m", "fp32", "fp32s", "tf32x3", "tf32"]
    for cfg_id, precs, nvecs in [(1, ALLP, [128]), (3, ALLP, [256]), (4, ALLP, [64, 128, 256, 512, 1024])]:
        cfg = inp.CONFIGS[cfg_id]
        pb = GpuProblem(cfg, seed=0, device=device)
        try:
            for nvec in nvecs:
                for prec in precs:
                    row = config_row(torch, B, cfg_id, prec, nvec, device, peak, pb=pb)
                    if cfg_id == 4 and nvec == 512:
                        row["also"] = "configs[2] (same mesh, 512 vectors, degree 24)"
                    if cfg_id == 3:
                        row["note"] = "one 256-vector chunk of configs[3]; the headline line runs all four"
                    rows.append(row)
        finally:
            pb.close()
    return rows



def tf32_tensor_peak():
    """Dense TF32 tensor peak in TFLOP/s: the measured bf16 peak x the nominal ratio of B200_PROFILING.md (1.1 / 2.25 PFLOP/s)."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["bf16_tflops"]) * 1.1 / 2.25, "MEASURED_PEAKS.json bf16_tflops x 1.1 / 2.25 (nominal TF32 : bf16)"
    except Exception:
        return 1100.0, "nominal 1.1 PFLOP/s dense TF32 (B200_PROFILING.md; MEASURED_PEAKS.json absent)"


def extra_kernels(torch, B, device, hbm_peak, pipe):
    """Rows for the NEXT components that are not part of a filter step: the BFP codec (HBM-bound) and the Rayleigh-Ritz
    projection / rotation (FMA-pipe bound; the roof is the issue rate measured in this run by chfsi_measure_pipe_peaks)."""
    dev = f"cuda:{device}"
    rows = []

    def timed(fn, reps=3):
        fn(); torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record(); torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    # ---- BFP codec on a face-slab stream of 2^28 FP32 values (1 GiB in): algorithmic bytes = 16 B in + n_bits/2 B out per block
    n = 1 << 28
    x = inp.make_ghost_values(1 << 20, seed=3)
    xd = torch.from_numpy(x).to(dev).repeat(n // x.size)
    for nbits in (16, 12, 10):
        sd = torch.empty(B.chfsi_bfp_stream_bytes(nbits, n), dtype=torch.uint8, device=dev)
        yd = torch.empty_like(xd)
        nbytes = 4.0 * n + sd.numel()
        t_enc = timed(lambda: B.chfsi_bfp_encode(nbits, xd, sd))
        t_dec = timed(lambda: B.chfsi_bfp_decode(nbits, sd, yd))
        for nm, t in (("bfp_encode", t_enc), ("bfp_decode", t_dec)):
            gbs = nbytes / (t * 1e-3) / 1e9
            rows.append({"kernel": nm, "n_bits": nbits, "values": n, "ms": round(t, 4), "bound": "hbm", "achieved_GBs": round(gbs, 1),
                         "peak_GBs": hbm_peak, "frac": round(gbs / hbm_peak, 4)})
        del sd, yd
    del xd
    torch.cuda.empty_cache()

    # ---- Rayleigh-Ritz pieces on configs[2]'s mesh rows (3.54M rows) x 256 vectors
    cfg = inp.CONFIGS[2]
    nv = 256
    mesh = B.chfsi_mesh_create(cfg.ncell, cfg.L, cfg.p, cfg.kfrac, device)
    B.chfsi_ham_set(mesh, None, None, None, None)
    try:
        g = torch.Generator(device=dev); g.manual_seed(77)
        Y = torch.empty((cfg.nnodes, 2, nv), dtype=torch.complex128, device=dev)
        Yr = torch.view_as_real(Y)
        for j0 in range(0, nv, 64):
            Yr[:, :, j0:j0 + 64, :] = torch.rand((cfg.nnodes, 2, 64, 2), generator=g, device=dev, dtype=torch.float64) - 0.5
        S = torch.empty((nv, nv), dtype=torch.complex128, device=dev)
        nrows = 2 * cfg.nnodes
        t = timed(lambda: B.chfsi_rr_project(mesh, Y, Y, S))
        nt = (nv + 63) // 64
        flops = 8.0 * nrows * 64 * 64 * (nt * (nt + 1) // 2)          # complex MAC = 8 flop; tiles on and above the diagonal
        rows.append({"kernel": "rr_project (Y^H M Y, Hermitian)", "rows": nrows, "nvec": nv, "ms": round(t, 3), "bound": "alu",
                     "achieved_TFs": round(flops / (t * 1e-3) / 1e12, 2), "peak_TFs": round(pipe["fp64_fma"], 2),
                     "frac": round(flops / (t * 1e-3) / 1e12 / pipe["fp64_fma"], 4), "dtype": "f64"})
        Q = torch.linalg.qr(torch.randn((nv, nv), dtype=torch.complex128, device=dev, generator=g))[0].contiguous()
        Yo = torch.empty_like(Y)
        wk = torch.empty(B.chfsi_rr_rotate_workspace_bytes(nv), dtype=torch.uint8, device=dev)
        flops = 8.0 * nrows * nv * nv
        for prec, nm, pk in ((B.FP32, "rr_rotate (FP64 diagonal + FP32 off-diagonal)", "fp32_fma"), (B.FP64, "rr_rotate (FP64)", "fp64_fma")):
            t = timed(lambda: B.chfsi_rr_rotate(prec, Y, Q, Yo, wk), reps=2)
            rows.append({"kernel": nm, "rows": nrows, "nvec": nv, "ms": round(t, 3), "bound": "alu",
                         "achieved_TFs": round(flops / (t * 1e-3) / 1e12, 2), "peak_TFs": round(pipe[pk], 2),
                         "frac": round(flops / (t * 1e-3) / 1e12 / pipe[pk], 4), "dtype": "f32 off-diagonal / f64 diagonal" if prec == B.FP32 else "f64"})
        # the same mixed rotation on tcgen05 (3xTF32): three TF32 products per term are executed; roof = the TF32 tensor peak,
        # taken as the measured bf16 peak of MEASURED_PEAKS.json x the guide's nominal TF32 : bf16 ratio (1.1 : 2.25)
        t = timed(lambda: B.chfsi_rr_rotate(B.TF32X3, Y, Q, Yo, wk), reps=3)
        tf32_peak, tf32_src = tf32_tensor_peak()
        rows.append({"kernel": "rr_rotate (FP64 diagonal + 3xTF32 off-diagonal on tcgen05)", "rows": nrows, "nvec": nv, "ms": round(t, 3),
                     "bound": "tensor", "achieved_TFs": round(3 * flops / (t * 1e-3) / 1e12, 2), "peak_TFs": round(tf32_peak, 1),
                     "frac": round(3 * flops / (t * 1e-3) / 1e12 / tf32_peak, 4), "peak_source": tf32_src,
                     "useful_TFs": round(flops / (t * 1e-3) / 1e12, 2), "hbm_GBs": round(2.0 * nrows * nv * 16 / (t * 1e-3) / 1e9, 1),
                     "dtype": "tf32 x3 off-diagonal (f32 accumulation) / f64 diagonal"})
    finally:
        B.chfsi_mesh_destroy(mesh)
        torch.cuda.empty_cache()

    # ---- Poisson: the Kx kernel and the batched PCG (Algorithm 2) on configs[3]'s mesh (96^3 nodes, p = 8), 64 right-hand sides
    cfg = inp.CONFIGS[3]
    nv = 16                                                   # 4 nv = 64 real columns
    mesh = B.chfsi_mesh_create(cfg.ncell, cfg.L, cfg.p, (0.0, 0.0, 0.0), device)
    B.chfsi_ham_set(mesh, None, None, None, None)
    try:
        g = torch.Generator(device=dev); g.manual_seed(78)
        U = torch.empty((cfg.nnodes, 2, nv), dtype=torch.complex128, device=dev)
        torch.view_as_real(U)[...] = torch.rand((cfg.nnodes, 2, nv, 2), generator=g, device=dev, dtype=torch.float64) - 0.5
        W = torch.empty_like(U)
        t = timed(lambda: B.chfsi_poisson_apply_K(mesh, U, W), reps=5)
        dofs = cfg.nnodes * 4.0 * nv
        nbytes = dofs * 32.0                                  # u read 8 B, w zero-filled 8 B, w read-modify-written 16 B
        rows.append({"kernel": "poisson Kx (memset + cell kernel)", "nodes": cfg.nnodes, "real_columns": 4 * nv, "ms": round(t, 4),
                     "dof_per_s": float(f"{dofs / (t * 1e-3):.4g}"), "bound": "hbm", "achieved_GBs": round(nbytes / (t * 1e-3) / 1e9, 1),
                     "peak_GBs": hbm_peak, "frac": round(nbytes / (t * 1e-3) / 1e9 / hbm_peak, 4), "dtype": "f64"})
        B.chfsi_poisson_set_quadrature(mesh, 1)
        t = timed(lambda: B.chfsi_poisson_apply_K(mesh, U, W), reps=3)
        B.chfsi_poisson_set_quadrature(mesh, 0)
        rows.append({"kernel": "poisson Kx, Gauss-Legendre form (the paper's six-contraction pipeline; untuned)", "nodes": cfg.nnodes,
                     "real_columns": 4 * nv, "ms": round(t, 4), "dof_per_s": float(f"{dofs / (t * 1e-3):.4g}"), "dtype": "f64"})
        mass = torch.from_numpy(B.chfsi_mesh_mass(mesh)).to(dev)
        F = U * mass[:, None, None]
        Fr = torch.view_as_real(F)
        Fr -= Fr.mean(dim=0, keepdim=True)                    # neutral right-hand sides
        kd = torch.from_numpy(B.chfsi_poisson_kdiag(mesh)).to(dev)
        # upper spectral bound of K_diag^-1 K: ten power steps in the K_diag inner product (harness side), plus 10 %
        V1 = torch.zeros((cfg.nnodes, 2, 1), dtype=torch.complex128, device=dev)
        W1 = torch.empty_like(V1)
        xv = torch.rand(cfg.nnodes, generator=g, device=dev, dtype=torch.float64) - 0.5
        lam = 1.0
        for _ in range(10):
            V1[:, 0, 0] = xv
            B.chfsi_poisson_apply_K(mesh, V1, W1)
            yv = W1[:, 0, 0].real / kd
            lam = float((kd * xv * yv).sum() / (kd * xv * xv).sum())
            xv = yv / yv.abs().max()
        lmax = 1.1 * lam
        X = torch.empty_like(F)
        wk = torch.empty(B.chfsi_poisson_workspace_bytes(mesh, nv), dtype=torch.uint8, device=dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        it, res = B.chfsi_poisson_pcg(mesh, F, X, 5, lmax / 30.0, lmax, 1e-10, 400, wk, check_every=10)
        e1.record(); torch.cuda.synchronize()
        tp = e0.elapsed_time(e1)
        rows.append({"kernel": "poisson PCG (Alg. 2, degree-5 Chebyshev-Jacobi, tol 1e-10)", "nodes": cfg.nnodes, "real_columns": 4 * nv,
                     "ms": round(tp, 2), "iterations_max": int(it.max()), "residual_max": float(res.max()),
                     "kx_dof_per_s": float(f"{dofs * 5 * int(it.max()) / (tp * 1e-3):.4g}"), "dtype": "f64"})
    finally:
        B.chfsi_mesh_destroy(mesh)
        torch.cuda.empty_cache()
    return rows

# --------------------------------------------------------------------------------------------
def run_e2e(torch, B, w, world, dist, barrier, n_steps):
    """The same filter through the C ABI with HOST buffers: every step uploads all of X from pinned host memory and
    downloads all of Y into pinned host memory inside the timed region.  The block moves through a FIXED ring of pinned
    slots (node ranges of a chunk are contiguous byte ranges, so every copy is a plain cudaMemcpyAsync); upload of chunk
    c+1 and download of chunk c-1 overlap the filter call on chunk c (three streams)."""
    cfg, nvec = w.cfg, w.nvec
    chunk = w.chunk or nvec
    nchunks = (nvec + chunk - 1) // chunk
    dev = w.X.device
    row_bytes = 2 * chunk * 16                                  # one node of a chunk
    slot_nodes = max(1, min(cfg.nnodes, int(1.0e9 // row_bytes)))    # ~1 GB slots
    npieces = (cfg.nnodes + slot_nodes - 1) // slot_nodes
    NSLOT = 4
    hin = [torch.empty((slot_nodes, 2, chunk), dtype=torch.complex128, pin_memory=True) for _ in range(NSLOT)]
    hout = [torch.empty((slot_nodes, 2, chunk), dtype=torch.complex128, pin_memory=True) for _ in range(NSLOT)]
    hin[0].copy_(w.X[:slot_nodes, :, :chunk])
    for h in hin[1:]:
        h.copy_(hin[0])
    Xd = [torch.empty((cfg.nnodes, 2, chunk), dtype=torch.complex128, device=dev) for _ in range(2)]
    Yd = [torch.empty((cfg.nnodes, 2, chunk), dtype=torch.complex128, device=dev) for _ in range(2)]
    work = w.pb.work(w.prec, w.recur, chunk)
    lam = w.lam
    s_in, s_out, stream = torch.cuda.Stream(), torch.cuda.Stream(), w.stream
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_c = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]
    state = {"piece": 0}

    def upload(c):
        with torch.cuda.stream(s_in):
            s_in.wait_event(ev_c[c % 2])                          # the filter call that read this buffer two chunks ago
            for p0 in range(npieces):
                n0, n1 = p0 * slot_nodes, min(cfg.nnodes, (p0 + 1) * slot_nodes)
                Xd[c % 2][n0:n1].copy_(hin[state["piece"] % NSLOT][: n1 - n0], non_blocking=True)
                state["piece"] += 1
            ev_in[c % 2].record(s_in)

    def download(c):
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_c[c % 2])
            for p0 in range(npieces):
                n0, n1 = p0 * slot_nodes, min(cfg.nnodes, (p0 + 1) * slot_nodes)
                hout[p0 % NSLOT][: n1 - n0].copy_(Yd[c % 2][n0:n1], non_blocking=True)
            ev_out[c % 2].record(s_out)

    def e2e_step():
        upload(0)
        for c in range(nchunks):
            if c + 1 < nchunks:
                upload(c + 1)
            stream.wait_event(ev_in[c % 2])
            stream.wait_event(ev_out[c % 2])                      # Yd[c % 2] was downloaded (two chunks ago)
            j0 = c * chunk
            nb = min(chunk, nvec - j0)
            B.chfsi_cheb_filter(w.pb.mesh, w.prec, w.recur, cfg.degree, w.a, w.b, w.a0, Xd[c % 2],
                                None if lam is None else lam[j0:j0 + nb], Yd[c % 2], work, stream=stream, nvec=nb)
            ev_c[c % 2].record(stream)
            download(c)

    for e in ev_c + ev_out:
        e.record(stream)
    e2e_step(); barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s_in.wait_stream(stream); s_out.wait_stream(stream)
    e0.record(s_in)
    for _ in range(n_steps):
        e2e_step()
        s_in.wait_stream(s_out)                                   # the next step's uploads start after this step's downloads were queued
    s_out.wait_stream(stream); s_out.wait_stream(s_in)
    e1.record(s_out)
    barrier()
    ms_e2e = e0.elapsed_time(e1) / n_steps
    if dist is not None:
        t = torch.tensor([ms_e2e], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_e2e = float(t.item())
    nbytes = cfg.nnodes * 2 * nvec * 16
    del Xd, Yd, hin, hout
    torch.cuda.empty_cache()
    return {"value": world * units_per_step(cfg, nvec) / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "ms_per_step": ms_e2e,
            "how": f"{nchunks} chunk(s) of {chunk} vectors; each chunk crosses PCIe as {npieces} contiguous node ranges through a fixed "
                   f"ring of {NSLOT}+{NSLOT} pinned slots of {slot_nodes * row_bytes / 1e9:.2f} GB; upload, filter and download "
                   f"pipelined on three streams"}


def run_ours(args, cfg):
    import torch
    from paper_2605_30128_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    if rank == 0:
        from paper_2605_30128_b200 import build as _build
        _build.build()                       # no-op when libchfsi.so is up to date
    if dist is not None:
        dist.barrier()
    B.lib()
    nvec = args.nvec or cfg.nvec

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    w = Workload(torch, B, cfg, args.prec, args.recur, nvec, local, 1234 + rank)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms_total, per_step = w.time_steps(args.steps, args.warmup, barrier)
    launches = B.chfsi_last_launch_count() * args.steps
    clocks = sampler.stop() if rank == 0 else None
    dev = f"cuda:{local}"
    ms_total, _ = aggregate_over_ranks(ms_total, 0.0, world, dist, dev)
    ms_step = ms_total / args.steps
    value = world * units_per_step(cfg, nvec) / (ms_step * 1e-3)
    assert bool(torch.isfinite(torch.view_as_real(w.Y[:, :, :8])).all()), "filter output is not finite"

    # ---- roofline of the dominant kernel (cell kernel), timed live with CUDA events on its stream
    big = units_per_step(cfg, nvec) > 5e9
    steps_prof = 1 if big else max(1, min(3, args.steps))
    cell_ms, cell_n, cell_bytes = w.cell_profile(steps_prof)
    peak, peak_src = measured_hbm_peak()
    achieved = cell_bytes / (cell_ms * 1e-3) / 1e9
    bpu = alg_bytes_per_unit(args.prec, args.recur)
    chunk_used = w.chunk
    roofline = {"bound": "hbm", "kernel": "cell kernel (gather + sum-factorised Laplacian + assembly + pointwise + update)",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "traffic": args.traffic if args.traffic is not None else ncu_traffic(args.config, args.prec, chunk_used or nvec),
                "avg_launch_ms": cell_ms / cell_n, "launches_per_step": cell_n // steps_prof,
                "share_of_step": (cell_ms / steps_prof) / ms_step,
                "alg_bytes_per_launch": cell_bytes / cell_n,
                "note": "launches timed with the nonlocal kernels on the same stream (the headline run forks them to a side stream)"}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    if args.no_e2e:
        nbytes = cfg.nnodes * 2 * nvec * 16
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "skipped": "--no-e2e"}
    else:
        e2e = run_e2e(torch, B, w, world, dist, barrier, max(1, min(args.steps, 2 if big else 5)))

    w.close()
    table, pipe, extra, eig = None, None, None, None
    if rank == 0 and world == 1 and not args.no_table:
        table = all_configs_table(torch, B, local, peak)
        pipe = B.chfsi_measure_pipe_peaks(local)
        extra = extra_kernels(torch, B, local, peak, pipe)
        eig = eigen_check(torch, B, local)

    # ---- CPU oracle baseline on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        per = max(1, args.ref_cols // 3)            # ~ a third of the single-process sample per core
        try:
            rate, dt, cores = cpu_oracle_rate_all_cores(cfg, per)
            cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle (numpy, one process per host core)", "seconds": dt,
                   "sample": f"{cores * per} of {cfg.nvec} columns of {cfg.name} ({per} per process), full degree {cfg.degree}, eq. 11 FP64"}
        except Exception as ex:                      # fall back to the single-process timing of the same oracle
            rate, dt, cores = cpu_oracle_rate(cfg, args.ref_cols)
            cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle (numpy, single process)", "seconds": dt,
                   "sample": f"{args.ref_cols} of {cfg.nvec} columns of {cfg.name}, full degree {cfg.degree}, eq. 11 FP64",
                   "note": f"all-cores run failed: {str(ex)[:80]}"}

    if rank == 0:
        nbytes = cfg.nnodes * 2 * nvec * 16
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "median_ms_per_step": float(np.median(per_step)),
            "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": DTYPE[args.prec], "data": "synthetic",
            "config": {"workload": workload_name(args, cfg, nvec, chunk_used),
                       "l2": f"inputs larger than L2 (each multivector {nbytes / 1e6:.0f} MB vs 126 MB L2)",
                       "parallelism": "columns sharded, no exchange" if world > 1 else "1 GPU"},
            "units_per_step": units_per_step(cfg, nvec), "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu,
            "gpu_launches": int(launches), "clocks": clocks,
            "roofline_whole_filter": {"alg_bytes_per_unit": bpu, "frac_of_hbm_peak": value / world * bpu / (peak * 1e9)},
            "all_configs": table,
            "pipe_peaks_TFs": pipe, "other_kernels": extra, "config4_eigenvalues": eig,
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--prec", default=None, choices=["fp64", "fp64m", "fp32", "fp32s", "tf32", "tf32x3"])
    ap.add_argument("--recur", default="residual", choices=["residual", "standard"])
    ap.add_argument("--nvec", type=int, default=0)
    ap.add_argument("--ref-cols", type=int, default=0, help="columns in the CPU-oracle sample")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-table", action="store_true", help="skip the all-config table")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per cell-kernel launch (overrides the value read from profiles/)")
    args = ap.parse_args()
    cfg = inp.CONFIGS[args.config]
    if args.ref_cols <= 0:
        # about 10-20 s of oracle time: ~1e7 units/s on one host core
        args.ref_cols = max(1, min(cfg.nvec, int(round(1.5e8 / (2.0 * cfg.nnodes * cfg.degree)))))
    if args.prec is None:
        args.prec = "fp64"            # the paper's reference arithmetic; --prec fp32 / fp32s select the inexact modes
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
