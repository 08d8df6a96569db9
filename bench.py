#!/usr/bin/env python
"""Benchmark of the Chebyshev-filter hot path (BASELINE.json metric) on B200.

A "step" is one `chfsi_cheb_filter` call -- residual S0, m-1 recurrence steps, recover S7, i.e.
every row of SURVEY.md §8(a) -- on BASELINE.json configs[1]: 8x8x8 periodic cells, side 16 Bohr,
p = 6 (48^3 nodes, 221,184 complex DoF), 128 complex128 vectors, 8 atoms x 8 projectors,
Chebyshev degree 20, FP64 throughout, the residual-based recurrence (eq. 11).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1] [--prec fp64]

N > 1 (under torchrun): the filter shards over columns with no exchange (the paper's band
partitioning in its n_r = 1 limit): every rank filters its own 128-vector block of
the same mesh, value = all ranks' units / max-over-ranks time, scaling "weak".
`--impl reference` times the CPU oracle (oracle/fe_oracle.py, as it stands) on a bounded sample.
Prints ONE JSON line.
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

from paper_2605_30128_b200 import inputs as inp  # noqa: E402

METRIC = "chebyshev_filter_throughput"
UNIT = "complex_DoF*vectors*degree/s"
FALLBACK_HBM_GBS = 6650.0        # /opt/skills/guides/B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum per cell-kernel launch from the committed `ncu --set full`
# captures (profiles/r1_final_c1_ncu_full.md), keyed by (config, precision); None where no capture exists
NCU_TRAFFIC = {(1, "fp64"): 1.823e9, (1, "fp32"): 1.826e9}


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


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


def units_per_step(cfg, nvec):
    return 2.0 * cfg.nnodes * nvec * cfg.degree


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


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    ncols = max(1, args.ref_cols // 4)      # each of the K + W steps is a bounded sample (~4 s): the run ends in about a minute
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
        "config": {"workload": f"BASELINE configs[{args.config}] ({cfg.name}): {cfg.ncell}^3 cells p={cfg.p}, "
                               f"{cfg.nvec} vectors, degree {cfg.degree}, eq. 11", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------
def run_ours(args, cfg):
    import torch
    from paper_2605_30128_b200 import binding as B
    from paper_2605_30128_b200.harness import GpuProblem

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
    dev = f"cuda:{local}"
    prec = B.PREC[args.prec]
    recur = B.RECUR_RESIDUAL if args.recur == "residual" else B.RECUR_STANDARD
    nvec = args.nvec or cfg.nvec
    chunk = cfg.chunk if (cfg.chunk and cfg.chunk < nvec) else 0

    pb = GpuProblem(cfg, seed=0, device=local)
    g = torch.Generator(device=dev); g.manual_seed(1234 + rank)
    shape = (cfg.nnodes, 2, nvec)
    X = torch.complex(torch.rand(shape, generator=g, device=dev, dtype=torch.float64) * 2 - 1,
                      torch.rand(shape, generator=g, device=dev, dtype=torch.float64) * 2 - 1)
    Y = torch.empty_like(X)
    a0, b = pb.lanczos_bounds(10)
    a = a0 + 0.1 * (b - a0)
    lam = pb.rayleigh_quotients(X) if recur == B.RECUR_RESIDUAL else None
    work = pb.work(prec, recur, chunk if chunk else nvec)
    stream = torch.cuda.current_stream()

    def step():
        B.chfsi_cheb_filter(pb.mesh, prec, recur, cfg.degree, a, b, a0, X, lam, Y, work, chunk=chunk, stream=stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = B.chfsi_last_launch_count() * args.steps
    clocks = sampler.stop() if rank == 0 else None
    if dist is not None:
        t = torch.tensor([ms_total], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = world * units_per_step(cfg, nvec) / (ms_step * 1e-3)
    assert bool(torch.isfinite(Y.real).all()), "filter output is not finite"

    # ---- roofline of the dominant kernel (cell kernel), timed live with CUDA events on its stream
    B.chfsi_profile_enable(pb.mesh, True)
    for _ in range(max(1, min(3, args.steps))):
        step()
    cell_ms, cell_n, cell_bytes = B.chfsi_profile_read(pb.mesh)
    B.chfsi_profile_enable(pb.mesh, False)
    peak, peak_src = measured_hbm_peak()
    achieved = cell_bytes / (cell_ms * 1e-3) / 1e9
    steps_prof = max(1, min(3, args.steps))
    roofline = {"bound": "hbm", "kernel": "cell_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src,
                "traffic": args.traffic if args.traffic is not None else (NCU_TRAFFIC.get((args.config, args.prec)) if nvec == cfg.nvec else None),
                "avg_launch_ms": cell_ms / cell_n, "launches_per_step": cell_n // steps_prof,
                "share_of_step": (cell_ms / steps_prof) / ms_step,
                "alg_bytes_per_launch": cell_bytes / cell_n}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    # (X and Y themselves are the device buffers: the host copy of X is what was uploaded before)
    nbytes = X.numel() * 16
    if args.no_e2e or nbytes > args.e2e_max_gb * 1e9:
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
               "skipped": f"host staging of 2 x {nbytes / 1e9:.1f} GB pinned buffers not attempted (--e2e-max-gb)"}
    else:
        # The host holds the block as `nblk` band blocks (column groups, each [M, 2, nvec/nblk] contiguous and
        # pinned); block i+1 is uploaded and block i-1 downloaded while block i is filtered (three streams).
        nblk = 4 if (nvec % 4 == 0 and nvec >= 64) else 1
        cw = nvec // nblk
        bshape = (cfg.nnodes, 2, cw)
        Xh = [torch.empty(bshape, dtype=torch.complex128, pin_memory=True) for _ in range(nblk)]
        Yh = [torch.empty(bshape, dtype=torch.complex128, pin_memory=True) for _ in range(nblk)]
        for i in range(nblk):
            Xh[i].copy_(X[:, :, i * cw:(i + 1) * cw])
        Xd = [torch.empty(bshape, dtype=torch.complex128, device=dev) for _ in range(nblk)]
        Yd = [torch.empty(bshape, dtype=torch.complex128, device=dev) for _ in range(nblk)]
        lam_b = [None if lam is None else lam[i * cw:(i + 1) * cw] for i in range(nblk)]
        work_b = pb.work(prec, recur, cw)
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        ev_in = [torch.cuda.Event() for _ in range(nblk)]
        ev_c = [torch.cuda.Event() for _ in range(nblk)]

        def e2e_step():
            for i in range(nblk):
                with torch.cuda.stream(s_in):
                    Xd[i].copy_(Xh[i], non_blocking=True)
                    ev_in[i].record(s_in)
                stream.wait_event(ev_in[i])
                B.chfsi_cheb_filter(pb.mesh, prec, recur, cfg.degree, a, b, a0, Xd[i], lam_b[i], Yd[i], work_b,
                                    stream=stream)
                ev_c[i].record(stream)
                s_out.wait_event(ev_c[i])
                with torch.cuda.stream(s_out):
                    Yh[i].copy_(Yd[i], non_blocking=True)

        e2e_step(); barrier()
        n_e2e = max(1, min(args.steps, 5))
        s_in.wait_stream(stream); s_out.wait_stream(stream)
        e0.record(s_in)
        for _ in range(n_e2e):
            e2e_step()
            s_in.wait_stream(s_out)          # the next step's uploads start after this step's downloads were queued
        s_out.wait_stream(stream); s_out.wait_stream(s_in)
        e1.record(s_out)
        barrier()
        ms_e2e = e0.elapsed_time(e1) / n_e2e
        if dist is not None:
            t = torch.tensor([ms_e2e], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms_e2e = float(t.item())
        e2e = {"value": world * units_per_step(cfg, nvec) / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "ms_per_step": ms_e2e,
               "how": f"{nblk} pinned host band blocks of {cw} vectors; upload, filter and download pipelined on three streams"}

    # ---- CPU oracle baseline on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        rate, dt, cores = cpu_oracle_rate(cfg, args.ref_cols)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"{args.ref_cols} of {cfg.nvec} columns of {cfg.name}, full degree {cfg.degree}, eq. 11 FP64"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if args.prec == "fp64" else "f32 product / f64 recurrence",
            "data": "synthetic",
            "config": {"workload": f"BASELINE configs[{args.config}] ({cfg.name}): {cfg.ncell}^3 cells, side {cfg.L} Bohr, "
                                   f"p={cfg.p}, {2 * cfg.nnodes} complex DoF, {nvec} complex128 vectors, "
                                   f"{cfg.natoms} atoms x {cfg.nproj} projectors, degree {cfg.degree}, "
                                   f"recurrence {args.recur}, prec {args.prec}, chunk {chunk or nvec}",
                       "l2": f"inputs larger than L2 (each multivector {nbytes / 1e6:.0f} MB vs 126 MB L2)",
                       "parallelism": "columns sharded, no exchange" if world > 1 else "1 GPU"},
            "units_per_step": units_per_step(cfg, nvec), "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu,
            "gpu_launches": int(launches), "clocks": clocks,
            "roofline_whole_filter": {"alg_bytes_per_unit": 64 if recur == B.RECUR_RESIDUAL else 48,
                                      "frac_of_hbm_peak": value / world * (64 if recur == B.RECUR_RESIDUAL else 48) / (peak * 1e9)},
        }
        print(json.dumps(line))
    pb.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--prec", default=None, choices=["fp64", "fp32"])
    ap.add_argument("--recur", default="residual", choices=["residual", "standard"])
    ap.add_argument("--nvec", type=int, default=0)
    ap.add_argument("--ref-cols", type=int, default=0, help="columns in the CPU-oracle sample")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-max-gb", type=float, default=8.0, help="skip the host-staged e2e leg above this block size")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per cell-kernel launch from the committed ncu capture (profiles/)")
    args = ap.parse_args()
    cfg = inp.CONFIGS[args.config]
    if args.ref_cols <= 0:
        # about 10-20 s of oracle time: ~8.5e6 units/s on one host core
        args.ref_cols = max(1, min(cfg.nvec, int(round(1.2e8 / (2.0 * cfg.nnodes * cfg.degree)))))
    if args.prec is None:
        args.prec = cfg.prec if args.config != 1 else "fp64"
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
