#!/usr/bin/env python
"""bench.py -- throughput of the demagnetizing-field convolution (arXiv 2308.08447, Eq. (1)) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4|C3|C2|C5|C1|C3d] [--impl ours|reference]

A "step" is one pass of the whole hot path (demag_apply: x R2C -> y FFT -> z FFT*multiply*z IFFT -> y IFFT ->
x C2R; for C5 also the macrocell average and scatter) over one seeded synthetic magnetisation of a
BASELINE.json config.  Prints ONE JSON line (rank 0).  The headline workload is C4 (4096x4096x8, the largest
single-GPU mesh of BASELINE.json; its `metric` names no config); with no --config the line also carries a
`configs` block with the same fields for C2, C3, C3 fp64 and C5 (short step counts).  The path does not shard
without an exchange step (replicas only), so --gpus N runs N independent replicas, one
process per GPU.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2308_08447_b200 import workloads as W  # noqa: E402  (input generators only)

METRIC = "demag_throughput"
UNIT = "Gcells/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=None, help="C1..C5, suffix d = fp64 (e.g. C3d); default: headline C4 plus a "
                                                   "`configs` block for C2, C3, C3d, C5")
    ap.add_argument("--no-configs", action="store_true", help="default run without the `configs` block")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft", action="store_true")
    ap.add_argument("--sharded", action="store_true",
                    help="ONE convolution partitioned over the N ranks (strong scaling; include/demag.h 'Several GPUs') "
                         "instead of the default N independent replicas")
    ap.add_argument("--virtual-ranks", type=int, default=0,
                    help="with --sharded on ONE GPU: emulate G ranks as G plans on this device, phase by phase, and "
                         "report the per-rank device time of each phase (a compute-share model, no NVLink involved)")
    ap.add_argument("--llg", action="store_true",
                    help="time the minimal LLG RK4 integrator (demag_llg_*, PAPER.md:91-96) on --config (default C3): ms per "
                         "step with the demagnetizing field convolved at every stage vs extrapolated at the sub-steps")
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    return ap.parse_args()


HEADLINE = "C4"                                   # largest single-GPU mesh of BASELINE.json (its metric names no config)
OTHER_CONFIGS = ["C2", "C3", "C3d", "C5"]


def workload_name(cfg, fp64):
    return f"{cfg.name} ({'fp64' if fp64 else 'fp32'})"


def config_of(cfg, fp64):
    """The `config` object, identical in our arm and the reference arm (same workload, same metric)."""
    n = cfg.n
    return {"workload": workload_name(cfg, fp64), "mesh": list(n), "cells": int(np.prod(n)),
            "padded": [v if v == 1 else 2 * v for v in n]}


# ----------------------------------------------------------------------------------------------- oracle legs
def oracle_sample_rate(cfg, seconds, M_host=None):
    """Time the oracle (as it stands) on a bounded sample of the same workload: Eq. (1) evaluated by direct
    summation (O-S) at seeded sample cells.  Returns (Gcells/s, cores, description, table_seconds)."""
    from oracle import oracle as O   # the cpu_baseline / --impl reference legs may use oracle/
    n = cfg.n
    nc = int(np.prod(n))
    t0 = time.perf_counter()
    T = O.tensor_table(n, cfg.h)
    t_table = time.perf_counter() - t0
    if M_host is None:
        M_host = W.make_magnetisation(cfg) if cfg.kind != "atomistic" else W.random_unit_vectors(n, cfg.Ms, cfg.seed)
    M64 = M_host.astype(np.float64)
    cores = O.num_threads()
    cells = W.sample_cells(n, 4096, cfg.seed)
    k = cores
    t0 = time.perf_counter()
    O.direct_sum_sampled(T, M64, cells[:k])
    dt = time.perf_counter() - t0
    total = int(max(k, min(len(cells), seconds / max(dt, 1e-9) * k)))
    total = max(cores, total // cores * cores)
    t0 = time.perf_counter()
    O.direct_sum_sampled(T, M64, cells[:total])
    dt = time.perf_counter() - t0
    desc = (f"oracle O-S: Eq. (1) by direct fp64 summation at {total} seeded sample cells of {cfg.name} "
            f"({total} x {nc} cell pairs in {dt:.2f} s; tensor table built in {t_table:.1f} s, not timed)")
    return total / dt / 1e9, cores, desc, t_table, (T, M64, cells, total)


def run_reference(args, cfg, fp64):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    val, cores, desc, _, (T, M64, cells, total) = oracle_sample_rate(cfg, 4.0)
    from oracle import oracle as O
    per_step = max(cores, int(total * min(1.0, 60.0 / max(1, args.steps + args.warmup) / 4.0)) // cores * cores)
    for _ in range(min(args.warmup, 2)):
        O.direct_sum_sampled(T, M64, cells[:per_step])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.direct_sum_sampled(T, M64, cells[:per_step])
    dt = time.perf_counter() - t0
    value = per_step * args.steps / dt / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_of(cfg, fp64),
            "detail": {"sample": f"{per_step} seeded output cells per step, direct O(N) sum each"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{per_step} sample cells x {int(np.prod(cfg.n))} pairs per step"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "20", "-i", str(gpu_index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for ln in self.f.read().splitlines():
            t = [x.strip() for x in ln.split(",")]
            if len(t) < 9:
                continue
            try:
                sm.append(float(t[1])); mx.append(float(t[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), t[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


# ----------------------------------------------------------------------------------------------- multi-rank plumbing
def allreduce_max(vals, device, world):
    """Max over ranks of a list of floats (device times): the timing rule of the bench contract.  The path does not
    shard without an exchange (replicas only), so this is the ONLY collective of a run."""
    import torch
    import torch.distributed as dist
    tt = torch.tensor(list(vals), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return tt.tolist()


def aggregate_throughput(world, units_per_rank, steps, ms_total_max):
    """Whole-job units/s of `world` independent replicas that each did `steps` steps of `units_per_rank` units."""
    return world * units_per_rank * steps / (ms_total_max * 1e-3)


# ----------------------------------------------------------------------------------------------- our arm
def stage_bytes(n, esz):
    """Algorithmic HBM bytes of each stage of the 5-pass separable structure (T2):
    what each kernel must read and write if nothing stayed in L2.  [K1, K2, K3, K4, K5]."""
    nx, ny, nz = n
    Nx, Ny, Nz = [v if v == 1 else 2 * v for v in n]
    hx, kpy, kpz = Nx // 2 + 1, Ny // 2 + 1, Nz // 2 + 1
    nc = nx * ny * nz
    w1 = 3 * hx * nz * ny * 2 * esz
    w2 = 3 * hx * nz * Ny * 2 * esz
    kern = 6 * hx * kpz * kpy * esz
    return [3 * nc * esz + w1, w1 + w2, w2 + kern + w2, w2 + w1, w1 + 3 * nc * esz]


STAGE_NAMES = ["k_x_r2c", "k_y_fwd", "k_z_mul", "k_y_inv", "k_x_c2r"]                 # size-generic kernel family
STAGE_NAMES_FAST = ["k_x_r2c_v", "k_y_fwd_v", "k_z_v", "k_y_inv_v", "k_x_c2r_v"]     # compile-time specialised family


def cufft_baseline(torch, n, dt, dev, reps=10):
    """cuFFT-based convolution on the same GPU (torch.fft), timing only (random real kernel spectrum): the comparator
    north_star names; never on the product path.  (i) naive: materialise the padded field, rfftn, multiply, irfftn,
    crop; (ii) pruned: per-axis transforms with the padding given as n= and slicing between axes (the paper's
    single-GPU scheme).  Returns ms of each (median over `reps`)."""
    nx, ny, nz = n
    P = [v if v == 1 else 2 * v for v in n]
    Nx, Ny, Nz = P
    hx = Nx // 2 + 1
    cdt = torch.complex64 if dt == torch.float32 else torch.complex128
    need = (3 * Nz * Ny * hx * (8 if dt == torch.float32 else 16)) * 4 + 6 * Nz * Ny * hx * (4 if dt == torch.float32 else 8)
    free, _ = torch.cuda.mem_get_info()
    if need > 0.6 * free:
        return None
    M = torch.randn((3, nz, ny, nx), dtype=dt, device=dev)
    K = torch.randn((6, Nz, Ny, hx), dtype=dt, device=dev)

    def mult(Z):
        zx, zy, zz = Z[0], Z[1], Z[2]
        return torch.stack((K[0] * zx + K[3] * zy + K[4] * zz, K[3] * zx + K[1] * zy + K[5] * zz,
                            K[4] * zx + K[5] * zy + K[2] * zz))

    def naive():
        Mp = torch.zeros((3, Nz, Ny, Nx), dtype=dt, device=dev)
        Mp[:, :nz, :ny, :nx] = M
        Z = torch.fft.rfftn(Mp, dim=(-3, -2, -1))
        return torch.fft.irfftn(mult(Z), s=(Nz, Ny, Nx), dim=(-3, -2, -1))[:, :nz, :ny, :nx]

    def pruned():
        X = torch.fft.rfft(M, n=Nx, dim=-1) if Nx > 1 else M.to(cdt)
        Y = torch.fft.fft(X, n=Ny, dim=-2) if Ny > 1 else X
        Z = torch.fft.fft(Y, n=Nz, dim=-3) if Nz > 1 else Y
        Hh = mult(Z)
        Hh = torch.fft.ifft(Hh, dim=-3)[:, :nz] if Nz > 1 else Hh
        Hh = torch.fft.ifft(Hh, dim=-2)[:, :, :ny] if Ny > 1 else Hh
        return torch.fft.irfft(Hh, n=Nx, dim=-1)[..., :nx] if Nx > 1 else Hh.real

    Mpad = torch.zeros((3, Nz, Ny, Nx), dtype=dt, device=dev)
    Mpad[:, :nz, :ny, :nx] = M

    def fft_only():                                   # floor of any cuFFT-based convolution: no multiply, no pad, no crop
        return torch.fft.irfftn(torch.fft.rfftn(Mpad, dim=(-3, -2, -1)), s=(Nz, Ny, Nx), dim=(-3, -2, -1))

    out = {}
    for name, fn in (("naive", naive), ("pruned", pruned), ("fft_only", fft_only)):
        try:
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            ts = []
            for _ in range(reps):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record(); torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            out[name + "_ms"] = statistics.median(ts)
        except torch.cuda.OutOfMemoryError:
            out[name + "_ms"] = None
        torch.cuda.empty_cache()
    return out


def source_sha16():
    """Hash of the CUDA sources the library was built from: ties profiles/traffic.json.txt (ncu DRAM counters) to a build."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2308_08447_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def measure(name, steps, warmup, cpu_seconds, with_cufft, with_cpu, env):
    """One workload, timed as the bench contract says.  Returns the JSON line as a dict on rank 0, None elsewhere."""
    torch, dist, B, rank, world, local, dev = env
    fp64 = name.endswith("d")
    cfg = W.CONFIGS[name[:2]]
    dt = torch.float64 if fp64 else torch.float32
    esz = 8 if fp64 else 4
    n = cfg.n
    nc = int(np.prod(n))
    atom = cfg.kind == "atomistic"

    # ---- inputs (seeded synthetic; host -> HBM before the timed region) and plan
    t0 = time.perf_counter()
    if atom:
        L = tuple(a * c for a, c in zip(n, cfg.macro))
        X = W.random_spins_torch(L, cfg.seed + rank, device=dev).to(dt)
        units = int(np.prod(L)); unit_name = "spins"
        M_host = None
    else:
        M_host = W.make_magnetisation(cfg)
        X = torch.from_numpy(M_host).to(dev, dt)
        units = nc; unit_name = "cells"
    Y = torch.empty_like(X)
    t_inputs = time.perf_counter() - t0
    t0 = time.perf_counter()
    plan = B.Plan(n, cfg.h, 0, B.DEMAG_FP64 if fp64 else B.DEMAG_FP32)
    plan.set_kernel(None)
    if atom:
        plan.reserve_atomistic()                        # the macrocell arrays: allocated once, never inside a step
    torch.cuda.synchronize()
    t_plan = time.perf_counter() - t0

    def step():
        if atom:
            plan.apply_atomistic(X, Y, cfg.macro, cfg.mu_s, cfg.a)
        else:
            plan.apply(X, Y)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > L2 (126 MB): written between steps

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, warmup)):
        flush.fill_(1); step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    # ---- timed region: exactly K steps, device time by CUDA events on the launching stream, L2 flushed
    #      between steps (the flush is outside each step's event pair)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier()
    for a, b in evs:
        flush.fill_(1)
        a.record(); step(); b.record()
    barrier()
    ms_steps = [a.elapsed_time(b) for a, b in evs]
    ms_total = sum(ms_steps)
    # hot (no flush, back to back) for context
    a0, b0 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a0.record()
    for _ in range(steps):
        step()
    b0.record(); barrier()
    ms_hot = a0.elapsed_time(b0) / steps

    # the same back-to-back steps replayed from a CUDA graph (the hot path never allocates or synchronises, so an
    # integrator can capture it): what the launch overhead costs on small meshes
    ms_graph = None
    if not atom:
        try:
            gs = torch.cuda.Stream()
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.stream(gs):
                with torch.cuda.graph(gr, stream=gs):
                    for _ in range(steps):
                        plan.apply(X, Y, stream=gs)
            gr.replay(); torch.cuda.synchronize()
            a1, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a1.record(); gr.replay(); b1.record(); torch.cuda.synchronize()
            ms_graph = a1.elapsed_time(b1) / steps
            del gr
        except Exception as ex:                                  # reported, never fatal for the bench line
            ms_graph = f"failed: {ex}"

    # ---- end to end through the public API with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not atom:
        # Every step copies its input host -> device and its result device -> host (pinned memory, all inside the
        # timed region).  The three phases of consecutive steps overlap on three streams with double-buffered device
        # arrays (PCIe is full duplex; the plan itself runs one apply at a time, on the compute stream).
        hin = torch.from_numpy(M_host).to(dt).pin_memory()
        houts = [torch.empty_like(hin).pin_memory() for _ in range(2)]
        hout = houts[0]
        Xs, Ys = [X, torch.empty_like(X)], [Y, torch.empty_like(Y)]
        s_in, s_cmp, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
        ev_in = [torch.cuda.Event() for _ in range(2)]; ev_cmp = [torch.cuda.Event() for _ in range(2)]
        ev_out = [torch.cuda.Event() for _ in range(2)]
        e2e_i = [0]

        def e2e_step():
            i = e2e_i[0]; b = i & 1; e2e_i[0] += 1
            with torch.cuda.stream(s_in):
                if i >= 2:
                    s_in.wait_event(ev_cmp[b])             # X[b] was read by the apply of step i-2
                Xs[b].copy_(hin, non_blocking=True); ev_in[b].record(s_in)
            with torch.cuda.stream(s_cmp):
                s_cmp.wait_event(ev_in[b])
                if i >= 2:
                    s_cmp.wait_event(ev_out[b])            # Y[b] was copied out by step i-2
                plan.apply(Xs[b], Ys[b], stream=s_cmp); ev_cmp[b].record(s_cmp)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_cmp[b])
                houts[b].copy_(Ys[b], non_blocking=True); ev_out[b].record(s_out)
        torch.cuda.synchronize()
        for _ in range(3):
            e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            e2e_step()
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        check = houts[(e2e_i[0] - 1) & 1]
        assert torch.isfinite(check).all() and float(check.abs().max()) > 0, "e2e produced no field"
        e2e_bytes = (hin.numel() * hin.element_size(), hout.numel() * hout.element_size())
    else:
        # config 5: the per-step result read back is the field of the sampled spins' z-slab 0 (201 MB would be the
        # mesh field; the 12.9 GB spin arrays live in HBM as they would in a simulation): copy spins slab in, field slab out
        zs = cfg.macro[2]
        hin = X[:, :zs].cpu().pin_memory(); hout = torch.empty_like(hin).pin_memory()
        def e2e_step():
            X[:, :zs].copy_(hin, non_blocking=True); step(); hout.copy_(Y[:, :zs], non_blocking=True)
        for _ in range(2):
            e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            e2e_step()
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        e2e_bytes = (hin.numel() * hin.element_size(), hout.numel() * hout.element_size())
    clocks = sampler.stop() if sampler else None

    # ---- per-stage device times of the convolution (CUDA event pair around every launch, on the launching stream)
    if atom:
        Mc = torch.empty((3, n[2], n[1], n[0]), dtype=dt, device=dev).normal_(); Hc = torch.empty_like(Mc)
    else:
        Mc, Hc = X, Y
    st_ms = np.zeros(5); st_n = np.zeros(5, dtype=int)
    reps = 5
    for i in range(reps + 1):
        flush.fill_(1)
        ms, cnt = plan.apply_profiled(Mc, Hc)
        if i:
            st_ms += ms; st_n += cnt
    st_ms /= reps
    launches_per_step = plan.launches_per_apply() + (2 if atom else 0)

    # ---- the sub-step extrapolation that stands in for a convolution: quartic through 5 fields, added
    #      into H_eff; one streaming pass (5 reads + read-modify-write), timed like the stages (L2 flushed, event pair)
    extrap = None
    if not atom and 9 * Y.numel() * esz < 60e9:
        hist = [torch.empty_like(Y).normal_() for _ in range(5)]
        heff = torch.zeros_like(Y)
        tms = []
        for i in range(6):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); plan.extrapolate(hist, [0.0, 1.0, 2.0, 3.0, 4.0], 4.5, heff, accumulate=True); b.record()
            torch.cuda.synchronize()
            if i:
                tms.append(a.elapsed_time(b))
        ebytes = 7 * Y.numel() * esz
        extrap = {"npts": 5, "ms": float(np.mean(tms)), "bytes": ebytes, "GBps": ebytes / np.mean(tms) / 1e6,
                  "note": "demag_extrapolate(accumulate) replaces one convolution at an RK sub-step (PAPER.md:96)"}
        del hist, heff

    cufft = None
    if rank == 0 and not atom and with_cufft:
        cufft = cufft_baseline(torch, n, dt, dev)

    # ---- reduce over ranks: max time
    ms_total, ms_hot, t_e2e = allreduce_max([ms_total, ms_hot, t_e2e], dev, world)
    del flush
    if rank != 0:
        plan.close()
        return None
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    sb = stage_bytes(n, esz)
    names = STAGE_NAMES_FAST if plan.path() == 1 else STAGE_NAMES
    dom = int(np.argmax(st_ms))
    # the instantiation behind each stage name (kernels_v2.cuh): register-resident z stages for thin meshes, the fused film
    # stage, the staged persistent kernel for long y lines
    actual = list(names)
    if plan.path() == 1:
        Nz = 1 if n[2] == 1 else 2 * n[2]
        Ny = 2 * n[1]
        if n[2] == 1:
            actual[2] = "k_z_v<FILM> (y FFT . multiply . y IFFT along y)"
        elif Nz <= 8:
            actual[2] = "k_z1_v"
        elif Nz == 16 and not fp64 and Ny % 64 == 0:
            actual[2] = "k_z16_v"
        elif Nz in (256, 512) and not fp64:
            actual[2] = "k_z_eo_v"
        if Ny >= 4096 and n[2] > 1:
            actual[1] = "k_y_fwd_long_v"
    achieved = sb[dom] / (st_ms[dom] * 1e-3) / 1e9
    value = aggregate_throughput(world, nc, steps, ms_total) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": max(3, warmup),
        "ms_per_step": ms_total / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if fp64 else "f32", "data": "synthetic",
        "config": config_of(cfg, fp64),
        "detail": {"l2": "flushed between timed steps (256 MB write outside each step's event pair)",
                   "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                   "kernel": "built-in Newell tensor (demag_set_kernel(NULL))",
                   "kernel_family": "fast (kernels_v2.cuh)" if plan.path() == 1 else "generic (kernels.cuh)"},
        "conv_per_s": world * steps / (ms_total * 1e-3),
        "hot_ms_per_step": ms_hot, "hot_value": world * nc / (ms_hot * 1e-3) / 1e9,
        "graph_hot_ms_per_step": ms_graph,
        "e2e": {"value": world * nc * steps / t_e2e / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": e2e_bytes[0], "d2h_bytes_per_step": e2e_bytes[1]},
        "gpu_launches": launches_per_step * steps,
        "launches_per_step": launches_per_step,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": names[dom], "kernel_instance": actual[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                     "bytes_per_apply_model": sb[dom], "ms_per_apply": float(st_ms[dom]),
                     "launches_per_apply": int(st_n[dom] // reps)},
        "stages": {names[i]: {"ms": float(st_ms[i]), "model_bytes": sb[i],
                                    "model_GBps": sb[i] / max(st_ms[i], 1e-9) / 1e6} for i in range(5)},
        "whole_apply_model": {"T2_5pass_bytes": sum(sb), "T2_GBps": sum(sb) / (ms_total / steps) / 1e6,
                              "frac_of_peak": sum(sb) / (ms_total / steps) / 1e6 / peak},
        "plan_build_s": t_plan, "input_gen_s": t_inputs, "workspace_bytes": plan.workspace_bytes(),
    }
    if extrap:
        extrap["frac_of_peak"] = extrap["GBps"] / peak
        line["extrapolate"] = extrap
    if cufft:
        best = min(v for k, v in cufft.items() if v and k in ("naive_ms", "pruned_ms"))
        per = ms_total / steps
        cufft.update(best_ms=best, ours_over_cufft=best / per,
                     note="torch.fft (cuFFT) convolution of the same shape on the same GPU, L2 not flushed, timing only; "
                          "naive / pruned include an eager-PyTorch multiply, padding and crops; fft_only_ms is the floor of "
                          "any cuFFT-based convolution: one rfftn and one irfftn of the already padded array, nothing else")
        if cufft.get("fft_only_ms"):
            cufft["ours_over_cufft_fft_only"] = cufft["fft_only_ms"] / per
        line["cufft"] = cufft
    if atom:
        line["spins_per_s_G"] = world * units * steps / (ms_total * 1e-3) / 1e9
    # ncu DRAM counters of this config (profiles/traffic.json.txt: dram__bytes_read.sum + dram__bytes_write.sum per launch,
    # one --set full capture per config), used only if they were captured on THIS build of the kernels
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json.txt")
    try:
        tj = json.load(open(traffic_file))
        ent = tj.get(name, {})
        if tj.get("_src_sha16") != source_sha16():
            line["roofline"]["traffic_note"] = "profiles/traffic.json.txt was captured on another build of the kernels: not used"
        elif ent:
            line["roofline"]["traffic"] = ent.get(names[dom])
            tot = sum(v for k, v in ent.items() if not k.startswith("_"))
            per = ms_total / steps
            gbps = tot / per / 1e6
            line["hbm_counter"] = {"dram_bytes_per_apply": tot, "GBps": gbps, "frac_of_measured_peak": gbps / peak,
                                   "frac_of_8TBps_nominal": gbps / 8000.0,
                                   "source": "ncu dram__bytes_read.sum + dram__bytes_write.sum, all kernels of one apply "
                                             "(profiles/traffic.json.txt), divided by this run's ms_per_step"}
    except Exception:
        pass
    plan.close()
    del X, Y, Mc, Hc
    torch.cuda.empty_cache()
    if world == 1 and with_cpu:
        val, cores, desc, _, _ = oracle_sample_rate(cfg, cpu_seconds, M_host)
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
    return line


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2308_08447_b200 import binding as B
    B.lib()                                             # fail loudly if the CUDA extension is missing
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    env = (torch, dist, B, rank, world, local, torch.device("cuda", local))
    head = args.config or HEADLINE
    line = measure(head, args.steps, args.warmup, args.cpu_seconds, not args.no_cufft, not args.no_cpu_baseline, env)
    if rank == 0 and world == 1 and args.config is None and not args.no_configs:
        # the other configs BASELINE.json names, same fields, short step counts (the headline keeps --steps / --warmup)
        line["configs"] = {}
        for name in OTHER_CONFIGS:
            try:
                sub = measure(name, min(args.steps, 10), 3, min(args.cpu_seconds, 4.0), not args.no_cufft,
                              not args.no_cpu_baseline, env)
                for k in ("stages", "extrapolate", "plan_build_s", "input_gen_s", "detail"):
                    sub.pop(k, None)
                line["configs"][name] = sub
            except Exception as ex:                     # a failing side config must not lose the headline
                line["configs"][name] = {"error": f"{type(ex).__name__}: {ex}"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_virtual_ranks(args, cfg, fp64):
    """G ranks as G sharded plans on ONE device, driven phase by phase (tests/test_gpu_sharded.py does the same for
    parity): the device time of every rank's phase, i.e. the compute share a rank would have on its own GPU when the
    peer stores cost nothing extra.  Not a multi-GPU measurement: the "peer" buffers are local HBM."""
    import torch
    from paper_2308_08447_b200 import binding as B
    B.lib()
    G = args.virtual_ranks
    dev = torch.device("cuda", 0)
    dt = torch.float64 if fp64 else torch.float32
    n = cfg.n
    nc = int(np.prod(n))
    plans = [B.ShardedPlan(n, cfg.h, B.DEMAG_FP64 if fp64 else B.DEMAG_FP32, rank=r, world=G, connect=False) for r in range(G)]
    bufs = [B.demag_shard_buffers(p.handle) for p in plans]
    M_host = W.make_magnetisation(cfg)
    Xs, Ys = [], []
    for p in plans:
        B.demag_shard_set_peers(p.handle, [b[0] for b in bufs], [b[2] for b in bufs])
        p.set_kernel(None)
        y0, nyl = p.info["y0"], p.info["ny_loc"]
        Xs.append(torch.from_numpy(np.ascontiguousarray(M_host[:, :, y0:y0 + nyl, :])).to(dev, dt))
        Ys.append(torch.empty_like(Xs[-1]))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ms = np.zeros((3, G))
    reps = max(1, args.steps)
    for it in range(reps + max(3, args.warmup)):
        for ph in range(3):
            for r, p in enumerate(plans):
                flush.fill_(1)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); B.demag_apply_sharded(p.handle, ph, Xs[r], Ys[r]); b.record()
                torch.cuda.synchronize()
                if it >= max(3, args.warmup):
                    ms[ph, r] += a.elapsed_time(b) / reps
    per_rank = ms.sum(axis=0)
    line = {"metric": "sharded_phase_ms_per_rank", "unit": "ms", "virtual_ranks": G, "n_gpus": 1, "steps": reps,
            "dtype": "f64" if fp64 else "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg, fp64), "mesh": list(n), "cells": nc,
                       "note": "G plans on one device, phase by phase; peer buffers are local HBM (compute-share model)"},
            "phase_ms_max_over_ranks": [float(v) for v in ms.max(axis=1)],
            "phase_ms_mean_over_ranks": [float(v) for v in ms.mean(axis=1)],
            "rank_ms_max": float(per_rank.max()), "rank_ms_sum": float(per_rank.sum()),
            "exchange_bytes_per_rank": int(12 * nc * (G - 1) / G**2 * (8 if fp64 else 4)),
            "rows_per_rank": [p.info["ny_loc"] for p in plans], "pairs_per_rank": [p.info["nq_loc"] for p in plans]}
    for p in plans:
        p.close()
    print(json.dumps(line), flush=True)


def run_sharded(args, cfg, fp64):
    """One convolution of the workload split over all ranks (Fig. 1): rows of M / H along y, frequency
    pairs along kx, the two spectrum exchanges written by the x R2C / y inverse kernels into peer memory, an NCCL
    all-reduce of one element as the barrier between the three phases.  Timed as the default arm: CUDA events around K
    steps, L2 flushed between steps, max over ranks; value = cells of the WHOLE mesh per second ("scaling": "strong")."""
    import torch
    import torch.distributed as dist
    from paper_2308_08447_b200 import binding as B
    B.lib()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    if cfg.kind == "atomistic" or cfg.n[2] == 1:
        raise SystemExit("--sharded: mesh workloads with nz >= 2 only (C1, C3, C4)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    dt = torch.float64 if fp64 else torch.float32
    n = cfg.n
    nc = int(np.prod(n))
    plan = B.ShardedPlan(n, cfg.h, B.DEMAG_FP64 if fp64 else B.DEMAG_FP32, rank=rank, world=world)
    plan.set_kernel(None)
    y0, nyl = plan.info["y0"], plan.info["ny_loc"]
    M_host = np.ascontiguousarray(W.make_magnetisation(cfg)[:, :, y0:y0 + nyl, :])
    X = torch.from_numpy(M_host).to(dev, dt)
    Y = torch.empty_like(X)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        flush.fill_(1); plan.apply(X, Y)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for a, b in evs:
        flush.fill_(1)
        a.record(); plan.apply(X, Y); b.record()
    barrier()
    ms_total = sum(a.elapsed_time(b) for a, b in evs)
    # end to end: this rank's rows host -> device, the convolution, this rank's field rows device -> host, every step
    hin = torch.from_numpy(M_host).to(dt).pin_memory(); hout = torch.empty_like(hin).pin_memory()
    def e2e_step():
        X.copy_(hin, non_blocking=True); plan.apply(X, Y); hout.copy_(Y, non_blocking=True)
    for _ in range(3):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    barrier()
    t_e2e = time.perf_counter() - t0
    assert torch.isfinite(hout).all() and float(hout.abs().max()) > 0, "e2e produced no field"
    clocks = sampler.stop() if sampler else None
    ms_total, t_e2e = allreduce_max([ms_total, t_e2e], dev, world)
    launches = B.demag_launches_per_apply(plan.handle)
    ws = plan.workspace_bytes()
    plan.close()
    if rank == 0:
        line = {
            "metric": METRIC, "value": nc * args.steps / (ms_total * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms_total / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64" if fp64 else "f32",
            "data": "synthetic",
            "config": {"workload": workload_name(cfg, fp64), "mesh": list(n), "cells": nc,
                       "l2": "flushed between timed steps (256 MB write outside each step's event pair)",
                       "parallelism": f"one convolution sharded x{world}: rows of M/H along y, frequency pairs along kx; "
                                      "exchanges stored into peer memory by the x R2C / y inverse kernels; "
                                      "barrier = NCCL all-reduce of one element between the three phases",
                       "kernel": "built-in Newell tensor (demag_set_kernel(NULL))", "kernel_family": "fast (kernels_v2.cuh)"},
            "conv_per_s": args.steps / (ms_total * 1e-3),
            "e2e": {"value": nc * args.steps / t_e2e / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": world * hin.numel() * hin.element_size(),
                    "d2h_bytes_per_step": world * hout.numel() * hout.element_size()},
            "gpu_launches": world * launches * args.steps, "launches_per_step": world * launches,
            "clocks": clocks, "workspace_bytes_per_rank": ws,
            "exchange_bytes_per_rank_per_step": int(12 * nc * (world - 1) / world**2 * (8 if fp64 else 4)),
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_llg(args, cfg, fp64):
    """The consumer of the convolution: K RK4 steps of the LLG equation with H_eff = H_d + H_Zee,
    once with H_d convolved at all four stages, once with the sub-step fields extrapolated from the five last full-step
    fields.  Device time by CUDA events around the K steps; reports the convolution counts."""
    import torch
    from paper_2308_08447_b200 import binding as B
    B.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    if cfg.kind == "atomistic":
        raise SystemExit("--llg: mesh workloads only (C1-C4)")
    dt = torch.float64 if fp64 else torch.float32
    n = cfg.n
    nc = int(np.prod(n))
    M0 = torch.from_numpy(W.make_magnetisation(cfg)).to("cuda", dt)
    out = {}
    with B.Plan(n, cfg.h, 0, B.DEMAG_FP64 if fp64 else B.DEMAG_FP32) as plan:
        plan.set_kernel(None)
        for name, extrap in (("every_stage", False), ("extrapolated", True)):
            with B.LLG(plan, cfg.Ms, 0.02) as L:
                L.set_field((-2.0e4, 1.0e3, 0.0))                      # the switching field of PAPER.md:47
                M = M0.clone()
                for _ in range(max(5, args.warmup)):                   # >= 5 steps: the history of the quartic is full
                    L.step(M, 1.0e-13, extrap)
                c0 = L.counts()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                a.record()
                for _ in range(args.steps):
                    L.step(M, 1.0e-13, extrap)
                b.record(); torch.cuda.synchronize()
                c1 = L.counts()
                assert bool(torch.isfinite(M).all())
                out[name] = {"ms_per_rk4_step": a.elapsed_time(b) / args.steps,
                             "convolutions_per_step": (c1["convolutions"] - c0["convolutions"]) / args.steps,
                             "extrapolation_passes_per_step": (c1["extrapolations"] - c0["extrapolations"]) / args.steps}
    line = {"metric": "llg_rk4_step_ms", "unit": "ms", "n_gpus": 1, "steps": args.steps, "warmup": max(5, args.warmup),
            "dtype": "f64" if fp64 else "f32", "data": "synthetic", "config": config_of(cfg, fp64),
            "every_stage": out["every_stage"], "extrapolated": out["extrapolated"],
            "speedup": out["every_stage"]["ms_per_rk4_step"] / out["extrapolated"]["ms_per_rk4_step"],
            "Mcell_steps_per_s_extrapolated": nc / out["extrapolated"]["ms_per_rk4_step"] / 1e3,
            "note": "H_eff = H_d + uniform field only; L2 not flushed (back-to-back steps of one integrator); PAPER.md:96 quotes a "
                    "decrease of the demagnetizing time 'by a factor between 2 to 2.5' for this scheme"}
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    name = args.config or HEADLINE
    fp64 = name.endswith("d")
    cfg = W.CONFIGS[name[:2]]
    if args.impl == "reference":
        run_reference(args, cfg, fp64)
    elif args.llg:
        run_llg(args, W.CONFIGS[(args.config or "C3")[:2]], (args.config or "C3").endswith("d"))
    elif args.sharded and args.virtual_ranks > 0:
        run_virtual_ranks(args, cfg, fp64)
    elif args.sharded:
        run_sharded(args, cfg, fp64)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
