#!/usr/bin/env python
"""bench.py -- R-ChFSI filter throughput (dof x vector x Chebyshev-step per second) on B200.

One "step" = one pass of the whole hot path (Algorithm 2: FP64 residual set-up, (m-1) x
[projection + couplings, fused cell kernel = S^-1approx, cell contraction, ordered assembly, recurrence bracket], recovery)
over all N/B vector blocks of the workload = one "SCF-equivalent pass".

Workload at N=1: the LARGEST single-GPU configuration of BASELINE.json, configs[4] (32^3 cells, p=6, Dirichlet, 7.19M stored
dofs, 5,000 vectors in blocks of 256, degree 30).  Its 5,000 FP32 vectors (144 GB) do not fit beside the operators (47 GB)
and the workspace, so a pass cycles through the distinct blocks that do fit (config.resident_blocks) and every timed call
filters a fresh device copy of a block (7.4 GB >> L2).  `--config 1|2|3` run the other configs (all blocks resident where
they fit), `--all-configs` prints one line per config 1-4.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 4] [--prec tf32]

Multi-GPU: the path does not shard in this build ("replicas only"): under torchrun every rank
filters its own replica of the workload on its own GPU; value = all ranks' units / max-over-ranks time.
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from pawfe_inputs import get_config, make_system, random_block, twin  # noqa: E402

METRIC = "chfsi_filter_dof_vec_steps_per_s"
UNIT = "dof*vec*steps/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sust=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sust=1400.0, src="fallback")


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline of the own arm, and the whole `--impl reference` arm)
# ------------------------------------------------------------------------------------------------
class OracleSample:
    """A bounded sample of the workload for the CPU oracle: the reduced-cell twin of the config (same p, h,
    potential, projector set, BC, k-point; 4^3 cells), B_o columns, m_o Chebyshev steps.  SpMM cost is
    linear in dofs, columns and steps, so dof*vec*steps/s of the sample is the oracle's rate."""

    def __init__(self, cfg_id: int, cols: int = 32, degree: int = 8):
        from oracle import chfsi
        from oracle.operators import PawOperators
        self.chfsi = chfsi
        base = get_config(cfg_id)
        self.cfg = twin(base, nc=4, natoms=3, nvec=cols, block=cols, degree=degree)
        self.ops = PawOperators(make_system(self.cfg))
        ops = self.ops
        X0 = random_block(self.cfg, cols, stream=7) * ops.mask[:, None]
        X = chfsi.s_orthonormalise(ops.apply_S, X0)
        self.X, self.lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
        self.bU = chfsi.lanczos_upper_bound(ops.apply_H, ops.apply_Sinv, ops.mesh.M, k=10, seed=1,
                                            dtype=ops.dtype, mask=ops.mask)
        self.units = float(ops.mesh.M) * cols * degree
        self.desc = (f"oracle.chfsi.filter_residual (FP64, scipy CSR) on the {self.cfg.ncells[0]}^3-cell twin of "
                     f"config {cfg_id} ({ops.mesh.M} dofs), {cols} vectors, degree {degree}; operators prebuilt")

    def step(self):
        o = self.ops
        self.chfsi.filter_residual(o.apply_H, o.apply_S, o.apply_Sinv, self.X, self.lam, self.cfg.degree,
                                   self.lam[0] - 0.1, self.lam[-1] + 0.05, self.bU)


def _cores_used() -> int:
    # scipy CSR products are single-threaded; the small dense numpy parts may use BLAS threads
    return 1


def _host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    smp = OracleSample(args.config)
    for _ in range(max(1, min(args.warmup, 2))):
        smp.step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        smp.step()
    dt = time.perf_counter() - t0
    val = smp.units * args.steps / dt
    cfg = get_config(args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "sample": smp.desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": _cores_used(), "host_cores": _host_cores(), "kind": "oracle",
                         "sample": smp.desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
            out, _ = self.p.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in out.strip().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nme, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
# multi-rank host logic (replicas only: no collective on the data path)
# ------------------------------------------------------------------------------------------------
def max_over_ranks(x: float, world: int, device=None) -> float:
    """Slowest rank's time: the job's time (bench contract).  Works with nccl (device tensor) and gloo (CPU)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank_per_step: float, steps: int, world: int, ms_max: float) -> float:
    """Aggregate throughput of `world` replicas that each processed the same units in ms_max (max over ranks)."""
    return world * units_per_rank_per_step * steps / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------------------
# own arm
# ------------------------------------------------------------------------------------------------
def run_own(args):
    import torch
    import torch.distributed as dist
    from paper_2604_26037_b200 import build
    build.build()
    from paper_2604_26037_b200 import PREC, FP64, context_from_system
    from paper_2604_26037_b200.harness import Harness

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libpawfe has no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    prec = PREC[args.prec]
    cfg = get_config(args.config)
    if args.block > 0:   # experiment only: another block width than BASELINE.json's (named in config.workload)
        import dataclasses
        cfg = dataclasses.replace(cfg, block=args.block, name=f"{cfg.name}_B{args.block}")
    sysd = make_system(cfg)
    stream = torch.cuda.current_stream()
    t_setup = time.perf_counter()
    ctx = context_from_system(sysd, device=local, stream=stream.cuda_stream)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t_setup
    M, N, B, m = ctx.num_dofs(), cfg.nvec, cfg.block, cfg.degree
    cplx = cfg.complex
    cw = 2 if cplx else 1
    hz = Harness(ctx, M, cplx)
    shape = (M, B, 2) if cplx else (M, B)
    nblk = (N + B - 1) // B
    widths = [min(B, N - b * B) for b in range(nblk)]     # the last block of config 4 has 136 vectors
    # plans, scratch and operand streams of the hot calls are built here, not inside the timed region (pawfe_prepare)
    ctx.prepare(prec, B, m)
    nbytes = ctx.filter_workspace(prec, B)
    tdt = torch.float64 if prec == FP64 else torch.float32
    es = (8 if prec == FP64 else 4) * cw
    blk_bytes = M * B * es
    # How many DISTINCT blocks stay resident.  All of them where they fit (configs 1-3); otherwise (config 4) as many as
    # leave room for the workspace, a scratch block and the FP64 temporaries of the input preparation below.
    free_b, _tot = torch.cuda.mem_get_info(dev)
    tmp_bytes = int(4.5 * M * B * 8 * cw)
    fit = int((free_b - nbytes - blk_bytes - tmp_bytes - (4 << 30)) // blk_bytes)
    nres = max(2, min(nblk, fit)) if args.resident_blocks <= 0 else min(nblk, args.resident_blocks)
    nres = min(nres, nblk)

    # inputs: seeded U[-0.5, 0.5] blocks, S-orthonormalised per block, Ritz values
    # from a per-block Rayleigh-Ritz, b_U from a 10-step Lanczos on H S^-1approx; all with the library's applies.
    gen = torch.Generator(device=dev).manual_seed(cfg.seed + 1000 * rank)
    blocks, lams = [], []
    for b in range(nres):
        X0 = torch.rand(shape, dtype=torch.float64, device=dev, generator=gen) - 0.5
        X = hz.s_orthonormalise(X0)
        del X0
        X, lam = hz.rayleigh_ritz(X)
        blocks.append(X.to(tdt).contiguous())
        del X
        lams.append(lam)
    torch.cuda.empty_cache()
    bU = hz.upper_bound(k=10, seed=1)
    b0 = min(l[0] for l in lams) - 0.1
    bW = min(max(l[-1] for l in lams), 0.5 * (b0 + bU))
    free_b, _tot = torch.cuda.mem_get_info(dev)
    room = int((free_b - nbytes - blk_bytes - (6 << 30)) // max(1, nres * blk_bytes))
    ring_n = max(1, min(args.steps + args.warmup, args.ring, room + 1))
    ring = [blocks] + [[x.clone() for x in blocks] for _ in range(ring_n - 1)]
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    # A block must not be filtered twice in place: with random (mid-spectrum) Ritz blocks the components below b0 grow by
    # ~1e5 per call.  When blocks are reused (cycled resident blocks, or fewer ring copies than steps), each call filters a
    # fresh device-to-device copy; the copy is inside the timed region (< 0.5% of a call).
    reuse = nres < nblk or ring_n < args.steps + args.warmup
    scratch = torch.empty_like(blocks[0]) if reuse else None

    def one_step(i):
        blks = ring[i % ring_n]
        for b in range(nblk):
            x, w = blks[b % nres], widths[b]
            if reuse:
                scratch.copy_(x)
                x = scratch
            ctx.cheb_filter(prec, m, b0, bW, bU, x, lams[b % nres][:w], B, w, ws, nbytes)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        one_step(i)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ctx.cell_timing(True)
    l0 = ctx.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for i in range(args.steps):
        one_step(args.warmup + i)
    ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    ncell_launch, cell_ms = ctx.cell_timing_read()
    nsetup, setup_ms = ctx.setup_timing_read()
    ctx.cell_timing(False)
    launches = ctx.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms = max_over_ranks(ms, world, dev)
    finite = all(bool(torch.isfinite(x).all()) for blks in ring for x in blks) and (scratch is None or bool(torch.isfinite(scratch).all()))

    # ---- end to end through the C ABI with HOST buffers: H2D of each block, filter, D2H of Psi_f, inside the timed region ----
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    cycled = nres < nblk
    if cycled:
        e2e_steps = 1
    if not cycled:
        # one pinned host copy of the block set per call (warm-up + e2e_steps): never filter a host block twice in place
        host_sets = [[x.cpu().pin_memory() for x in ring[0]] for _ in range(1 + e2e_steps)]
    else:
        # cycled resident blocks: two pinned SOURCE blocks and two PAIRS of pinned WORK blocks; each call filters one pair in
        # place (copies of the pair's second block run under the first block's filter) while a helper thread refills the
        # other pair from the sources -- the host-side refill is not part of the path
        src = [ring[0][k].cpu().pin_memory() for k in range(2)]
        work = [[torch.empty_like(src[0]).pin_memory() for _ in range(2)] for _ in range(2)]
    del ring, blocks, ws, scratch  # the host-buffer call owns its own device block and workspace
    torch.cuda.empty_cache()

    def e2e_pass_all(k):
        hs = host_sets[k]
        # the pass's blocks in one call: copies of blocks k+1 / k-1 run under block k's filter
        ctx.cheb_filter_host_set(prec, m, b0, bW, bU, [x.data_ptr() for x in hs], [lams[b][:widths[b]] for b in range(nblk)],
                                 [B] * nblk, widths)

    def e2e_pass_cycled(nb):
        import threading

        def refill(pair):
            for q in range(2):
                work[pair][q].copy_(src[q])
        refill(0)
        for b0_ in range(0, nb, 2):
            pair = (b0_ // 2) % 2
            t = None
            if b0_ + 2 < nb:
                t = threading.Thread(target=refill, args=(1 - pair,))
                t.start()
            ws_ = [widths[(b0_ + q) % nblk] for q in range(min(2, nb - b0_))]
            ctx.cheb_filter_host_set(prec, m, b0, bW, bU, [work[pair][q].data_ptr() for q in range(len(ws_))],
                                     [lams[q][:w] for q, w in enumerate(ws_)], [B] * len(ws_), ws_)
            if t is not None:
                t.join()

    if cycled:
        e2e_pass_cycled(2)          # warm-up: sizes the library's internal device block and workspace
    else:
        e2e_pass_all(0)
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        if cycled:
            e2e_pass_cycled(nblk)
        else:
            e2e_pass_all(1 + k)
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    e2e_s = max_over_ranks(e2e_s, world, dev)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    units = float(M) * N * m                      # per rank per step
    value = whole_job_value(units, args.steps, world, ms)
    peaks = _peaks()
    n = (cfg.p + 1) ** 3
    ncell = cfg.ncells[0] * cfg.ncells[1] * cfg.ncells[2]
    kname = ctx.cell_kernel_name(prec, B)
    fused = "tcgen05" in kname
    passes = 3 if "3xtf32" in kname else 1
    # the cell kernel is launched (m - 1) x passes times per filter call, each time on the call's own width
    launches_per_step = sum(1 for _ in widths) * (m - 1) * passes
    cell_avg_ms = cell_ms / max(1, ncell_launch)
    Bavg = float(N) / nblk                         # mean block width of a pass (config 4: 19 x 256 + 136)
    flops_launch = 2.0 * n * n * Bavg * ncell * (4 if cplx else 1)
    tflops = flops_launch / (cell_avg_ms * 1e-3) / 1e12 if cell_avg_ms > 0 else 0.0
    # Roofline of the dominant kernel.  k_cell_tcgen05 now IS the fused Chebyshev step (gather, S^-1approx
    # through the K-extension, contraction, ordered assembly, bracket of Alg. 2 step 4), so its algorithmic bytes per launch
    # are SURVEY.md 8(d)'s per-step figure: the H^e stream 4 n^2 N_c (x2 complex) + 20 B per dof*vec (read R_Y 4, R_X 4,
    # Y FP64 8, write R_X 4; x2 complex).  FP32 mode (three passes): the same bytes per pass for the first pass.
    bytes_launch = 4.0 * n * n * ncell * cw + 20.0 * M * Bavg * cw
    gbs = bytes_launch / (cell_avg_ms * 1e-3) / 1e9 if cell_avg_ms > 0 else 0.0
    if fused:
        peak_t = 0.5 * peaks["bf16_sust"]
        roof = {"kernel": f"k_cell_tcgen05 ({kname}: fused step)", "bound": "hbm", "achieved": gbs, "peak": peaks["hbm"], "unit": "GB/s",
                "frac": gbs / peaks["hbm"], "traffic": None,
                "traffic_source": "not measured in this run; ncu --set full captures per launch: profiles/r02_cell_kernel_ordered.md",
                "peak_source": f"{peaks['src']} copy bandwidth", "algorithmic_bytes_per_launch": bytes_launch,
                "algorithmic_bytes_per_dof_vec": bytes_launch / (M * Bavg),
                "tensor": {"achieved_tflops": tflops, "peak_tflops": peak_t, "frac": tflops / peak_t,
                           "peak_source": f"0.5 x {peaks['src']} sustained bf16 (nominal TF32:bf16 ratio; TF32 itself not measured)"}}
    else:
        mhz = (clocks or {}).get("sm_mhz") or 1965.0
        peak = 148 * 128 * 2 * mhz * 1e6 / 1e12 * (0.5 if prec == FP64 else 1.0)
        roof = {"kernel": kname, "bound": "tensor" if "dmma" in kname else "alu", "achieved": tflops, "peak": peak, "unit": "TFLOP/s",
                "frac": tflops / peak if peak else None, "traffic": None,
                "peak_source": "148 SM x 128 lanes x 2 flop x SM clock under load (FP64: half, the DMMA / DFMA rate)"}
    roof.update({"launches": ncell_launch, "avg_ms": cell_avg_ms, "share_of_step": cell_ms / ms})
    # whole-step and recurrence-only views: total = a1-a8; recurrence-only = total minus the residual set-up
    step_bytes = bytes_launch / (M * Bavg)
    rec_ms = ms - setup_ms
    rec_value = world * float(M) * N * (m - 1) * args.steps / (rec_ms * 1e-3) if rec_ms > 0 else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {"fp64": "f64", "fp32": "f32", "tf32": "tf32"}[args.prec], "data": "synthetic",
        "config": {"workload": cfg.name, "dofs": M, "vectors": N, "block": B, "degree": m, "precision": args.prec,
                   "cells": ncell, "fe_order": cfg.p, "atoms": cfg.natoms, "projectors": cfg.nproj,
                   "pairs": ctx.num_pairs(), "parallelism": "replicas only" if world > 1 else "single GPU",
                   "cache": f"inputs >> L2: {nres} distinct resident blocks of {blk_bytes / 2**30:.2f} GiB x {ring_n} ring copies"
                            f" + {nbytes / 2**30:.1f} GiB workspace; every timed call filters a block that is not in L2",
                   "resident_blocks": nres, "blocks_per_pass": nblk, "filters_fresh_copy": reuse,
                   "bounds": [b0, bW, bU], "finite": finite, "setup_s": t_setup},
        "clocks": clocks,
        "e2e": {"value": world * units / e2e_s, "unit": UNIT, "h2d_bytes_per_step": nblk * blk_bytes,
                "d2h_bytes_per_step": nblk * blk_bytes, "steps": e2e_steps,
                "how": "pawfe_cheb_filter_host_set on pairs of pinned work blocks (refilled by a helper thread between calls)" if cycled
                       else "pawfe_cheb_filter_host_set (copies pipelined under the filters)"},
        "gpu_launches": launches,
        "roofline": roof,
        "step_hbm": {"algorithmic_bytes_per_dof_vec_step": step_bytes,
                     "achieved_gbs": step_bytes * value / world / 1e9, "peak_gbs": peaks["hbm"],
                     "frac": step_bytes * value / world / 1e9 / peaks["hbm"]},
        "phases": {"residual_setup_ms_per_step": setup_ms / args.steps, "residual_setup_share": setup_ms / ms,
                   "recurrence_only_value": rec_value, "recurrence_only_unit": "dof*vec*(m-1 steps)/s, residual set-up excluded",
                   "cell_kernel_launches_expected_per_step": launches_per_step, "filter_calls_timed": nsetup},
    }
    if world == 1 and not args.no_cpu_baseline:
        smp = OracleSample(args.config)
        smp.step()
        t0 = time.perf_counter()
        reps = 0
        while reps < 3 or (time.perf_counter() - t0 < 10.0 and reps < 50):
            smp.step()
            reps += 1
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": smp.units * reps / dt, "unit": UNIT, "cores": _cores_used(), "host_cores": _host_cores(),
                                "kind": "oracle", "sample": smp.desc + f"; {reps} calls in {dt:.1f} s"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_all_configs(args):
    """one line per config 1-4 (each in its own process, so that every config starts from an empty device)"""
    for c in (1, 2, 3, 4):
        cmd = [sys.executable, os.path.abspath(__file__), "--config", str(c), "--steps", str(args.steps), "--warmup", str(args.warmup),
               "--prec", args.prec, "--no-cpu-baseline"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        out = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
        print(out[-1] if out else json.dumps({"config": c, "error": r.stderr[-500:]}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--prec", default="tf32", choices=["fp64", "fp32", "tf32"])
    ap.add_argument("--ring", type=int, default=8)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--resident-blocks", type=int, default=0, help="distinct vector blocks kept in HBM (0 = all)")
    ap.add_argument("--block", type=int, default=0, help="override the config's block width B (0 = BASELINE.json's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--all-configs", action="store_true", help="one line per config 1-4, each in its own process")
    args = ap.parse_args()
    if args.all_configs:
        run_all_configs(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_own(args)


if __name__ == "__main__":
    main()
