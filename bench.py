#!/usr/bin/env python
"""bench.py - unrolled COSMO iterations/s (forward + backward, batched) on B200, with roofline + CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--ckpt full|lean] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: cdu_forward (K_unroll ADMM
iterations: xi assembly, PCG, relaxation, cone projections, checkpoint store) + cdu_backward (BPTT: cone VJPs
incl. Dalecki-Krein, adjoint PCG, Eq. 6), SURVEY.md 8(a) rows S1-S13. One JSON line is printed by rank 0.

metric = "unrolled COSMO iters/s (fwd+bwd, batched)" (BASELINE.json): value = K_unroll * steps * n_gpus / time,
i.e. batch-wide ADMM iterations (each advancing all B problems, forward and reverse) per second.
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

import workloads as W  # noqa: E402

METRIC = "unrolled_cosmo_iters_per_s_fwd_bwd_batched"
UNIT = "iters/s"
WORKLOADS = {"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5}
FP32_ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x FP32 lanes x 2 (FMA) x max SM clock
FP64_ALU_PEAK_TFLOPS = FP32_ALU_PEAK_TFLOPS / 2.0        # assumed 1:2, not measured


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
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
            except Exception:
                continue
            for n, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


# ---------------------------------------------------------------------------------------------------------
# algorithmic work per launch
# ---------------------------------------------------------------------------------------------------------
def csr_stream_bytes(M, w):
    return M.nnz * (w + 4) + 4 * (M.shape[0] + 1)


def lin_bytes(wl, ncg_fwd, ncg_bwd, full_ckpt):
    """Algorithmic HBM bytes of ONE launch of the forward / backward linear-step kernel over the batch, with the
    single-pass (a = 1) operator of SURVEY.md 8(d): per problem
      fwd: S_A (2 + (ncg+1)) + S_P (ncg+1) + 8 (3n + 5m) + checkpoint write
      bwd: S_A (3 + ncg')    + S_P ncg'    + 8 (4n + 8m) + checkpoint read
    ncg / ncg' = measured mean CG iterations per solve (all passes) in this run; the state is fp64 (8 bytes)."""
    w = 4 if wl.dtype == "f32" else 8
    f = b = 0.0
    for pr in wl.problems:
        SA, SP = csr_stream_bytes(pr.A, w), csr_stream_bytes(pr.P, w) if pr.P.nnz else 0
        ck = 8 * (pr.n + 2 * pr.m) + (8 * (pr.n + pr.m) if full_ckpt else 0)
        f += SA * (2 + ncg_fwd + 1) + SP * (ncg_fwd + 1) + 8 * (3 * pr.n + 5 * pr.m) + ck
        b += SA * (3 + ncg_bwd) + SP * ncg_bwd + 8 * (4 * pr.n + 8 * pr.m) + ck
    return f, b


def psd_orders(wl):
    return [d for pr in wl.problems for (k, d) in pr.cones if k == W.generators.PSD]


def jacobi_flops(ps, sweeps_sum_per_launch):
    """Two-sided Jacobi as executed: per sweep 12 p^3 flops (2x2 block update 32 flops x (p/2)^2 blocks + eigenvector
    update 8 flops x p x p/2 pairs, p-1 rounds), plus 1.5 p^3 for the clamp/rebuild. sweeps = measured."""
    if not ps:
        return 0.0
    p3 = float(np.mean([p ** 3 for p in ps]))
    return 12.0 * p3 * sweeps_sum_per_launch + 1.5 * p3 * len(ps)


# ---------------------------------------------------------------------------------------------------------
def make_workload(cfg, rank, batch=None, K=None, p=None):
    wl = W.make_config(cfg, batch=batch, K=K, p=p, seed_offset=7919 * rank)   # weak scaling: own instances per rank
    return wl


def cpu_oracle_time(wl, n_problems, K_sample):
    """Oracle (as it stands) forward+backward on a bounded sample; returns seconds per problem-iteration."""
    from oracle import cosmo_oracle as O
    t0 = time.perf_counter()
    for b in range(n_problems):
        pr = wl.problems[b]
        un = O.unroll(pr, K_sample, wl.rho[:K_sample], wl.alpha[:K_sample], wl.sigma, wl.x0[b], wl.s0[b], wl.y0[b])
        cot = O.terminal_loss_grad(pr, un.xs[-1], un.ss[-1], un.ys[-1], np.zeros(pr.n))
        O.backward(pr, un, *cot)
    dt = time.perf_counter() - t0
    return dt / (n_problems * K_sample), dt


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        return len(os.sched_getaffinity(0))


CPU_SAMPLE = {1: (4, 20), 2: (2, 50), 3: (8, 100), 4: (1, 100), 5: (1, 12)}   # (problems, iterations)


def cpu_baseline(wl, cfg):
    npb, ks = CPU_SAMPLE[cfg]
    npb, ks = min(npb, wl.batch), min(ks, wl.K)
    per_pi, total = cpu_oracle_time(wl, npb, ks)
    return dict(value=1.0 / (per_pi * wl.batch), unit=UNIT, cores=blas_threads(), kind="oracle",
                sample=f"{npb} of {wl.batch} problems x {ks} of {wl.K} unrolled iterations, fwd+bwd, {total:.1f} s; "
                       f"extrapolated x{wl.batch / npb:.0f} problems", host_cores=len(os.sched_getaffinity(0)))


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(cfg, 0, args.batch, args.unroll, args.p)
    npb, ks = CPU_SAMPLE[cfg]
    npb, ks = min(npb, wl.batch), min(ks, wl.K)
    for _ in range(args.warmup):
        cpu_oracle_time(wl, 1, min(ks, 3))
    t = []
    for _ in range(args.steps):
        per_pi, _ = cpu_oracle_time(wl, npb, ks)
        t.append(per_pi)
    per_pi = float(np.mean(t))
    ms_step = per_pi * wl.batch * wl.K * 1e3
    val = 1.0 / (per_pi * wl.batch)
    line = dict(metric=METRIC, value=val, unit=UNIT, impl="reference", n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic",
                config=dict(workload=wl.name, batch=wl.batch, K_unroll=wl.K, note="fp64 CPU oracle on a bounded sample, extrapolated to the batch"),
                cpu_baseline=dict(value=val, unit=UNIT, kind="oracle", cores=blas_threads(),
                                  sample=f"{npb} of {wl.batch} problems x {ks} of {wl.K} iterations per step"),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(WORKLOADS))
    ap.add_argument("--ckpt", default="full", choices=["full", "lean"])
    ap.add_argument("--batch", type=int, default=None, help="override the batch size (debug)")
    ap.add_argument("--unroll", type=int, default=None, help="override K_unroll (debug)")
    ap.add_argument("--p", type=int, default=None, help="override the graph order / n (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cg-refine", type=int, default=-2, help="-2: workload default (handle default: one refinement pass for fp32)")
    ap.add_argument("--cg-refine-tol", type=float, default=0.0)
    ap.add_argument("--tensor-cores", type=int, default=-1)
    ap.add_argument("--team-size", type=int, default=0, help="CTAs per problem in the linear step (0: automatic) (debug)")
    ap.add_argument("--no-batch", type=int, default=0, help="1: lane groups per row instead of warp row batches (debug)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = WORKLOADS[args.workload]
    if args.cg_refine == -2:
        args.cg_refine = -1
        if cfg == 3 and args.cg_refine_tol == 0.0:
            args.cg_refine_tol = 1e-2              # the parity-tested setting of cfg3 (tests/test_parity_gpu.py)
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist
    import paper_2606_13825_b200 as cdu

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    wl = make_workload(cfg, rank, args.batch, args.unroll, args.p)
    packed = W.pack_batch(wl.problems, wl.dtype)
    full = args.ckpt == "full"
    h = cdu.cdu_create(packed, K_max=wl.K, ckpt_mode=cdu.CDU_CKPT_FULL if full else cdu.CDU_CKPT_LEAN,
                       cg_refine=args.cg_refine, cg_refine_tol=args.cg_refine_tol, use_tensor_cores=args.tensor_cores,
                       no_batch=args.no_batch, team_size=args.team_size)
    tdt = torch.float32 if wl.dtype == "f32" else torch.float64
    N, M = h.N, h.M
    rng = np.random.default_rng(W.generators.BASE_SEED + 31337 + rank)
    host = dict(rho=wl.rho, alpha=wl.alpha, x0=np.concatenate(wl.x0), s0=np.concatenate(wl.s0), y0=np.concatenate(wl.y0),
                gx=rng.standard_normal(N), gs=rng.standard_normal(M), gy=rng.standard_normal(M))
    pin = {k: torch.as_tensor(v, dtype=tdt).pin_memory() for k, v in host.items()}
    dev = {k: v.cuda() for k, v in pin.items()}
    out_f = tuple(torch.empty(n, dtype=tdt, device="cuda") for n in (N, M, M))
    out_b = {k: torch.empty(n, dtype=tdt, device="cuda") for k, n in
             dict(g_rho=wl.K, g_alpha=wl.K, g_sigma=1, g_x0=N, g_s0=M, g_y0=M).items()}
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step_dev():
        h.forward(wl.K, dev["rho"], dev["alpha"], wl.sigma, dev["x0"], dev["s0"], dev["y0"], out=out_f)
        g = h.backward(dev["gx"], dev["gs"], dev["gy"], out=out_b)
        if world > 1:   # the one real exchange: hyper-parameters are shared by every rank's batch
            for k in ("g_rho", "g_alpha", "g_sigma"):
                dist.all_reduce(g[k])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        flush.fill_(1)
        step_dev()
    barrier()
    l0 = h.stats()["launches"]
    h.profile(True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    prof = {}
    barrier()
    for i in range(args.steps):
        flush.fill_(i)            # L2 flush between timed iterations (not inside the event pair)
        ev[i][0].record()
        step_dev()
        ev[i][1].record()
        ev[i][1].synchronize()
        for k, v in h.get_profile().items():
            a = prof.setdefault(k, dict(ms=0.0, launches=0))
            a["ms"] += v["ms"]; a["launches"] += v["launches"]
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    h.profile(False)
    st = h.stats()
    launches = st["launches"] - l0
    ms = float(sum(a.elapsed_time(b) for a, b in ev))
    if world > 1:
        t = torch.tensor([ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    ms_step = ms / args.steps
    value = wl.K * world / (ms_step * 1e-3)

    # ---- end-to-end through the C ABI with HOST buffers (copies inside the timed region) ------------------------
    e2e = None
    if not args.no_e2e:
        hout_f = tuple(torch.empty(n, dtype=tdt).pin_memory() for n in (N, M, M))
        hout_b = {k: torch.empty(n, dtype=tdt).pin_memory() for k, n in
                  dict(g_rho=wl.K, g_alpha=wl.K, g_sigma=1, g_x0=N, g_s0=M, g_y0=M).items()}

        def step_host():
            h.forward(wl.K, pin["rho"], pin["alpha"], wl.sigma, pin["x0"], pin["s0"], pin["y0"], out=hout_f, host=True)
            h.backward(pin["gx"], pin["gs"], pin["gy"], out=hout_b, host=True)
            if world > 1:
                for k in ("g_rho", "g_alpha", "g_sigma"):
                    t_ = hout_b[k].cuda(non_blocking=True); dist.all_reduce(t_); hout_b[k].copy_(t_)

        step_host()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nst = max(1, min(args.steps, 3))
        tot = 0.0
        for i in range(nst):
            flush.fill_(i)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e0.record(); step_host(); e1.record(); e1.synchronize()
            tot += max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3)
        if world > 1:
            t = torch.tensor([tot], device="cuda", dtype=torch.float64); dist.all_reduce(t, op=dist.ReduceOp.MAX); tot = float(t.item())
        esz = 4 if wl.dtype == "f32" else 8
        e2e = dict(value=wl.K * world / (tot / nst * 1e-3), unit=UNIT,
                   h2d_bytes_per_step=esz * (2 * wl.K + 2 * (N + 2 * M)), d2h_bytes_per_step=esz * (2 * wl.K + 1 + 2 * (N + 2 * M)),
                   note="problem data resident in the handle (the paper trains for 100 epochs on a fixed set of instances, "
                        "L289-291); per step: theta, z0, cotangent in; z_K and all gradients out")

    # ---- roofline of the dominant kernel class ---------------------------------------------------------------
    peaks = load_peaks()
    dom = max(prof, key=lambda k: prof[k]["ms"]) if prof else None
    roof = None
    if dom and prof[dom]["launches"]:
        dur = prof[dom]["ms"] * 1e-3 / prof[dom]["launches"]          # average launch duration, seconds
        nsolve = wl.batch * wl.K
        ncg_f = st["cg_iters_fwd"] / nsolve
        ncg_b = st["cg_iters_bwd"] / nsolve
        share = prof[dom]["ms"] / ms
        if dom in ("lin_fwd", "lin_bwd"):
            bf, bb = lin_bytes(wl, ncg_f, ncg_b, full)
            nb = bf if dom == "lin_fwd" else bb
            if dom == "lin_bwd" and psd_orders(wl):
                nb = nb / 2.0   # two launches (pre / post) per iteration share the bytes
            ach = nb / dur / 1e9
            roof = dict(kernel=dom, bound="hbm", achieved=ach, peak=peaks["hbm_gbs"], unit="GB/s", frac=ach / peaks["hbm_gbs"],
                        traffic=None, peak_source=peaks["source"], frac_of_8TBs=ach / 8000.0,
                        cg_iters_per_solve=dict(fwd=ncg_f, bwd=ncg_b))
        elif dom in ("psd_fwd_small", "psd_bwd_small"):
            ps = psd_orders(wl)
            if dom == "psd_fwd_small":
                fl = jacobi_flops(ps, st["eig_sweeps_sum"] / wl.K)
            else:
                fl = 8.0 * float(np.sum([p ** 3 for p in ps])) + (0.0 if full else jacobi_flops(ps, st["eig_sweeps_sum"] / wl.K))
            pk = FP32_ALU_PEAK_TFLOPS if wl.dtype == "f32" else FP64_ALU_PEAK_TFLOPS
            ach = fl / dur / 1e12
            roof = dict(kernel=dom, bound="alu", achieved=ach, peak=pk, unit="TFLOP/s", frac=ach / pk, traffic=None,
                        peak_source="derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md)",
                        sweeps_per_matrix=st["eig_sweeps_sum"] / max(1, wl.K * len(ps)))
        elif dom == "gemm_large":
            ps = psd_orders(wl)
            fl = 2.0 * float(np.sum([p ** 3 for p in ps]))
            pk = peaks["bf16_sustained"] * 0.5    # TF32 = bf16 x nominal ratio 1.1/2.25 (guide)
            ach = fl / dur / 1e12
            roof = dict(kernel=dom, bound="tensor", achieved=ach, peak=pk, unit="TFLOP/s", frac=ach / pk, traffic=None,
                        peak_source=peaks["source"] + " bf16 sustained x 0.5 (tf32 nominal ratio)")
        else:   # eig_large: latency/L2-bound Jacobi; report executed FMA flops against the fp32 ALU peak
            ps = psd_orders(wl)
            fl = float(np.mean([8.0 * (1.0 - 16.0 / p) * p ** 3 for p in ps])) * st["eig_sweeps_sum"] / wl.K
            ach = fl / dur / 1e12
            roof = dict(kernel=dom, bound="alu", achieved=ach, peak=FP32_ALU_PEAK_TFLOPS, unit="TFLOP/s",
                        frac=ach / FP32_ALU_PEAK_TFLOPS, traffic=None,
                        peak_source="derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md)",
                        note="blocked one-sided Jacobi: Gram + apply products, 8 (1 - 16/p) p^3 flops per sweep as if every pair rotated; "
                             "bound by the latency of the 32 x 32 inner sweeps (DESIGN.md)")
        roof["share_of_step"] = share
        roof["avg_launch_ms"] = dur * 1e3
        tr = os.path.join(ROOT, "profiles", f"traffic_{args.workload}.json")
        if os.path.exists(tr):
            try:
                with open(tr) as f:
                    roof["traffic"] = json.load(f).get(dom)
            except Exception:
                pass

    if rank == 0:
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=ms_step,
                    higher_is_better=True, scaling="weak", vs_baseline=None, dtype=wl.dtype, data="synthetic",
                    config=dict(workload=wl.name, batch_per_gpu=wl.batch, K_unroll=wl.K, checkpoint=args.ckpt,
                                l2="flushed between timed steps (256 MiB write)", state="fp64", cg_refine=args.cg_refine, cg_refine_tol=args.cg_refine_tol,
                                parallelism=f"batch-sharded x{world}, all-reduce of 2K+1 shared-theta gradients" if world > 1 else "single GPU"),
                    problem_iters_per_s=value * wl.batch, problems_per_s=value * wl.batch / wl.K,
                    device_mem_mb=st["device_bytes"] / 2 ** 20, ckpt_mem_mb=st["ckpt_bytes"] / 2 ** 20,
                    cg_iters_per_solve=dict(fwd=st["cg_iters_fwd"] / (wl.batch * wl.K), bwd=st["cg_iters_bwd"] / (wl.batch * wl.K), max=st["cg_iters_max"]),
                    eig_sweeps_max=st["eig_sweeps_max"], flags=st["flags_or"],
                    gpu_launches=int(launches), clocks=clocks, e2e=e2e, roofline=roof,
                    kernel_ms_per_step={k: v["ms"] / args.steps for k, v in prof.items() if v["launches"]})
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(wl, cfg)
        print(json.dumps(line))
    h.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
