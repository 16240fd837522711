#!/usr/bin/env python
"""bench.py -- B200 benchmark of the MSPCG hot path (BASELINE.json configs[1] = "C2", operator-only benchmark).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C2] [--no-extras]

One "step" = one pass of the whole hot path over one batch of synthetic input = the operator work of one outer MSPCG
iteration on the C2 lattice (16^3 x 32, Ls 16, 8^4 Dirichlet blocks):
    one multi-splitting preconditioner application  z = M^-1 r  (6 inner CG iterations, fp16 storage / fp32
    arithmetic, all 32 blocks batched)  +  one full-lattice D^dag D application in the sloppy
    outer precision fp32 (A2-A6),
both on NATIVE-layout vectors already resident in HBM.  value = GFLOP/s with the flop convention of SURVEY 8(d)
(hop 1320, bidiagonal 5D op 72, xpay 48, dense 5D contraction 48*Ls per 5D site; halo-shell sites count as work).
The JSON line also carries: e2e (same step through the C-ABI *_host calls, host<->device copies in the timed
region), roofline (dominant kernel, algorithmic bytes / CUDA-event time vs the measured HBM peak), cpu_baseline (the
CPU oracle on a bounded sample), clocks, and "extras" (per-precision operator numbers, CG vs MSPCG time-to-solution).

Multi-GPU: the path does not shard (BASELINE.json: one GPU, no collectives) -> replicas only: under torchrun every
rank runs the same workload on its own GPU, no data-path collective, value = sum over ranks / max time ("weak").
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

from paper_2104_05615_b200 import synth  # noqa: E402

METRIC = "mspcg_precond_dslash_step_gflops"
UNIT = "GFLOP/s"


# ------------------------------------------------------------------------------------------------ work models
def stage_sites(geo, full):
    """4D sites per block on which each of the five kernels of eq. 16 writes: (K1, K2, K3, K4, K5)."""
    if full:
        v = geo["vh"]
        return dict(nblk=1, nE0=v, nO=v, nE=v)
    return dict(nblk=geo["nblk"], nE0=geo["nE0"], nO=geo["nO1"], nE=geo["nE2"])


def flops_normal(st, Ls, executed=False):
    """Flops of one D^dag D (or A_s, all blocks) application; SURVEY 8(d) convention.  executed=True: what the library runs --
    on the halo sites of a Dirichlet block kernel 3 applies the product matrix M5^-dag M5^-1 as ONE contraction and has no
    xpay operand, so one contraction and the xpay are not executed there."""
    hop, bid, xpay, dense = 1320, 72, 48, 48 * Ls
    per_block = (bid * st["nE0"] + (hop + dense) * st["nO"] + (hop + 2 * dense + xpay) * st["nE"]
                 + (hop + dense) * st["nO"] + (hop + bid + xpay) * st["nE0"]) * Ls
    if executed:
        per_block -= (dense + xpay) * (st["nE"] - st["nE0"]) * Ls
    return per_block * st["nblk"]


def bytes_normal(st, Ls, w, ng, fused_pupdate=False, with_dot=False):
    """Algorithmic HBM bytes per kernel class of one D^dag D application: every input site, output site and link read
    or written exactly once per kernel (ideal neighbour reuse).  Returns dict class -> bytes per launch."""
    site = Ls * 24 * w
    link = 8 * ng * w
    n = st["nblk"]
    k1 = (4 if fused_pupdate else 2) * st["nE0"] * site
    k2 = (st["nE0"] + st["nO"]) * site + st["nO"] * link
    k3 = (st["nO"] + st["nE0"] + st["nE"] + st["nE0"]) * site + st["nE"] * link
    k4 = (st["nE"] + st["nO"]) * site + st["nO"] * link
    k5 = (st["nO"] + st["nE0"] + (st["nE0"] if with_dot else 0) + st["nE0"]) * site + st["nE0"] * link
    return dict(mphi=k1 * n, hop_k2=k2 * n, hop_k3=k3 * n, hop_k4=k4 * n, hop_k5=k5 * n)


def precond_work(geo, Ls, k, w_in, w_io, ng, executed=False):
    """Flops and algorithmic bytes of one M^-1 application (k inner iterations)."""
    st = stage_sites(geo, False)
    fl = k * flops_normal(st, Ls, executed)
    by = 0
    for it in range(k):
        b = bytes_normal(st, Ls, w_in, ng, fused_pupdate=it > 0, with_dot=True)
        if it == 0:
            b["mphi"] = 3 * st["nE0"] * Ls * 24 * w_in * st["nblk"]
        by += sum(b.values())
        v = st["nE0"] * Ls * 24 * st["nblk"]
        wx = 4 if w_in == 2 else w_in
        by += v * (3 * w_in + 2 * wx + 2 * w_in) if it < k - 1 else v * (w_in + wx + w_io)   # x,r update / final z
    by += st["nE0"] * Ls * 24 * st["nblk"] * (w_io * (2 if w_in == 2 else 1) + w_in)         # max-abs + scaled copy
    return fl, by


# ------------------------------------------------------------------------------------------------ clocks sampler
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except Exception:
                continue
            for nme, val in zip(names, r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    power_w_max=max(pw) if pw else None, samples=len(sm), reasons=sorted(reasons))


# ------------------------------------------------------------------------------------------------ workload set-up
def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic():
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture, if any."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    return json.load(open(p)) if os.path.exists(p) else {}


def initial_T_abi(Ls, Lh):
    """Untrained transfer matrix (reading R20): spin identity, keeps the Lh/2 slices next to each domain wall.
    float64 [4*Lh][4*Ls][re,im] as include/mspcg.h asks."""
    T = np.zeros((Lh, 4, Ls, 4, 2))
    for a in range(Lh):
        s = a if a < Lh // 2 else Ls - Lh + a
        for m in range(4):
            T[a, m, s, m, 0] = 1.0
    return T.reshape(-1)


def make_inputs(cfg):
    dims, Ls = cfg["dims"], cfg["Ls"]
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, cfg["eps"], cfg["gauge_seed"]), dims)
    src = synth.gaussian_spinor_abi(dims, Ls, cfg["src_seed"])
    return U, src


def timed(torch, fn, steps, warmup, barrier=None):
    """W warm-up calls, then exactly K calls between CUDA events on the current stream; returns ms total."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    return e0.elapsed_time(e1)


def max_over_ranks(ms, world, device):
    """Replicas only: the only cross-rank step is the max of the device-timed region."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(flops_step, ms_step, world):
    """Whole-job throughput of N independent replicas: N x (work of one replica) / (slowest replica's time)."""
    return world * flops_step / (ms_step * 1e-3) / 1e9


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2104_05615_b200 import F16, F32, F64, LAYOUT_NATIVE, Mspcg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    barrier = None
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        barrier = dist.barrier
    cfg = dict(synth.CONFIGS[args.workload])
    if args.block:
        cfg["block"] = tuple(int(x) for x in args.block.split(","))
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    U, src = make_inputs(cfg)
    g = Mspcg(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    if args.reduced:   # profiling aid: the step's preconditioner becomes the reduced-Ls one (untrained T, eq. 20-21)
        g.set_reduced_ls(args.reduced, initial_T_abi(Ls, args.reduced), 0.5)
    ws = g.configure(F32, F16, args.recon)
    g.set_block_group(args.group)
    g.load_gauge(U, -1)
    geo = g.geometry()
    d_src = torch.as_tensor(src.reshape(-1)).cuda()
    r32 = g.pack(d_src, F32)
    big = ws > 100 * 2**30      # largest instance: no room for the fp64 ABI copies of the end-to-end leg
    if big:
        del d_src
        torch.cuda.empty_cache()
    z32, q32 = g.new_native(F32), g.new_native(F32)

    def step():
        g.apply_precond(r32, k, F32, LAYOUT_NATIVE, out=z32, use_reduced=1 if args.reduced else 0)
        g.apply_MdagM(r32, F32, LAYOUT_NATIVE, out=q32)

    # ---- work model of one step
    fl_pre, by_pre = precond_work(geo, Ls, k, 2, 4, args.recon)
    st_full = stage_sites(geo, True)
    fl_op = flops_normal(st_full, Ls)
    by_op = sum(bytes_normal(st_full, Ls, 4, args.recon).values())
    flops_step = fl_pre + fl_op
    flops_exec = precond_work(geo, Ls, k, 2, 4, args.recon, executed=True)[0] + fl_op

    # ---- the timed region (device-resident inputs)
    sampler = ClockSampler(local)
    sampler.start()
    n0 = g.launch_count()
    ms = timed(torch, step, args.steps, args.warmup, barrier)
    launches = (g.launch_count() - n0) // (args.steps + args.warmup) * args.steps
    clocks = sampler.stop()
    ms = max_over_ranks(ms, world, "cuda")
    ms_step = ms / args.steps
    value = aggregate_value(flops_step, ms_step, world)

    # ---- end to end: same step through the *_host entry points, pinned host buffers, copies inside the timed region
    if big:
        ms_e2e = float("nan")
    else:
        # the step's vectors are fp32 (sloppy outer precision): single-precision host buffers in the ABI layout (mspcg_apply_*_host32)
        h_in = torch.as_tensor(src.reshape(-1).astype(np.float32)).pin_memory()
        h_z, h_q = torch.empty_like(h_in).pin_memory(), torch.empty_like(h_in).pin_memory()

        def step_host():
            g.apply_precond_host32(h_in, h_z, k, F32)
            g.apply_MdagM_host32(h_in, h_q, F32)

        e2e_steps = max(2, min(args.steps, 5))
        ms_e2e = timed(torch, step_host, e2e_steps, 1, barrier) / e2e_steps
        h64 = torch.as_tensor(src.reshape(-1)).pin_memory()      # the fp64 wire format of the ABI, for comparison
        h64z, h64q = torch.empty_like(h64).pin_memory(), torch.empty_like(h64).pin_memory()

        def step_host64():
            g.apply_precond_host(h64, h64z, k, F32)
            g.apply_MdagM_host(h64, h64q, F32)
        ms_e2e64 = timed(torch, step_host64, 2, 1, barrier) / 2
    ms_e2e = max_over_ranks(ms_e2e, world, "cuda")
    nb = src.size * 4
    e2e = dict(value=world * flops_step / (ms_e2e * 1e-3) / 1e9, unit=UNIT, ms_per_step=ms_e2e,
               h2d_bytes_per_step=2 * nb, d2h_bytes_per_step=2 * nb, host_dtype="f32 (mspcg_apply_*_host32)",
               ms_per_step_f64_host_buffers=None if big else ms_e2e64)
    if big:
        e2e = dict(value=None, unit=UNIT, skipped="workspace > 100 GiB: no device room for the fp64 ABI staging of the host leg",
                   h2d_bytes_per_step=0, d2h_bytes_per_step=0)

    # ---- roofline of the dominant kernel: instrumented repetition of the same steps (CUDA events per launch)
    peak, peak_src = peaks()
    g.timing(True)
    for _ in range(args.steps):
        step()
    tm = g.timing_read()
    g.timing(False)
    st_blk = stage_sites(geo, False)
    bb = bytes_normal(st_blk, Ls, 2, args.recon, fused_pupdate=True, with_dot=True)
    bf = bytes_normal(st_full, Ls, 4, args.recon)
    alg = {"blk.hop_k2k4": 0.5 * (bb["hop_k2"] + bb["hop_k4"]), "blk.hop_k3": bb["hop_k3"], "blk.hop_k5": bb["hop_k5"],
           "blk.mphi": bb["mphi"], "full.hop_k2k4": 0.5 * (bf["hop_k2"] + bf["hop_k4"]), "full.hop_k3": bf["hop_k3"],
           "full.hop_k5": bf["hop_k5"], "full.mphi": bf["mphi"]}
    if args.group and args.group < geo["nblk"]:   # a launch covers one group of blocks only
        ngroups = -(-geo["nblk"] // args.group)
        alg = {n: (b / ngroups if n.startswith("blk.") else b) for n, b in alg.items()}
    kern = {}
    tot_ms = sum(v["ms"] for v in tm.values())
    for name, v in tm.items():
        if v["launches"] == 0:
            continue
        avg = v["ms"] / v["launches"]
        ent = dict(launches_per_step=v["launches"] / args.steps, avg_ms=avg, share=v["ms"] / tot_ms)
        if name in alg:
            ent["alg_bytes"] = alg[name]
            ent["GBps"] = alg[name] / (avg * 1e-3) / 1e9
            ent["frac"] = ent["GBps"] / peak
        kern[name] = ent
    dom = max((n for n in kern if n in alg), key=lambda n: tm[n]["ms"])
    prof = ncu_traffic()
    traffic = prof.get(dom)
    roofline = dict(bound="hbm", kernel=dom, achieved=kern[dom]["GBps"], peak=peak, unit="GB/s", frac=kern[dom]["frac"],
                    traffic=traffic, peak_source=peak_src, alg_bytes_per_launch=kern[dom]["alg_bytes"],
                    avg_launch_ms=kern[dom]["avg_ms"], share_of_step=kern[dom]["share"],
                    # utilisation of the tensor pipe by the SU(3) and M5^-1 contractions of this kernel, from the committed
                    # ncu --set full capture (profiles/traffic.json), not measured in this run
                    tensor_pipe_pct_ncu=(prof.get("tensor_pipe_pct") or {}).get(dom))

    out = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
               ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f16/f32",
               data="synthetic", impl="ours",
               config=dict(workload=f"{args.workload}: {dims[0]}x{dims[1]}x{dims[2]}x{dims[3]} Ls={Ls} blocks {block} "
                                    f"M_pre(k={k}, fp16 storage/fp32 math) + DdagD(fp32)" + (f" [reduced-Ls {args.reduced}: flop model of the full-Ls step, not a headline]" if args.reduced else ""),
                           parallelism="replicas only", block_group=args.group,
                           l2="working set of a step %.0f MiB > 126 MB L2 (no flush)" % (ws / 2**20), workspace_bytes=ws,
                           flops_per_step=flops_step, flops_executed_per_step=flops_exec, alg_bytes_per_step=by_pre + by_op),
               value_flops_executed=aggregate_value(flops_exec, ms_step, world),
               gpu_launches=launches, clocks=clocks, e2e=e2e, roofline=roofline, kernels=kern,
               step_GBps_algorithmic=(by_pre + by_op) / (ms_step * 1e-3) / 1e9)
    if rank == 0 and world == 1 and not args.no_extras and not big:
        out["extras"] = extras(torch, g, cfg, U, src, d_src, geo, peak, args)
        out["cpu_baseline"] = cpu_baseline(cfg, U, src, geo, args.workload)
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def extras(torch, g, cfg, U, src, d_src, geo, peak, args):
    """Per-precision operator numbers (C2: "in fp16 storage with fp32 accumulation and in fp64") and CG vs MSPCG
    time-to-solution on the same lattice.  Outside the headline timed region."""
    from paper_2104_05615_b200 import F16, F32, F64, LAYOUT_NATIVE, Mspcg
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    st_full = stage_sites(geo, True)
    ex = {}
    steps, warm = max(3, args.steps), 3

    def op_entry(ms, flops, nbytes):
        return dict(ms=ms, GFLOPs=flops / (ms * 1e-3) / 1e9, GBps_algorithmic=nbytes / (ms * 1e-3) / 1e9,
                    hbm_frac=nbytes / (ms * 1e-3) / 1e9 / peak)

    def time_op(ctx, prec, w):
        v, o = ctx.pack(d_src, prec), ctx.new_native(prec)
        ms = timed(torch, lambda: ctx.apply_MdagM(v, prec, LAYOUT_NATIVE, out=o), steps, warm) / steps
        return op_entry(ms, flops_normal(st_full, Ls), sum(bytes_normal(st_full, Ls, w, 18).values()))

    def time_pre(ctx, io, w_in, w_io):
        v, o = ctx.pack(d_src, io), ctx.new_native(io)
        ms = timed(torch, lambda: ctx.apply_precond(v, k, io, LAYOUT_NATIVE, out=o), steps, warm) / steps
        fl, by = precond_work(geo, Ls, k, w_in, w_io, 18)
        return op_entry(ms, fl, by)

    ex["DdagD_fp64"] = time_op(g, F64, 8)
    ex["DdagD_fp32"] = time_op(g, F32, 4)
    ex["Mpre_k%d_fp16_io32" % k] = time_pre(g, F32, 2, 4)
    # time to solution, plain CG vs MSPCG, sloppy fp32 + fp64 reliable updates, preconditioner fp16
    sol = {}
    for name, pre in (("CG", False), ("MSPCG", True)):
        x, s = g.solve(d_src, tol=1e-10, max_iter=200000, use_precond=pre, n_inner=k, sloppy_prec=F32, delta=0.1)
        sol[name] = solve_entry(s)
    ex["solve_tol1e-10_fp32outer_fp16inner"] = sol
    del x
    g.close()
    torch.cuda.empty_cache()
    # reduced-Ls preconditioner: T trained with the library (eq. 22; set-up step, its time reported, not
    # part of the solve) on residual vectors of a full-Ls MSPCG run, then MSPCG with z = T^dag CG_k[Mhat](T r) + mu r
    # T is the identity in 4D site and colour (eq. 21), so it is trained on a sample lattice of at most 16^3 x 32 sites with the same
    # Moebius parameters, mass and link roughness (its own seeds) and Dirichlet blocks of at most half its extent, and then
    # used on the full lattice -- the paper likewise trains once per ensemble.
    Lh, mu = cfg.get("Ls_hat", Ls // 2), args.mu
    T, info, train_s, tdims, tblock = train_T_on_sample(torch, cfg, U, src, args)
    gr = Mspcg(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    gr.set_reduced_ls(Lh, T, mu)
    gr.configure(F32, F16, 18)
    gr.load_gauge(U, -1)
    v, o = gr.pack(d_src, F32), gr.new_native(F32)
    ms = timed(torch, lambda: gr.apply_precond(v, k, F32, LAYOUT_NATIVE, out=o, use_reduced=1), steps, warm) / steps
    x, s = gr.solve(d_src, tol=1e-10, max_iter=200000, use_precond=True, n_inner=k, sloppy_prec=F32, delta=0.1, use_reduced_ls=True)
    ex["reducedLs%d_trainedT_mu%.2f" % (Lh, mu)] = dict(
        Mpre_ms=ms, train_seconds=train_s, train_steps=args.train_steps, train_lattice=list(tdims), train_block=list(tblock), chi2_first=float(info["chi2"][0]), chi2_last=float(info["chi2"][-1]),
        solve=solve_entry(s))
    del x, v, o
    gr.close()
    torch.cuda.empty_cache()
    g2 = Mspcg(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    g2.configure(F16, F64, 18)
    g2.load_gauge(U, -1)
    ex["DdagD_fp16"] = time_op(g2, F16, 2)
    if Ls in (8, 12, 16):
        ex["M5inv_tcgen05_fp16"] = time_m5inv(torch, g2, d_src, Ls, steps, warm, peak)
    ex["Mpre_k%d_fp64" % k] = time_pre(g2, F64, 8, 8)
    g2.close()
    torch.cuda.empty_cache()
    # the same solves with an fp16 sloppy outer iteration (vectors rescaled at every residual replacement)
    g3 = Mspcg(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    g3.configure(F16, F16, 18)
    g3.load_gauge(U, -1)
    sol = {}
    cap = 3 * ex["solve_tol1e-10_fp32outer_fp16inner"]["CG"]["outer_iters"]   # plain fp16 CG can stagnate on ill-conditioned systems (rc = ENOCONV then)
    for name, pre in (("CG", False), ("MSPCG", True)):
        x, s = g3.solve(d_src, tol=1e-10, max_iter=cap, use_precond=pre, n_inner=k, sloppy_prec=F16, delta=0.1)
        sol[name] = solve_entry(s)
    ex["solve_tol1e-10_fp16outer_fp16inner"] = sol
    del x
    g3.close()
    return ex


def train_T_on_sample(torch, cfg, U, src, args):
    """T of the reduced-Ls preconditioner (eq. 21) trained with the library (eq. 22) on a sample lattice of at most 16^3 x 32 sites with the
    configuration's parameters (its own seeds; Dirichlet blocks at most half its extent); T is site and colour independent (R20)."""
    from paper_2104_05615_b200.train_reduced_ls import train
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    Lh, mu = cfg.get("Ls_hat", Ls // 2), args.mu
    tdims = tuple(min(d, 16 if i < 3 else 32) for i, d in enumerate(dims))
    tblock = tuple(min(b, t // 2) if b < d else t for b, t, d in zip(block, tdims, dims))
    if tdims == tuple(dims):
        U_t, src_t, tblock = U, src, block
    else:
        U_t = synth.gauge_natural_to_abi(synth.random_su3_links(tdims, cfg["eps"], cfg["gauge_seed"] + 100), tdims)
        src_t = synth.gaussian_spinor_abi(tdims, Ls, cfg["src_seed"] + 100)
    t0 = time.time()
    T, info = train(tdims, Ls, dict(b=cfg["b"], c=cfg["c"], M5=cfg["M5"]), cfg["mf"], tblock, U_t, src_t, Lh, mu, k,
                    n_vec=12, span=120, n_steps=args.train_steps, momentum=0.5)
    torch.cuda.synchronize()
    return T, info, time.time() - t0, tdims, tblock


def solve_entry(s):
    return dict(seconds=s["seconds"], outer_iters=s["iters"], reliable_updates=s["reliable_updates"],
                inner_applies=s["inner_applies"], outer_applies=s["outer_applies"], true_res=s["true_res"], rc=s["rc"])


def run_solves(args):
    """Time to solution on one GPU (BASELINE.json metric, Tables 3-4): plain CG, MSPCG and MSPCG with the reduced-Ls
    preconditioner on the workload, sloppy outer precision --sloppy (fp32 or fp16) with fp64 residual replacement, fp16 preconditioner, 1e-10."""
    import torch
    from paper_2104_05615_b200 import F16, F32, Mspcg
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    cfg = dict(synth.CONFIGS[args.workload])
    if args.block:
        cfg["block"] = tuple(int(x) for x in args.block.split(","))
    if args.n_inner:
        cfg["n_inner"] = args.n_inner
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    sloppy = F16 if args.sloppy == 16 else F32
    U, src = make_inputs(cfg)
    out = dict(impl="ours", mode="solves", workload=args.workload, lattice=list(dims), Ls=Ls, block=list(block), n_inner=k, mf=cfg["mf"],
               sloppy_bits=args.sloppy, recon=args.recon, tol=1e-10, solves={})
    Lh = cfg.get("Ls_hat", Ls // 2)
    T = None
    if args.reduced_solve:
        T, info, train_s, tdims, tblock = train_T_on_sample(torch, cfg, U, src, args)
        out["reduced"] = dict(Ls_hat=Lh, mu=args.mu, train_seconds=train_s, train_steps=args.train_steps, train_lattice=list(tdims),
                              train_block=list(tblock), chi2_first=float(info["chi2"][0]), chi2_last=float(info["chi2"][-1]))
    g = Mspcg(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    if T is not None:
        g.set_reduced_ls(Lh, T, args.mu)
    out["workspace_bytes"] = g.configure(sloppy, F16, args.recon)
    g.set_block_group(args.group)
    out["block_group"] = args.group
    g.load_gauge(U, -1)
    del U
    d_src = torch.as_tensor(src.reshape(-1)).cuda()
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))
    sampler.start()
    cap = args.max_iter
    for name, kw in (("CG", dict(use_precond=False)), ("MSPCG", dict(use_precond=True, n_inner=k)),
                     ("MSPCG_reducedLs", dict(use_precond=True, n_inner=k, use_reduced_ls=True))):
        if name == "MSPCG_reducedLs" and T is None:
            continue
        x, st = g.solve(d_src, tol=1e-10, max_iter=cap, sloppy_prec=sloppy, delta=0.1, **kw)
        del x
        out["solves"][name] = solve_entry(st)
    out["clocks"] = sampler.stop()
    print(json.dumps(out))


def time_m5inv(torch, g, d_src, Ls, steps, warm, peak):
    """The dense 5D contraction M5^-1 on its own as a tcgen05 GEMM (mspcg_apply_M5inv): four buffer pairs in rotation (one fp16
    vector pair is smaller than L2); flops by the minimal count 48*Ls per 5D site and as issued (8x: the delta_jj' zeros of the B operand)."""
    from paper_2104_05615_b200 import F16
    ins = [g.pack(d_src, F16) for _ in range(4)]
    outs = [g.new_native(F16) for _ in range(4)]
    cnt = [0]

    def m5():
        g.apply_M5inv(ins[cnt[0] & 3], False, out=outs[cnt[0] & 3])
        cnt[0] += 1
    ms = timed(torch, m5, 4 * steps, 4 * warm) / (4 * steps)
    n5 = ins[0].numel() * ins[0].element_size() // 48
    nbytes, flops = 2.0 * 48 * n5, 48.0 * Ls * n5
    return dict(ms=ms, GFLOPs=flops / (ms * 1e-3) / 1e9, GBps_algorithmic=nbytes / (ms * 1e-3) / 1e9, hbm_frac=nbytes / (ms * 1e-3) / 1e9 / peak,
                GFLOPs_issued_on_tensor_cores=8 * flops / (ms * 1e-3) / 1e9,
                note="tcgen05.mma kind::f16, fp32 accumulation in TMEM, operands and results moved by tensor-map TMA; 4 buffer pairs rotated")


def run_m5inv(args):
    import torch
    from paper_2104_05615_b200 import F16, Mspcg
    cfg = synth.CONFIGS[args.workload]
    g = Mspcg(cfg["dims"], cfg["Ls"], cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], cfg["block"])
    g.configure(F16, F16, 18)
    d_src = torch.as_tensor(synth.gaussian_spinor_abi(cfg["dims"], cfg["Ls"], cfg["src_seed"]).reshape(-1)).cuda()
    print(json.dumps(dict(impl="ours", mode="m5inv", workload=args.workload, M5inv_tcgen05_fp16=time_m5inv(torch, g, d_src, cfg["Ls"], max(3, args.steps), 3, peaks()[0]))))


def oracle_sample(cfg, U, src, geo):
    """The bounded CPU sample: the oracle's M^-1 on ONE Dirichlet block (k inner iterations) + one full-lattice
    D^dag D, fp64, plain C with OpenMP over sites.  Returns (callable running one sample, flops of the sample, ora)."""
    from oracle.cbind import OracleC
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    ora = OracleC(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    ora.load_gauge(U, -1)
    fl_pre, _ = precond_work(geo, Ls, k, 8, 8, 18)
    flops = fl_pre / geo["nblk"] + flops_normal(stage_sites(geo, True), Ls)

    def run():
        ora.apply_precond(src, k, only_block=0)
        ora.apply_MdagM(src)
    return run, flops, ora


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(cfg, U, src, geo, workload):
    """The oracle as it stands on the host cores: the bounded sample on all cores and on one core (a second process with
    OMP_NUM_THREADS=1), and full CG / MSPCG time-to-solution on C1."""
    run, flops, ora = oracle_sample(cfg, U, src, geo)
    t0 = time.time()
    run()
    dt = time.time() - t0
    out = dict(value=flops / dt / 1e9, unit=UNIT, cores=ora.threads, kind="oracle", seconds=dt, cpu_model=cpu_model(),
               sample="oracle M_pre on 1 of %d blocks (k=%d) + 1 full-lattice DdagD, fp64, same lattice" % (geo["nblk"], cfg["n_inner"]))
    try:   # one core: the same sample in a fresh process (the OpenMP thread count is fixed at library load)
        env = dict(os.environ, OMP_NUM_THREADS="1")
        res = subprocess.run([sys.executable, os.path.abspath(__file__), "--impl", "reference", "--steps", "1", "--warmup", "0",
                              "--workload", workload], env=env, capture_output=True, text=True, timeout=600)
        one = json.loads(res.stdout.strip().splitlines()[-1])
        out["value_1core"] = one["value"]
        out["seconds_1core"] = one["ms_per_step"] * 1e-3
    except Exception as e:   # noqa: BLE001
        out["value_1core"] = None
        out["note_1core"] = "one-core run failed: %r" % (e,)
    out["C1_time_to_solution"] = oracle_solves("C1")
    return out


def oracle_solves(workload):
    """Full CG and MSPCG solves to 1e-10 on the CPU oracle (fp64 throughout): seconds, outer iterations, inner applications."""
    from oracle.cbind import OracleC
    cfg = synth.CONFIGS[workload]
    U, src = make_inputs(cfg)
    ora = OracleC(cfg["dims"], cfg["Ls"], cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], cfg["block"])
    ora.load_gauge(U, -1)
    res = dict(lattice=list(cfg["dims"]), Ls=cfg["Ls"], block=list(cfg["block"]), n_inner=cfg["n_inner"], cores=ora.threads)
    for name, pre in (("CG", False), ("MSPCG", True)):
        t0 = time.time()
        _, st = ora.solve(src, tol=1e-10, use_precond=pre, n_inner=cfg["n_inner"])
        res[name] = dict(seconds=time.time() - t0, outer_iters=st["iters"], inner_applies=st["inner_applies"], true_res=st["true_res"], rc=st["rc"])
    return res


def host_geometry(cfg):
    """Site counts of the stage lists of one Dirichlet block (pad of two, L1 overshoot d; even d<=2, odd d<=1),
    counted here with numpy so that the oracle arm loads nothing of the product library."""
    dims, block = cfg["dims"], cfg["block"]
    cut = [b != l for b, l in zip(block, dims)]
    axes = [np.arange(-2, b + 2) if c else np.arange(0, b) for b, c in zip(block, cut)]
    X = np.meshgrid(*axes, indexing="ij")
    d = sum(((-x).clip(0) + (x - (b - 1)).clip(0)) if c else 0 * x for x, b, c in zip(X, block, cut))
    par = sum(X) % 2
    nblk = int(np.prod([l // b for l, b in zip(dims, block)]))
    return dict(nblk=nblk, nE0=int(((par == 0) & (d == 0)).sum()), nE2=int(((par == 0) & (d <= 2)).sum()),
                nO1=int(((par == 1) & (d <= 1)).sum()), vh=int(np.prod(dims)) // 2)


def run_reference(args):
    """The reference arm of this tier is the CPU oracle, as it stands, on the box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if args.cpu_solves:   # full oracle solves on a lattice that finishes in minutes
        print(json.dumps(dict(impl="reference", cpu_model=cpu_model(), time_to_solution=oracle_solves(args.cpu_solves))))
        return
    cfg = synth.CONFIGS[args.workload]
    U, src = make_inputs(cfg)
    geo = host_geometry(cfg)
    run, flops, ora = oracle_sample(cfg, U, src, geo)
    for _ in range(args.warmup):
        run()
    t0 = time.time()
    for _ in range(args.steps):
        run()
    dt = (time.time() - t0) / args.steps
    val = flops / dt / 1e9
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    sample = "oracle M_pre on 1 of %d blocks (k=%d) + 1 full-lattice DdagD per step, fp64" % (geo["nblk"], k)
    print(json.dumps(dict(
        metric=METRIC, value=val, unit=UNIT, n_gpus=int(os.environ.get("WORLD_SIZE", "1")), steps=args.steps, warmup=args.warmup,
        ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
        impl="reference",
        config=dict(workload=f"{args.workload}: {dims[0]}x{dims[1]}x{dims[2]}x{dims[3]} Ls={Ls} blocks {block} (bounded sample)",
                    parallelism="host cores"),
        gpu_launches=0,
        cpu_baseline=dict(value=val, unit=UNIT, cores=ora.threads, kind="oracle", sample=sample, cpu_model=cpu_model()),
        e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", choices=sorted(synth.CONFIGS))
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--block", default="", help="override the Dirichlet block, e.g. 12,12,12,12 (C5 block-size sweep)")
    ap.add_argument("--recon", type=int, default=18, choices=[12, 18], help="link storage of the low-precision copies (12 = two rows, R8)")
    ap.add_argument("--train-steps", type=int, default=100, help="line-search steps of the T training in the extras")
    ap.add_argument("--mu", type=float, default=0.85, help="shift mu of the reduced-Ls preconditioner in the extras (PAPER.md:309 eq. 20; the paper's tuned values: 0.437-0.85)")
    ap.add_argument("--cpu-solves", default="", choices=["", "C1", "C3p"], help="with --impl reference: full CG and MSPCG solves on the CPU oracle on this lattice (C3p = reduced C3: 12^3 x 24, Ls 8)")
    ap.add_argument("--m5inv-only", action="store_true", help="time only the stand-alone M5^-1 contraction (mspcg_apply_M5inv) on the workload and print its entry")
    ap.add_argument("--group", type=int, default=0, help="Dirichlet blocks per L2-resident group of the preconditioner (mspcg_set_block_group; 0 = all at once)")
    ap.add_argument("--solves", action="store_true", help="time to solution instead of the step benchmark: CG, MSPCG (and reduced-Ls MSPCG with --reduced-solve) on --workload")
    ap.add_argument("--reduced-solve", action="store_true", help="with --solves: also train T on a sample lattice and solve with the reduced-Ls preconditioner")
    ap.add_argument("--sloppy", type=int, default=32, choices=[16, 32], help="with --solves: bits of the sloppy outer iteration")
    ap.add_argument("--n-inner", type=int, default=0, help="with --solves: inner iterations (default: the configuration's)")
    ap.add_argument("--max-iter", type=int, default=200000)
    ap.add_argument("--reduced", type=int, default=0, help="profiling aid: run the step with the reduced-Ls preconditioner at this Ls_hat")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.m5inv_only:
        run_m5inv(args)
    elif args.solves:
        run_solves(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
