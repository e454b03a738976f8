#!/usr/bin/env python
"""bench.py -- one JSON line for the Light Interaction sparse-attention hot path on B200.

A "step" = one pass of the whole hot path (li_block_select + li_sparse_attn) over
one synthetic `mid` workload (BASELINE.json configs[1]; the config `metric` is quoted on).  value = effective
TFLOP/s counted over attended blocks only (4*d*valid_q*valid_k per (head, query block), from the actual mask).
Multi-GPU: the path has no exchange step: `--gpus N` runs N independent replicas, one per
rank, weak scaling, no collective on the data path.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config mid|long|tiny|adaptive|dense-equivalence]
  python bench.py --impl reference ...      # times the CPU oracle (oracle/li_oracle.py) on a bounded sample
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

import numpy as np
import torch

import li_workloads as W

METRIC = "sparse-attn effective TFLOP/s over attended blocks (select + attention, ms/call in ms_per_step)"
UNIT = "TFLOP/s"
# roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum of the attention kernel per launch, taken from the
# `ncu --set full` capture that profiles/traffic.json names for the workload (written from the extracted --page raw rows;
# null when no capture of this workload is committed).
def ncu_traffic(workload: str):
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(path) as f:
            e = json.load(f).get(workload)
        return (int(e["dram_bytes"]), f"profiles/{e['source']}") if e else (None, None)
    except (OSError, ValueError, KeyError):
        return None, None


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"bf16_tflops": float(d["bf16_tflops"]), "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "hbm_gbs": float(d["hbm_gbs"]), "source": "measured"}
    return {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0, "source": "fallback"}


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self.stop = index, [], threading.Event()
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop.wait(0.1)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm, mx, reasons, pw = [], 0.0, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                try:
                    pw.append(float(r[2]))
                except ValueError:
                    pass
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(pw) if pw else None}


# ------------------------------------------------------------------------------------------ CPU oracle arm
def oracle_sample(prob: W.Problem, n_heads: int, tiles_per_head=None):
    """Times oracle/li_oracle.py, as it stands, on a bounded sample of `prob`: the first n_heads heads of call 0
    (select for those heads + attention for their query blocks).  Returns (seconds, effective flops, description)."""
    from oracle import li_oracle as O
    s = prob.spec
    nh = min(n_heads, s.H)
    q = prob.u16(prob.q[:1, :nh].contiguous())
    kc = prob.u16(prob.k_cache[:, :nh].contiguous())
    vc = prob.u16(prob.v_cache[:, :nh].contiguous())
    fi = prob.frame_idx[prob.frame_off[0]:prob.frame_off[1]]
    fo = np.asarray([0, len(fi)], np.int32)
    tiles = None
    nq = prob.Nqb if tiles_per_head is None else min(tiles_per_head, prob.Nqb)
    if tiles_per_head is not None:
        tiles = [(0, h, i) for h in range(nh) for i in range(nq)]
    t0 = time.perf_counter()
    if s.block3d is not None:
        sel, _ = O.block_select_3d(q, kc, fi, fo, s.n_cur_frames, *s.grid, *s.block3d, prob.top_k[:1])
        O.sparse_attn_3d(q, kc, vc, fi, fo, s.n_cur_frames, *s.grid, *s.block3d, sel, tiles=tiles)
    else:
        sel, _ = O.block_select(q, kc, fi, fo, s.n_cur_frames, s.block, s.block, prob.top_k[:1])
        O.sparse_attn(q, kc, vc, fi, fo, s.n_cur_frames, s.block, s.block, sel, tiles=tiles)
    dt = time.perf_counter() - t0
    sub = W.Problem(s, prob.q[:1, :nh], prob.k_cache, prob.v_cache, fi, fo, prob.top_k[:1])
    vq, vk = sub.block_sizes(s.n_cur_frames), sub.block_sizes(sub.n_hist_frames(0))   # valid tokens per block
    Lc = s.n_cur_frames * s.frame_tokens
    flops = 0
    for h in range(nh):
        for i in range(nq):
            flops += 4 * s.d * int(vq[i]) * (Lc + int(sum(vk[int(m)] for m in sel[0][h, i])))
    desc = f"{s.name}: call 0, heads 0..{nh - 1} of {s.H}, query blocks 0..{nq - 1} of {prob.Nqb}, select + attention"
    return dt, flops, desc


def cpu_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        n = [int(i.get("num_threads", 1)) for i in threadpool_info() if i.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    prob = W.build(W.spec_by_name(args.config, H=args.ref_heads if args.config != "tiny" else None))
    times, flops, desc = [], 0, ""
    for it in range(args.warmup + args.steps):
        dt, flops, desc = oracle_sample(prob, args.ref_heads, args.ref_tiles)
        if it >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    val = flops / t / 1e12
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.config, "sample": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ multi-rank plumbing
def max_over_ranks(values, device, world):
    """Device-side timings of this rank -> the slowest rank's (the job's) timings.  The path has no exchange step
    (replicas only), so this all-reduce of a few scalars AFTER the timed region is the only collective."""
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def job_throughput(flops_per_replica_step, steps, world, total_ms):
    """Whole-job TFLOP/s: every rank runs one replica of the workload (weak scaling)."""
    return world * flops_per_replica_step * steps / (total_ms * 1e-3) / 1e12


# ------------------------------------------------------------------------------------------ CUDA arm
def run_cuda(args):
    import torch.distributed as dist

    import paper_2605_31158_b200 as li

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    li.lib()                                   # fail loudly if libli.so is missing

    spec = W.spec_by_name(args.config)
    prob = W.build(spec)                       # every rank: an independent replica of the same workload
    s = prob.spec
    # host side (pinned): what changes every step in the AR loop = Q, the chunk's K/V pages, the frame list
    q_host = prob.q.pin_memory()
    fi_host = torch.from_numpy(prob.frame_idx).pin_memory()
    cur_pages = sorted(set(int(prob.frame_idx[prob.frame_off[b + 1] - 1 - j]) for b in range(prob.B)
                           for j in range(s.n_cur_frames)))
    kcur_host = prob.k_cache[cur_pages].pin_memory()
    vcur_host = prob.v_cache[cur_pages].pin_memory()
    cur_idx = torch.tensor(cur_pages, device=dev)

    q = prob.q.to(dev)
    kc = prob.k_cache.to(dev)
    vc = prob.v_cache.to(dev)
    fi = torch.from_numpy(prob.frame_idx).to(dev)
    fp8 = args.kv == "fp8"
    if fp8:
        # FP8 (E4M3) K/V pages: one scale per head = max |value| of the pool / 448; the pool is quantised
        # once here (untimed), the chunk's pages again inside every end-to-end step (quantise-on-write)
        k_scale = (kc.float().abs().amax(dim=(0, 2, 3)) / 448.0).contiguous()
        v_scale = (vc.float().abs().amax(dim=(0, 2, 3)) / 448.0).contiguous()
        k8, v8 = torch.empty(kc.shape, dtype=torch.uint8, device=dev), torch.empty(vc.shape, dtype=torch.uint8, device=dev)
        ctx = li.Context(q, k8, v8, fi, prob.frame_off, s.n_cur_frames, s.block, grid=s.grid, block3d=s.block3d,
                         k_scale=k_scale, v_scale=v_scale)
        li.li_quantize_pages(ctx, kc, vc, torch.arange(s.n_pages, dtype=torch.int32, device=dev))
        kcur_dev, vcur_dev = kc[cur_pages].contiguous(), vc[cur_pages].contiguous()
        cur_idx32 = torch.tensor(cur_pages, dtype=torch.int32, device=dev)
        del kc, vc
        args.no_extras = True
    else:
        ctx = li.Context(q, kc, vc, fi, prob.frame_off, s.n_cur_frames, s.block, grid=s.grid, block3d=s.block3d)
    buf = li.Buffers(ctx, prob.kmax, want_scores=False, want_lse=True)
    o_host = torch.empty(buf.o.shape, dtype=buf.o.dtype).pin_memory()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2
    flush_words = flush.view(torch.int64)[::16]                            # one 8-byte word of every 128-byte line
    stream = torch.cuda.current_stream()

    def flush_l2(tag: int):
        """Between timed steps: WRITE a buffer twice the size of the L2 (evicts every line of the workload), then READ one
        word of each of its lines, so that the dirty lines the write left behind are written back now and not under the
        first kernel of the next step (the HBM-bound pool kernel would otherwise share the bus with ~126 MB of
        write-backs).  Both passes run outside the CUDA events."""
        flush.fill_(tag & 0xff)
        flush_words.sum()

    def step(ev=None):
        if ev is not None:
            ev[0].record(stream)
        li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, None, stream)
        if ev is not None:
            ev[1].record(stream)
        li.li_sparse_attn(ctx, buf.sel_idx, buf.sel_cnt, buf.kmax, buf.o, buf.lse, buf.workspace, stream)
        if ev is not None:
            ev[2].record(stream)

    def e2e_step():
        q.copy_(q_host, non_blocking=True)
        fi.copy_(fi_host, non_blocking=True)
        if fp8:
            kcur_dev.copy_(kcur_host, non_blocking=True)
            vcur_dev.copy_(vcur_host, non_blocking=True)
            li.li_quantize_pages(ctx, kcur_dev, vcur_dev, cur_idx32, stream)
        elif contiguous_cur:
            kc[cur_pages[0]:cur_pages[-1] + 1].copy_(kcur_host, non_blocking=True)
            vc[cur_pages[0]:cur_pages[-1] + 1].copy_(vcur_host, non_blocking=True)
        else:
            kc.index_copy_(0, cur_idx, kcur_host.to(dev, non_blocking=True))
            vc.index_copy_(0, cur_idx, vcur_host.to(dev, non_blocking=True))
        step()
        o_host.copy_(buf.o, non_blocking=True)

    contiguous_cur = cur_pages == list(range(cur_pages[0], cur_pages[-1] + 1))

    # End-to-end leg, pipelined by head groups (heads are independent): the step's inputs are copied,
    # computed and read back group by group on three streams, so that host->device copies, kernels and the
    # device->host copy of O overlap inside ONE step.  Same work, same bytes, same C-ABI calls (on head slices).
    # Needs B == 1 (a head slice of O is then contiguous); otherwise the plain sequence above is used.
    G = args.e2e_groups if (prob.B == 1 and args.e2e_groups > 1 and s.H % args.e2e_groups == 0 and not fp8) else 1
    if G > 1:
        Hg = s.H // G
        hs = [slice(g * Hg, (g + 1) * Hg) for g in range(G)]
        qh_g = [q_host[:, h_].contiguous().pin_memory() for h_ in hs]
        kh_g = [kcur_host[:, h_].contiguous().pin_memory() for h_ in hs]
        vh_g = [vcur_host[:, h_].contiguous().pin_memory() for h_ in hs]
        ctx_g = [li.Context(q[:, h_], kc[:, h_], vc[:, h_], fi, prob.frame_off, s.n_cur_frames, s.block, grid=s.grid,
                            block3d=s.block3d) for h_ in hs]
        buf_g = [li.Buffers(c, prob.kmax, want_scores=False, want_lse=True) for c in ctx_g]
        oh_g = [torch.empty(b_.o.shape, dtype=b_.o.dtype).pin_memory() for b_ in buf_g]
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        ev_in = [torch.cuda.Event() for _ in range(G)]
        ev_cmp = [torch.cuda.Event() for _ in range(G)]
        ev_out = [torch.cuda.Event() for _ in range(G)]

        def e2e_step_pipelined(first):
            if not first:
                s_in.wait_event(ev_cmp[G - 1])           # the previous step's kernels still read q / the chunk pages
            for g in range(G):
                with torch.cuda.stream(s_in):
                    if g == 0:
                        fi.copy_(fi_host, non_blocking=True)
                    q[:, hs[g]].copy_(qh_g[g], non_blocking=True)
                    for pi, pg in enumerate(cur_pages):
                        kc[pg, hs[g]].copy_(kh_g[g][pi], non_blocking=True)
                        vc[pg, hs[g]].copy_(vh_g[g][pi], non_blocking=True)
                    ev_in[g].record(s_in)
                stream.wait_event(ev_in[g])
                if not first:
                    stream.wait_event(ev_out[g])         # the previous step's O of this group is still being read back
                li.li_block_select(ctx_g[g], prob.top_k, buf_g[g].kmax, buf_g[g].sel_idx, buf_g[g].sel_cnt,
                                   buf_g[g].workspace, None, stream)
                li.li_sparse_attn(ctx_g[g], buf_g[g].sel_idx, buf_g[g].sel_cnt, buf_g[g].kmax, buf_g[g].o, buf_g[g].lse,
                                  buf_g[g].workspace, stream)
                ev_cmp[g].record(stream)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_cmp[g])
                    oh_g[g].copy_(buf_g[g].o, non_blocking=True)
                    ev_out[g].record(s_out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        flush_l2(1)
        step()
    torch.cuda.synchronize()
    sel_idx = buf.sel_idx.cpu().numpy()
    sel_cnt = buf.sel_cnt.cpu().numpy()
    flops = W.effective_flops(prob, [sel_idx[b] for b in range(prob.B)], [sel_cnt[b] for b in range(prob.B)])

    # ---- device-resident timing: K steps, L2 flushed between them, CUDA events on the launching stream ----
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    li.reset_launch_count()
    barrier()
    with ClockSampler(local) as clk:
        t_wall0 = time.perf_counter()
        for k in range(args.steps):
            flush_l2(k & 0xff)
            step(evs[k])
        barrier()
        launches = li.launch_count()            # counted by the library inside the timed region
        t_wall = time.perf_counter() - t_wall0
        while time.perf_counter() - t_wall0 < 0.6:      # very short runs: keep the same load up until the
            step()                                      # sampler has a few readings (not timed, not counted)
            torch.cuda.synchronize()
    sel_ms = np.asarray([e[0].elapsed_time(e[1]) for e in evs])
    att_ms = np.asarray([e[1].elapsed_time(e[2]) for e in evs])
    step_ms = np.asarray([e[0].elapsed_time(e[2]) for e in evs])
    total_ms = float(step_ms.sum())

    # ---- end to end: pinned host -> device copies of the step's inputs and device -> host read of O, timed ----
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if G > 1:
        o_mono = buf.o.clone()                           # the monolithic step's output on the same inputs
        for k in range(2):
            e2e_step_pipelined(k == 0)
        barrier()
        got = torch.cat([t.to(dev) for t in oh_g], dim=1).float()
        assert (got - o_mono.float()).abs().max().item() <= 4e-3, "head-pipelined e2e output differs from the monolithic step"
        e0.record(stream)
        s_in.wait_event(e0)
        for k in range(args.steps):
            e2e_step_pipelined(k == 0)
        stream.wait_event(ev_out[G - 1])                 # the step's result is on the host when the clock stops
        e1.record(stream)
    else:
        for _ in range(2):
            e2e_step()
        barrier()
        e0.record(stream)
        for k in range(args.steps):
            e2e_step()
        e1.record(stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    h2d = q_host.numel() * 2 + fi_host.numel() * 4 + kcur_host.numel() * 2 + vcur_host.numel() * 2
    d2h = o_host.numel() * 2

    # ---- extras: L2-warm attention, and the cost of the paged gather = attention over the frame-paged
    #      pool minus attention over the same context laid out contiguously with an identity frame list ----
    extras = {}
    if world == 1 and not args.no_extras:
        def time_attn(cx, n=10, cold=True):
            ts = []
            for _ in range(n):
                if cold:
                    flush_l2(3)
                a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                li.li_sparse_attn(cx, buf.sel_idx, buf.sel_cnt, buf.kmax, buf.o, buf.lse, buf.workspace, stream)
                b_.record(stream)
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b_))
            return float(np.mean(ts[2:]))
        extras["attn_ms_l2_warm"] = time_attn(ctx, cold=False)
        ts = []
        for _ in range(12):                              # select with the pooled history keys reused (denoising steps 2..K)
            flush_l2(5)
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, None, stream, reuse_kbar=True)
            b_.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b_))
        extras["select_ms_reuse_kbar"] = float(np.mean(ts[2:]))
        if s.grid is not None:
            # 3-D tiling: select from page-resident patch sums (li_pool_pages once per written page, then
            # li_block_select_cached); the chunk's pages are the ones (re)pooled every step
            cache = torch.empty(li.li_slice_cache_bytes(ctx) // 4, dtype=torch.float32, device=dev)
            li.li_pool_pages(ctx, torch.arange(s.n_pages, dtype=torch.int32, device=dev), cache, stream)
            cur_t = torch.tensor(cur_pages, dtype=torch.int32, device=dev)
            t_sel, t_pool = [], []
            for _ in range(12):
                flush_l2(6)
                a, b_, c_ = (torch.cuda.Event(enable_timing=True) for _ in range(3))
                a.record(stream)
                li.li_pool_pages(ctx, cur_t, cache, stream)
                b_.record(stream)
                li.li_block_select_cached(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, cache, buf.workspace, None, stream)
                c_.record(stream)
                torch.cuda.synchronize()
                t_pool.append(a.elapsed_time(b_)); t_sel.append(b_.elapsed_time(c_))
            extras["pool_pages_ms_chunk"] = float(np.mean(t_pool[2:]))
            extras["select_ms_slice_cache"] = float(np.mean(t_sel[2:]))
            li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, None, stream)
            del cache
        order = torch.from_numpy(prob.frame_idx.astype(np.int64)).to(dev)
        free_b = torch.cuda.mem_get_info()[0]
        need_b = 2 * order.numel() * kc[0].numel() * 2
        if need_b < free_b // 2:
            kc2, vc2 = kc.index_select(0, order), vc.index_select(0, order)
            ident = torch.arange(order.numel(), dtype=torch.int32, device=dev)
            ctx2 = li.Context(q, kc2, vc2, ident, prob.frame_off, s.n_cur_frames, s.block, grid=s.grid, block3d=s.block3d)
            t_paged, t_ident = time_attn(ctx), time_attn(ctx2)
            extras["attn_ms_paged"] = t_paged
            extras["attn_ms_identity_contiguous"] = t_ident
            extras["gather_overhead_frac"] = (t_paged - t_ident) / t_ident
            del kc2, vc2, ctx2
        # li_context_policy (Eq. 1-4, once per chunk): latency at the latent size of one 4-frame chunk of this grid
        # (16 channels x 4 frames x 60 x 104, bf16), and the streaming MSE against the HBM roofline on 2 x 256 MiB
        def time_policy(n, reps=12):
            z1 = torch.randn(n, device=dev).to(torch.bfloat16)
            z2 = torch.randn(n, device=dev).to(torch.bfloat16)
            ema = torch.zeros(2, dtype=torch.float32, device=dev)
            pages = torch.arange(32, dtype=torch.int32, device=dev)
            out = torch.empty(64, dtype=torch.int32, device=dev)
            res = torch.zeros(24, dtype=torch.uint8, device=dev)
            ws = torch.empty(li.lib().li_policy_workspace_bytes(), dtype=torch.uint8, device=dev)
            sp = torch.rand(8, device=dev)
            ts = []
            for _ in range(reps):
                flush_l2(7)
                a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                li.li_context_policy(z1, z2, ema, 0.3, 0.02, 16, sp, 0.45, pages[:4], pages[4:24], pages[24:28], out, res, ws,
                                     stream=stream)
                b_.record(stream)
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b_))
            return float(np.mean(ts[2:]))
        extras["policy_ms_chunk_latents"] = time_policy(16 * 4 * 60 * 104)
        n_big = 128 << 20
        t_big = time_policy(n_big)
        extras["policy_ms_2x256MiB"] = t_big
        extras["policy_mse_gbs"] = 2 * n_big * 2 / (t_big * 1e-3) / 1e9
        # sustained load: the board power cap pulls the SM clock down after ~50-100 ms of back-to-back steps, so a long
        # run is slower per step than the short timed region above (MEASURED_PEAKS.json's burst vs sustained figures)
        n_sus = max(50, min(300, int(250.0 / max(float(step_ms.mean()), 1e-3))))
        a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for k in range(n_sus + n_sus // 3):
            if k == n_sus // 3:
                a.record(stream)
            step()
        b_.record(stream)
        torch.cuda.synchronize()
        extras["step_ms_sustained"] = a.elapsed_time(b_) / n_sus
        extras["step_ms_sustained_note"] = f"{n_sus} back-to-back steps after {n_sus // 3} untimed ones, no L2 flush"
        if s.name == "dense-equivalence":
            # BASELINE.json configs[4], second half: li_block_select ALONE on the `long` shapes (Lk = 56160), timed as an
            # HBM-bound kernel: algorithmic bytes (Lq + L_hist) * d * 2 * H over its CUDA-event time, against the copy peak
            lprob = W.build(W.spec_by_name("long"))
            ls = lprob.spec
            lctx = li.Context(lprob.q.to(dev), lprob.k_cache.to(dev), lprob.v_cache.to(dev), torch.from_numpy(lprob.frame_idx).to(dev),
                              lprob.frame_off, ls.n_cur_frames, ls.block)
            lbuf = li.Buffers(lctx, lprob.kmax, want_scores=False, want_lse=False)
            ts = []
            for _ in range(14):
                flush_l2(9)
                a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                li.li_block_select(lctx, lprob.top_k, lbuf.kmax, lbuf.sel_idx, lbuf.sel_cnt, lbuf.workspace, None, stream)
                b_.record(stream)
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b_))
            lbytes = (lprob.Lq + lprob.L_hist(0)) * ls.d * 2 * ls.H
            t_sel = float(np.mean(ts[2:]))
            extras["block_select_alone_long"] = {"ms": t_sel, "bytes": int(lbytes), "gbs": lbytes / (t_sel * 1e-3) / 1e9,
                                                 "frac_of_hbm_peak": lbytes / (t_sel * 1e-3) / 1e9 / peaks()["hbm_gbs"], "Lk": lprob.L_hist(0) + lprob.Lq}

    total_ms, e2e_ms = max_over_ranks([total_ms, e2e_ms], dev, world)
    if rank == 0:
        pk = peaks()
        value = job_throughput(flops, args.steps, world, total_ms)
        e2e_val = job_throughput(flops, args.steps, world, e2e_ms)
        attn_tflops = flops / (float(att_ms.mean()) * 1e-3) / 1e12
        # FP8 pages: the tensor roofline is the fp8 one = the measured bf16 peak x the guide's nominal ratio (2x); the
        # select kernels read Q in bf16 and the historical K in one byte per element
        tpeak = pk["bf16_tflops"] * (2.0 if fp8 else 1.0)
        sel_bytes = sum((2 * prob.Lq + (1 if fp8 else 2) * prob.L_hist(b)) * s.d * s.H for b in range(prob.B))
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "fp8-e4m3 (K/V pages, Q rows and probabilities; fp32 accumulation)" if fp8 else "bf16", "data": "synthetic",
            "config": {"workload": s.name, "B": prob.B, "H": s.H, "d": s.d, "Lq": prob.Lq, "frame_tokens": s.frame_tokens,
                       "block": s.block, "block3d": s.block3d, "grid": s.grid, "kv": args.kv, "Lk": [prob.L_hist(b) + prob.Lq for b in range(prob.B)],
                       "top_k": [int(x) for x in prob.top_k], "M": [prob.M(b) for b in range(prob.B)],
                       "l2": "flushed between timed steps (256 MiB written, then read back so that no dirty line is left)", "multi_gpu": "replicas only (no collective)"},
            "effective_flops_per_step": int(flops),
            "select_ms": float(sel_ms.mean()), "attn_ms": float(att_ms.mean()), "attn_ms_min": float(att_ms.min()),
            "select_overhead_frac_of_attn": float(sel_ms.mean() / att_ms.mean()),
            "select_gbs": sel_bytes / (float(sel_ms.mean()) * 1e-3) / 1e9,
            "frac_of_peak_burst": attn_tflops / tpeak, "frac_of_peak_sustained": attn_tflops / (pk["bf16_tflops_sustained"] * (2.0 if fp8 else 1.0)),
            "roofline": {"bound": "tensor", "achieved": attn_tflops, "peak": tpeak, "unit": "TFLOP/s",
                         "frac": attn_tflops / tpeak, "traffic": None if fp8 else ncu_traffic(s.name)[0],
                         "traffic_source": None if fp8 else ncu_traffic(s.name)[1],
                         "kernel": "li_sparse_attn_fp8_kernel" if fp8 else "li_sparse_attn_kernel",
                         "peak_source": pk["source"] + (" burst bf16 x 2 (nominal fp8 : bf16 ratio)" if fp8 else " burst bf16")},
            "roofline_select": {"bound": "hbm", "achieved": sel_bytes / (float(sel_ms.mean()) * 1e-3) / 1e9, "peak": pk["hbm_gbs"],
                                "unit": "GB/s", "frac": sel_bytes / (float(sel_ms.mean()) * 1e-3) / 1e9 / pk["hbm_gbs"],
                                "kernel": "li_pool_kernel + li_score_topk_kernel"},
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": e2e_ms / args.steps,
                    "head_groups": G,
                    "note": "per step: Q, frame list and the chunk's K/V pages copied from pinned host memory, O read back; "
                            "the historical K/V cache stays resident (it is the cache)"
                            + ("; copies, kernels and read-back pipelined over %d head groups on three streams" % G if G > 1 else "")},
            "gpu_launches": int(launches), "clocks": clk.summary(),
        }
        line.update(extras)
        if "step_ms_sustained" in extras:
            # the long run against the SUSTAINED peak (the kernel is timed inside a long step there): whole step, select included
            line["step_sustained_frac_of_sustained_peak"] = flops / (extras["step_ms_sustained"] * 1e-3) / 1e12 / pk["bf16_tflops_sustained"]
        if not args.no_cpu and world == 1 and not fp8:
            dt, fl, desc = oracle_sample(prob, args.ref_heads, args.ref_tiles)
            line["cpu_baseline"] = {"value": fl / dt / 1e12, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                                    "sample": desc, "seconds": dt}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--e2e-groups", type=int, default=4, help="head groups the end-to-end leg is pipelined over (1 = plain sequence)")
    ap.add_argument("--config", default="mid", choices=["tiny", "mid", "long", "adaptive", "dense-equivalence", "mid3d", "long3d", "mid3d448"])
    ap.add_argument("--kv", default="bf16", choices=["bf16", "fp8"], help="precision of the K/V pages (fp8: E4M3 codes + per-head scales)")
    ap.add_argument("--ref-heads", type=int, default=24, help="heads in the oracle's bounded sample")
    ap.add_argument("--ref-tiles", type=int, default=None, help="query blocks per head in the oracle's sample (default all)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-extras", action="store_true", help="skip the L2-warm / gather-overhead measurements")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.steps == 20 and args.warmup == 5:
            args.steps, args.warmup = 2, 1
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
