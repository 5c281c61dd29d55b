#!/usr/bin/env python
"""bench.py -- sampled edges/s of the fused temporal-attention forward+backward (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

One step = tg_attn_fused_fwd + tg_attn_fused_bwd over one mini-batch block (config 4, the skewed
bf16 block BASELINE.json names as the roofline target, unless --config says otherwise).
`value` is measured with the inputs resident in HBM; `e2e` repeats the step through the same C-ABI
calls starting from pinned HOST buffers (sampler lists + Q/K/V/dO in, O/dQ/dK/dV out, block build
inside).  `roofline` is for the dominant kernel, timed live with CUDA events on the launch stream.
`cpu_baseline` / `--impl reference` time the CPU oracle (oracle/, as it stands) on a bounded sample.
N > 1 (torchrun): every rank runs an independent mini-batch (seed = rank): weak scaling, no collective.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "sampled_edges_per_s_fused_attn_fwd_bwd"
UNIT = "edges/s"
HBM_NOMINAL_GBS = 8000.0      # BASELINE.json: "vs 8 TB/s"
HBM_FALLBACK_GBS = 6650.0     # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def measured_hbm_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def make_workloads(cfg: int, seed: int, src_nodes: int = 0):
    from paper_2607_05095_b200 import workloads as W
    if src_nodes > 0:   # diagnostic: config 4's degree structure over `src_nodes` source nodes (16: every gather hits L1)
        assert cfg == 4, "--src-nodes is a config-4 diagnostic"
        w = W.config4(seed, n_src_nodes=src_nodes)
        w.name += f"_src{src_nodes}"
        return [w]
    if cfg == 1:
        return [W.config1(seed)]
    if cfg == 2:
        return list(W.config2(seed))
    if cfg == 3:
        return [W.config3(seed)]
    if cfg == 4:
        return [W.config4(seed)]
    if cfg == 40:  # config 4 with per-edge K/V rows (dedup_mode 0): the genuinely HBM-bound variant
        return [W.config4(seed, dedup_mode=0)]
    if cfg == 5:
        return [W.config5(seed)]
    raise SystemExit(f"unknown --config {cfg}")


def compulsory_bytes(R, E, U, H, D, b, dedup):
    """what the fused forward / backward must move once."""
    F = H * D
    fwd = R * F * b + 2 * U * F * b + 4 * (R + 1) + (4 * E if dedup else 0) + R * F * b + 4 * R * H
    bwd = 3 * R * F * b + 2 * U * F * b + 4 * R * H + 4 * (R + 1) + (4 * E if dedup else 0) + 4 * (U + 1) + 4 * E + R * F * b + 2 * U * F * b
    return fwd, bwd


def kernel_bytes(R, E, U, H, D, b, dedup):
    """Algorithmic bytes per launch of each of the three tier kernels."""
    F = H * D
    idx = 4 * E if dedup else 0
    fwd = 2 * R * F * b + 2 * U * F * b + 4 * (R + 1) + idx + 4 * R * H
    bwd_dst = (2 if b == 2 else 3) * R * F * b + 2 * U * F * b + 4 * R * H + 4 * (R + 1) + idx + R * F * b + 8 * R * H
    bwd_src = 2 * R * F * b + 2 * U * F * b + 8 * R * H + 4 * (U + 1) + 4 * E + 2 * U * F * b
    return {"fwd": fwd, "bwd_dst": bwd_dst, "bwd_src": bwd_src}


class ClockSampler:
    FIELDS = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append([x.strip() for x in ln.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            pass
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 6 for n, v in zip(names, r[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on a bounded sample
# ---------------------------------------------------------------------------------------------------------------
def oracle_sample(w, target_edges: int):
    """Destination-prefix sub-block of about target_edges edges, in oracle inputs (float64)."""
    import oracle
    ob = oracle.block_build(w.R, w.root_idx, w.nbr_node, None, None, w.dedup_mode)
    Rs = int(np.searchsorted(ob.indptr, target_edges, side="left"))
    Rs = max(1, min(Rs, w.R))
    Es = int(ob.indptr[Rs])
    q, k, v, do = w.features(ob.U)
    f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    return dict(indptr=ob.indptr[:Rs + 1].copy(), kv_row=ob.kv_row[:Es].copy(), q=f64(q[:Rs]), k=f64(k), v=f64(v), do=f64(do[:Rs]),
                Rs=Rs, Es=Es, U=ob.U, scale=w.scale)


def oracle_step(s):
    import oracle
    oracle.attn_fwd(s["indptr"], s["kv_row"], s["q"], s["k"], s["v"], s["scale"])
    oracle.attn_bwd(s["indptr"], s["kv_row"], s["q"], s["k"], s["v"], s["do"], s["scale"])


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    ws = make_workloads(args.config, args.seed)
    samples = [oracle_sample(w, args.ref_edges // len(ws)) for w in ws]
    for _ in range(args.warmup):
        for s in samples:
            oracle_step(s)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        for s in samples:
            oracle_step(s)
    dt = (time.perf_counter() - t0) / args.steps
    edges = sum(s["Es"] for s in samples)
    val = edges / dt
    sample = f"destination prefix, {edges} of {sum(w.E for w in ws)} edges ({sum(s['Rs'] for s in samples)} roots), all {sum(s['U'] for s in samples)} K/V rows"
    w0 = ws[0]
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config{args.config}:{'+'.join(w.name for w in ws)}", "H": w0.H, "D": w0.D, "storage": w0.dtype, "seed": args.seed},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ---------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------
def reduce_over_ranks(total_ms: float, edges_local: int, world: int, device: str):
    """Replicas only: every rank times its own independent mini-batch; the job's time is the MAX over
    ranks and its work the SUM of the ranks' edges.  No data-path collective."""
    if world <= 1:
        return total_ms, edges_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([total_ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e = torch.tensor([edges_local], device=device, dtype=torch.int64)
    dist.all_reduce(e)
    return float(t.item()), int(e.item())


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2607_05095_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libfasttg has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()

    ws = make_workloads(args.config, args.seed + rank, args.src_nodes)          # each rank: its own independent mini-batch
    TDT = {"f32": torch.float32, "bf16": torch.bfloat16}
    blocks = []
    for w in ws:
        dt = TDT[w.dtype]
        U = w.num_unique_rows()
        q, k, v, do = w.features(U)
        hostbuf = dict(root=torch.from_numpy(w.root_idx).pin_memory(), nbr=torch.from_numpy(w.nbr_node).pin_memory(),
                       q=torch.from_numpy(q).to(dt).pin_memory(), k=torch.from_numpy(k).to(dt).pin_memory(),
                       v=torch.from_numpy(v).to(dt).pin_memory(), do=torch.from_numpy(do).to(dt).pin_memory())
        blk = B.block_build(w.R, hostbuf["root"].cuda(), hostbuf["nbr"].cuda(), None, None, w.dedup_mode)
        assert blk.U == U
        d = {n: hostbuf[n].cuda() for n in ("q", "k", "v", "do")}
        out = dict(O=torch.empty_like(d["q"]), lse=torch.empty(w.R, w.H, dtype=torch.float32, device="cuda"),
                   dQ=torch.empty_like(d["q"]), dK=torch.empty_like(d["k"]), dV=torch.empty_like(d["v"]))
        blocks.append(dict(w=w, blk=blk, host=hostbuf, dev=d, out=out, info=blk.info()))

    def step(ev=None):
        for bi, b in enumerate(blocks):
            w, blk, d, o = b["w"], b["blk"], b["dev"], b["out"]
            if ev is not None: ev[bi][0].record()
            B.attn_fused_fwd(blk, d["q"], d["k"], d["v"], w.scale, out=(o["O"], o["lse"]))
            if ev is not None: ev[bi][1].record()
            B.attn_fused_bwd_dst(blk, d["q"], d["k"], d["v"], o["O"], o["lse"], d["do"], w.scale, o["dQ"])
            if ev is not None: ev[bi][2].record()
            B.attn_fused_bwd_src(blk, d["q"], d["k"], d["v"], d["do"], w.scale, o["dK"], o["dV"])
            if ev is not None: ev[bi][3].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    evs = [[[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in blocks] for _ in range(args.steps)]
    barrier()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = B.launch_count()
    t_start.record()
    for i in range(args.steps):
        step(evs[i])
    t_end.record()
    launches = B.launch_count() - launches0
    barrier()
    total_ms = t_start.elapsed_time(t_end)
    clocks = sampler.stop() if rank == 0 else None
    E_local = sum(b["w"].E for b in blocks)
    total_ms, E_all = reduce_over_ranks(total_ms, E_local, world, "cuda")
    ms_per_step = total_ms / args.steps
    value = E_all / (ms_per_step * 1e-3)

    # per-kernel durations (this rank), averaged over the timed steps
    kms = {"fwd": 0.0, "bwd_dst": 0.0, "bwd_src": 0.0}
    per_block = [dict(kms) for _ in blocks]
    for i in range(args.steps):
        for bi in range(len(blocks)):
            e = evs[i][bi]
            for j, n in enumerate(("fwd", "bwd_dst", "bwd_src")):
                per_block[bi][n] += e[j].elapsed_time(e[j + 1]) / args.steps
    for pb in per_block:
        for n in kms:
            kms[n] += pb[n]

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---------------- rank 0: roofline, e2e, extras, cpu baseline ----------------
    peak, peak_src = measured_hbm_gbs()
    bi_dom = max(range(len(blocks)), key=lambda i: sum(per_block[i].values()))
    b = blocks[bi_dom]
    w = b["w"]
    eb = 2 if w.dtype == "bf16" else 4
    kb = kernel_bytes(w.R, w.E, b["blk"].U, w.H, w.D, eb, w.dedup_mode)
    dom = max(per_block[bi_dom], key=per_block[bi_dom].get)
    achieved = kb[dom] / (per_block[bi_dom][dom] * 1e-3) / 1e9
    # DRAM bytes of the dominant call from the committed ncu capture (profiles/traffic.csv), per call like `achieved`
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tp):
        for ln in open(tp).read().splitlines()[1:]:
            f = ln.split(",")
            if len(f) >= 3 and f[0] == str(args.config) and f[1] == dom:
                traffic = int(f[2])
    roofline = {"bound": "hbm", "kernel": {"fwd": "tg_attn_fused_fwd", "bwd_dst": "tg_attn_fused_bwd_dst", "bwd_src": "tg_attn_fused_bwd_src"}[dom]
                + f" = tg_warp_kernel + tg_hub_kernel + 2 x tg_group_kernel <{ {'fwd': 'FwdOp', 'bwd_dst': 'Bwd1Op', 'bwd_src': 'Bwd2Op'}[dom] }>", "achieved": achieved,
                "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "algorithmic_bytes_per_launch": kb[dom], "kernel_ms": per_block[bi_dom][dom]}
    comp = 0
    for bb in blocks:
        ww = bb["w"]
        f, g = compulsory_bytes(ww.R, ww.E, bb["blk"].U, ww.H, ww.D, 2 if ww.dtype == "bf16" else 4, ww.dedup_mode)
        comp += f + g
    hbm_gbs = comp / (ms_per_step * 1e-3) / 1e9 * (1 if world == 1 else 1)
    hbm = {"compulsory_bytes_per_step": comp, "achieved_gbs": hbm_gbs, "frac_of_8TBs": hbm_gbs / HBM_NOMINAL_GBS,
           "frac_of_measured_copy": hbm_gbs / peak}

    # end to end from pinned host buffers, through the same C-ABI calls.  Three streams and two sets of device buffers:
    # the H2D copies of step i+1 and the D2H copies of step i-1 overlap step i's block build and kernels (PCIe is full
    # duplex); every step still moves all of its inputs in and all of its results out inside the timed region.
    IN, OUT = ("root", "nbr", "q", "k", "v", "do"), ("O", "dQ", "dK", "dV")
    s_in, s_cmp, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    NB = 2
    ev_in, ev_cmp, ev_out = ([torch.cuda.Event() for _ in range(NB)] for _ in range(3))
    h2d = d2h = 0
    for bb in blocks:
        bb["hout"] = {n: torch.empty(bb["out"][n].shape, dtype=bb["out"][n].dtype).pin_memory() for n in OUT}
        bb["din"] = [{n: torch.empty_like(bb["host"][n], device="cuda") for n in IN} for _ in range(NB)]
        bb["dout"] = [{n: torch.empty_like(bb["out"][n]) for n in OUT + ("lse",)} for _ in range(NB)]
        h2d += sum(t.numel() * t.element_size() for t in bb["host"].values())
        d2h += sum(t.numel() * t.element_size() for t in bb["hout"].values())

    def e2e_h2d(k):
        with torch.cuda.stream(s_in):
            s_in.wait_event(ev_cmp[k])                       # the step that last read these device buffers is done
            for bb in blocks:
                for n in IN:
                    bb["din"][k][n].copy_(bb["host"][n], non_blocking=True)
            ev_in[k].record(s_in)

    def e2e_compute(k):
        with torch.cuda.stream(s_cmp):
            s_cmp.wait_event(ev_in[k])
            s_cmp.wait_event(ev_out[k])                      # the results last written into these buffers have left
            for bb in blocks:
                ww, di, do_ = bb["w"], bb["din"][k], bb["dout"][k]
                blk = B.block_build(ww.R, di["root"], di["nbr"], None, None, ww.dedup_mode)
                O, lse = B.attn_fused_fwd(blk, di["q"], di["k"], di["v"], ww.scale, out=(do_["O"], do_["lse"]))
                B.attn_fused_bwd(blk, di["q"], di["k"], di["v"], O, lse, di["do"], ww.scale, out=(do_["dQ"], do_["dK"], do_["dV"]))
            ev_cmp[k].record(s_cmp)

    def e2e_d2h(k):
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_cmp[k])
            for bb in blocks:
                for n in OUT:
                    bb["hout"][n].copy_(bb["dout"][k][n], non_blocking=True)
            ev_out[k].record(s_out)

    def e2e_run(n):
        e2e_h2d(0)
        for i in range(n):
            k = i % NB
            if i + 1 < n:
                e2e_h2d((i + 1) % NB)
            e2e_compute(k)
            e2e_d2h(k)

    e2e_steps = max(2, min(args.steps, args.e2e_steps))
    e2e_run(2)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e2e_run(e2e_steps)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    e2e = {"value": E_local / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
           "ms_per_step": e2e_ms, "steps": e2e_steps,
           "includes": "per step: H2D of sampler lists + Q/K/V/dO from pinned memory, tg_block_build, fused fwd+bwd, D2H of O/dQ/dK/dV; "
                       "double-buffered on three streams (copies of neighbouring steps overlap the kernels)"}
    for bb in blocks:
        del bb["din"], bb["dout"]

    # extras: block build and the unfused chain, timed separately (never folded into the headline)
    extras = {}
    bb = blocks[bi_dom]
    root_d, nbr_d = bb["host"]["root"].cuda(), bb["host"]["nbr"].cuda()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(3):
        B.block_build(w.R, root_d, nbr_d, None, None, w.dedup_mode)
    torch.cuda.synchronize()
    extras["block_build_ms"] = (time.perf_counter() - t0) * 1e3 / 3
    if not args.no_unfused:
        d, o, blk = bb["dev"], bb["out"], bb["blk"]
        s = torch.empty(w.E, w.H, dtype=torch.float32, device="cuda")
        a = torch.empty_like(s)
        def unfused():
            B.sddmm(blk, d["q"], d["k"], w.scale, out=s)
            B.edge_softmax_fwd(blk, s, out=a)
            B.aggregate_fwd(blk, a, d["v"], out=o["O"])
            dV, da = B.aggregate_bwd(blk, a, d["v"], d["do"])
            ds = B.edge_softmax_bwd(blk, a, da)
            B.aggregate_fwd(blk, ds, d["k"], out=o["dQ"])
            B.aggregate_bwd(blk, ds, None, d["q"], want_dw=False)
        unfused()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(3):
            unfused()
        e1.record()
        torch.cuda.synchronize()
        extras["unfused_chain_ms"] = e0.elapsed_time(e1) / 3
        del s, a
        # NEXT-1: the full TGAT edge term on the same block -- per-edge key/value rows make it the
        # rho = 1, HBM-bound regime.  Compulsory bytes = the base step's + Ke, Ve read once by the forward and by the
        # backward, dKe, dVe written once.
        if w.E * w.H * w.D * eb * 4 < 24e9:
            gen = torch.Generator(device="cuda").manual_seed(1234)
            ke = (torch.randn(w.E, w.H, w.D, device="cuda", generator=gen) / math.sqrt(w.D)).to(d["q"].dtype)
            ve = (torch.randn(w.E, w.H, w.D, device="cuda", generator=gen) / math.sqrt(w.D)).to(d["q"].dtype)
            def edge_step():
                O, lse = B.attn_edge_fused_fwd(blk, d["q"], d["k"], d["v"], ke, ve, w.scale, 0.2, out=(o["O"], o["lse"]))
                return B.attn_edge_fused_bwd(blk, d["q"], d["k"], d["v"], ke, ve, O, lse, d["do"], w.scale, 0.2)
            edge_step()
            torch.cuda.synchronize()
            e0.record()
            for _ in range(3):
                edge_step()
            e1.record()
            torch.cuda.synchronize()
            ems = e0.elapsed_time(e1) / 3
            f_, g_ = compulsory_bytes(w.R, w.E, bb["blk"].U, w.H, w.D, eb, w.dedup_mode)
            ebytes = f_ + g_ + 6 * w.E * w.H * w.D * eb
            extras["edge_term"] = {"ms_per_step": ems, "edges_per_s": w.E / (ems * 1e-3), "compulsory_bytes": ebytes,
                                   "achieved_gbs": ebytes / (ems * 1e-3) / 1e9, "frac_of_measured_copy": ebytes / (ems * 1e-3) / 1e9 / peak,
                                   "slope": 0.2}
            del ke, ve
        # NEXT-2: SlimCache's device half on the same block -- cache lookup of the unique source ids, then
        # reconstruction of the per-edge K rows from (transferred unique rows || resident cache) through inv_Idx = kv_row.
        # Algorithmic bytes: n rows written, every unique row read once, the two index arrays.
        if w.E * w.H * w.D * eb < 24e9:
            U_ = bb["blk"].U
            n_ids = int(bb["blk"].uniq_node.max().item()) + 1 if U_ else 1
            slot = torch.full((n_ids,), -1, dtype=torch.int32, device="cuda")
            deg_u = (bb["blk"].t_indptr[1:] - bb["blk"].t_indptr[:-1]).long()
            hot = torch.argsort(deg_u, descending=True)[: U_ // 3]              # the most referenced third is "resident"
            slot[bb["blk"].uniq_node[hot]] = torch.arange(hot.numel(), dtype=torch.int32, device="cuda")
            cache_rows = d["k"][hot].contiguous()
            m_, fresh_ids = B.cache_lookup(bb["blk"].uniq_node, slot)
            fresh_rows = d["k"][(m_ >= 0).nonzero().squeeze(1)].contiguous()
            outk = torch.empty(w.E, w.H, w.D, dtype=d["k"].dtype, device="cuda")
            B.feature_reconstruct(bb["blk"].kv_row, m_, fresh_rows, cache_rows, out=outk)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(3):
                B.feature_reconstruct(bb["blk"].kv_row, m_, fresh_rows, cache_rows, out=outk)
            e1.record()
            torch.cuda.synchronize()
            rms = e0.elapsed_time(e1) / 3
            rb = w.H * w.D * eb
            rbytes = w.E * rb + U_ * rb + 4 * w.E + 4 * U_
            extras["slimcache_reconstruct"] = {"ms": rms, "rows": w.E, "row_bytes": rb, "unique_rows": U_, "resident_rows": int(hot.numel()),
                                               "transferred_rows": int(fresh_ids.numel()), "algorithmic_bytes": rbytes,
                                               "achieved_gbs": rbytes / (rms * 1e-3) / 1e9, "frac_of_measured_copy": rbytes / (rms * 1e-3) / 1e9 / peak}
            del outk, fresh_rows, cache_rows, slot
    extras["kernel_ms"] = kms
    extras["schedule"] = bb["info"]

    # CPU oracle on a bounded sample of the same workload
    cpu = None
    if not args.no_cpu:
        import oracle
        oracle.build()
        samples = [oracle_sample(bb_["w"], args.cpu_edges // len(blocks)) for bb_ in blocks]
        for s_ in samples:
            oracle_step(s_)
        ts = []
        for _ in range(3):
            t0 = time.perf_counter()
            for s_ in samples:
                oracle_step(s_)
            ts.append(time.perf_counter() - t0)
        edges = sum(s_["Es"] for s_ in samples)
        cpu = {"value": edges / float(np.median(ts)), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"destination prefix, {edges} of {E_local} edges, all K/V rows; median of 3 fwd+bwd runs"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic",
        "config": {"workload": f"config{args.config}:{'+'.join(x['w'].name for x in blocks)}", "R": sum(x["w"].R for x in blocks), "E": E_local,
                   "U": sum(x["blk"].U for x in blocks), "H": w.H, "D": w.D, "storage": w.dtype, "accumulate": "f32", "dedup_mode": w.dedup_mode,
                   "seed": args.seed, "per_rank": "independent mini-batch per rank (seed + rank)",
                   "l2": f"no flush: resident tensors {comp / 1e6:.0f} MB per step vs 126 MB L2" if comp > 2.5e8 else "working set fits in L2 (launch-bound config); no flush"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "hbm": hbm,
        "cpu_baseline": cpu, "extras": extras,
    }
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--cpu-edges", type=int, default=2_000_000)
    ap.add_argument("--ref-edges", type=int, default=1_000_000)
    ap.add_argument("--src-nodes", type=int, default=0, help="diagnostic (config 4): number of source nodes; not the headline workload")
    ap.add_argument("--probe-gather", action="store_true", help="diagnostic: print the measured L1 / L2 row-gather bandwidth and exit")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-unfused", action="store_true")
    args = ap.parse_args()
    if args.probe_gather:
        from paper_2607_05095_b200 import binding as B
        rows = {"l1_64rows_16KB": 64, "l1_512rows_128KB": 512, "l2_65536rows_16MB": 65536, "dram_8Mrows_2GB": 8 << 20}
        print(json.dumps({"probe": "256-byte row gathers, 8 lanes x 2 LDG.128 per row", "unit": "GB/s",
                          **{k: round(B.probe_gather(v), 1) for k, v in rows.items()}}))
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
