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
    import workloads as W
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


def call_bytes(R, E, U, H, D, b, dedup):
    """Algorithmic bytes of each of the three C-ABI calls: a PARTITION of SURVEY.md §8(d)'s step bytes (their sum is
    compulsory_bytes()).  The backward reads Q, O, dO, K, V, LSE and kv_row once: charged to the destination-major call;
    the source-major call is charged only what it alone must move (t_indptr, t_dst, dK, dV).  What it re-reads (Q, dO,
    K, V rows, the {lse, delta} table) is not compulsory and shows up in `traffic`, not here."""
    F = H * D
    idx = 4 * E if dedup else 0
    fwd = R * F * b + 2 * U * F * b + 4 * (R + 1) + idx + R * F * b + 4 * R * H
    bwd_dst = 3 * R * F * b + 2 * U * F * b + 4 * R * H + 4 * (R + 1) + idx + R * F * b
    bwd_src = 4 * (U + 1) + 4 * E + 2 * U * F * b
    return {"fwd": fwd, "bwd_dst": bwd_dst, "bwd_src": bwd_src}


def gathered_bytes(E, H, D, b):
    """Bytes each call brings through the L1 gather path: two F*b-byte rows per edge; the source-major
    call also gathers the 8*H-byte {lse, delta} record of the edge's destination."""
    F = H * D
    return {"fwd": 2 * E * F * b, "bwd_dst": 2 * E * F * b, "bwd_src": 2 * E * F * b + 8 * H * E}


def build_stamp():
    """Hash of the CUDA sources + flags the loaded library was built from (paper_2607_05095_b200/csrc/build/stamp.txt)."""
    try:
        return open(os.path.join(ROOT, "paper_2607_05095_b200", "csrc", "build", "stamp.txt")).read().strip()[:16]
    except Exception:
        return None


def committed_traffic(cfg, stamp):
    """ncu dram__bytes_read.sum + dram__bytes_write.sum per C-ABI call from profiles/traffic.csv (config,call,bytes,build);
    returned only for rows captured on the build that is running now."""
    out, src = {}, None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tp):
        for ln in open(tp).read().splitlines()[1:]:
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 4 and f[0] == str(cfg) and stamp and f[3] == stamp:
                out[f[1]] = int(f[2]); src = f"profiles/traffic.csv (ncu --set full, build {stamp})"
    return out, src


class ClockSampler:
    """SM clock and throttle reasons sampled through NVML from a thread of this process every ~2 ms while the timed
    region runs (a `nvidia-smi -lms` child does not produce a single line inside a 30 ms region)."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int):
        self.index, self.sm, self.mask, self.max_mhz, self.h, self.err = index, [], 0, None, None, None
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                try:
                    phys = int(vis.split(",")[index])
                except Exception:
                    phys = index
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # noqa: BLE001
            self.err = f"nvml unavailable: {e}"

    def _sample(self):
        nv = self.nv
        self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
        try:
            get = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
            self.mask |= int(get(self.h))
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample()
            except Exception as e:  # noqa: BLE001
                self.err = str(e)
                return
            time.sleep(0.002)

    def start(self):
        if self.h is None:
            return
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def stop(self):
        if self.h is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [self.err or "nvml unavailable"], "samples": 0}
        self._stop.set()
        if self._t is not None:
            self._t.join(timeout=2)
        reasons = sorted(n for bit, n in self.REASONS.items() if self.mask & bit)
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(self.sm), "source": "nvml, sampled during the timed region"}


# ---------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on a bounded sample
# ---------------------------------------------------------------------------------------------------------------
def oracle_sample(w, target_edges):
    """Destination-prefix sub-block of about target_edges edges (None: the whole block), in oracle inputs (float64)."""
    import oracle
    ob = oracle.block_build(w.R, w.root_idx, w.nbr_node, None, None, w.dedup_mode)
    if target_edges is None or target_edges >= w.E:
        Rs = w.R
    else:
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


def config_dict(args, ws, Us):
    """`config` of the JSON line: identical for both arms (the driver compares them)."""
    w0 = ws[0]
    comp = 0
    for w, U in zip(ws, Us):
        f, g = compulsory_bytes(w.R, w.E, U, w.H, w.D, 2 if w.dtype == "bf16" else 4, w.dedup_mode)
        comp += f + g
    return {"workload": f"config{args.config}:{'+'.join(w.name for w in ws)}", "R": sum(w.R for w in ws), "E": sum(w.E for w in ws),
            "U": int(sum(Us)), "H": w0.H, "D": w0.D, "storage": w0.dtype, "accumulate": "f32", "dedup_mode": w0.dedup_mode,
            "seed": args.seed, "per_rank": "independent mini-batch per rank (seed + rank)",
            "l2": f"no flush: resident tensors {comp / 1e6:.0f} MB per step vs 126 MB L2" if comp > 2.5e8
                  else "working set fits in L2 (launch-bound config): warm-L2 headline, cold-L2 (256 MB flush before every step) in extras.l2"}, comp


def oracle_cpu_baseline(ws, full_edges_cap, sample_edges):
    """the oracle as it stands on the host cores, fused forward + backward, generation and block build
    excluded; all cores on the whole workload (a destination prefix when it exceeds full_edges_cap edges), median of 5,
    and 1 thread on a bounded destination-prefix sample, median of 3."""
    import oracle
    oracle.build()
    ncores = oracle.num_threads()
    E_all = sum(w.E for w in ws)
    cap = None if E_all <= full_edges_cap else full_edges_cap // len(ws)
    full = [oracle_sample(w, cap) for w in ws]
    for s_ in full:
        oracle_step(s_)
    ts = []
    for _ in range(5):
        t0 = time.perf_counter()
        for s_ in full:
            oracle_step(s_)
        ts.append(time.perf_counter() - t0)
    e_full = sum(s_["Es"] for s_ in full)
    small = [oracle_sample(w, sample_edges // len(ws)) for w in ws] if E_all > sample_edges else full
    oracle.set_num_threads(1)
    t1 = []
    for _ in range(3):
        t0 = time.perf_counter()
        for s_ in small:
            oracle_step(s_)
        t1.append(time.perf_counter() - t0)
    oracle.set_num_threads(ncores)
    e_small = sum(s_["Es"] for s_ in small)
    return {"value": e_full / float(np.median(ts)), "unit": UNIT, "cores": ncores, "kind": "oracle",
            "sample": (f"whole workload, {e_full} edges" if e_full == E_all else f"destination prefix, {e_full} of {E_all} edges")
                      + ", all K/V rows; median of 5 fwd+bwd runs",
            "one_thread": {"value": e_small / float(np.median(t1)), "unit": UNIT, "cores": 1,
                           "sample": f"destination prefix, {e_small} of {E_all} edges; median of 3"}}


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
    sample = f"each step = destination prefix, {edges} of {sum(w.E for w in ws)} edges ({sum(s['Rs'] for s in samples)} roots), all {sum(s['U'] for s in samples)} K/V rows"
    cfg, _ = config_dict(args, ws, [s["U"] for s in samples])
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": cfg,
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


def run_extras(args, B, blocks, bi_dom, extras, peak):
    """Timed separately, never folded into the headline: block build, the unfused chain, next-1 (edge term), next-2 (SlimCache)."""
    import torch
    bb = blocks[bi_dom]
    w = bb["w"]
    eb = 2 if w.dtype == "bf16" else 4
    root_d, nbr_d = bb["host"]["root"].cuda(), bb["host"]["nbr"].cuda()
    B.block_build(w.R, root_d, nbr_d, None, None, w.dedup_mode)      # warm-up: allocator and first-launch costs
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(5):
        B.block_build(w.R, root_d, nbr_d, None, None, w.dedup_mode)
    torch.cuda.synchronize()
    bms = (time.perf_counter() - t0) * 1e3 / 5
    # the same call with its outputs and workspace pre-allocated (block_build(reuse=...): no torch.empty inside), timed by CUDA
    # events on the launching stream; the call still ends with its one synchronisation, so host gaps between calls are inside
    rb = B.block_build(w.R, root_d, nbr_d, None, None, w.dedup_mode)
    be = [torch.cuda.Event(enable_timing=True) for _ in range(11)]
    torch.cuda.synchronize()
    retries0 = B.block_build_retries()
    be[0].record()
    for i in range(10):
        rb = B.block_build(w.R, root_d, nbr_d, None, None, w.dedup_mode, reuse=rb)
        be[i + 1].record()
    torch.cuda.synchronize()
    bms_pre = float(np.median([be[i].elapsed_time(be[i + 1]) for i in range(10)]))
    assert torch.equal(rb.kv_row, bb["blk"].kv_row) and rb.U == bb["blk"].U
    U_ = bb["blk"].U
    # A0's algorithmic bytes: the sampler lists in (root_idx i32, nbr_node i64), every public index array out once
    bbytes = 12 * w.E + 4 * (w.R + 1) + 4 * w.E + ((4 * w.E + 8 * U_ + 4 * (U_ + 1) + 8 * w.E) if w.dedup_mode else 0)
    extras["block_build_ms"] = bms
    extras["block_build"] = {"ms": bms, "algorithmic_bytes": bbytes, "achieved_gbs": bbytes / (bms * 1e-3) / 1e9,
                             "frac_of_measured_copy": bbytes / (bms * 1e-3) / 1e9 / peak,
                             "timing": "host wall clock around 5 calls (the call synchronises to return U), output allocation included",
                             "ms_preallocated": bms_pre, "frac_of_measured_copy_preallocated": bbytes / (bms_pre * 1e-3) / 1e9 / peak,
                             "timing_preallocated": "median of 10 calls with outputs and workspace reused, CUDA events on the launching stream",
                             "retries_in_timed_calls": B.block_build_retries() - retries0}
    del rb
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


def run_next34(args, B, blocks, bi_dom, extras, peak):
    """NEXT-4 (plain AGG through both partitionings) and NEXT-3 (device sampler), timed separately."""
    import torch
    bb = blocks[bi_dom]
    w, blk, d, o = bb["w"], bb["blk"], bb["dev"], bb["out"]
    eb = 2 if w.dtype == "bf16" else 4
    F = w.H * w.D
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def tm(fn, n=5):
        fn()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    if F % 4 == 0 and w.E * F * 4 < 24e9:
        coo = B.block_coo_dst(blk)
        U_ = blk.U
        Yc, Xc = torch.empty(w.R, w.H, w.D, dtype=torch.float32, device="cuda"), torch.empty(U_, w.H, w.D, dtype=torch.float32, device="cuda")
        dXs = torch.empty_like(d["v"])
        res = {}
        # algorithmic bytes: rows in once, rows out once, the index arrays each scheme needs (CSR: indptr + one index; COO: two per-edge arrays)
        csr_f = U_ * F * eb + w.R * F * eb + 4 * w.E + 4 * (w.R + 1)
        csr_b = w.R * F * eb + U_ * F * eb + 4 * w.E + 4 * (U_ + 1)
        coo_f = U_ * F * eb + w.R * F * 4 + 8 * w.E
        coo_b = w.R * F * eb + U_ * F * 4 + 8 * w.E
        for name, fn, nb in (("csr_fwd", lambda: B.aggregate_fwd(blk, None, d["v"], out=o["O"]), csr_f),
                             ("csr_bwd", lambda: B.aggregate_bwd(blk, None, None, d["do"], want_dw=False), csr_b),
                             ("coo_atomic_fwd", lambda: B.aggregate_coo(blk, d["v"], coo, out=Yc), coo_f),
                             ("coo_atomic_bwd", lambda: B.aggregate_coo(blk, d["do"], coo, backward=True, out=Xc), coo_b)):
            ms = tm(fn)
            res[name] = {"ms": ms, "algorithmic_bytes": nb, "achieved_gbs": nb / (ms * 1e-3) / 1e9, "frac_of_measured_copy": nb / (ms * 1e-3) / 1e9 / peak,
                         "edges_per_s": w.E / (ms * 1e-3)}
        res["note"] = ("plain AGG h_v = sum v_u (PAPER.md:215) on this block: CSR gather (tg_aggregate_fwd/_bwd, w = NULL, no float atomics) vs the paper's "
                       "COO thread-per-edge red.global.add.v4.f32 (tg_aggregate_coo, PAPER.md:219-223, float32 output, zero-fill included)")
        extras["plain_agg"] = res
        del Yc, Xc, dXs, coo
    if not args.no_sampler:
        import workloads as W
        n_nodes, n_events, n_roots, k = 100_000, 5_000_000, 200_000, 10
        u, v, t = W._event_stream(args.seed, 2, n_nodes, n_events)
        ud, vd, td = (torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (u.astype(np.int64), v.astype(np.int64), t.astype(np.float32)))
        t_build = tm(lambda: B.tcsr_build(n_nodes, ud, vd, td), 3)
        g = B.tcsr_build(n_nodes, ud, vd, td)
        r = np.random.default_rng(args.seed)
        ev = r.integers(n_events // 2, n_events, n_roots)
        rn = torch.from_numpy(np.where(r.random(n_roots) < 0.5, u[ev], v[ev]).astype(np.int64)).cuda()
        rc = torch.from_numpy(ev.astype(np.int64)).cuda()
        out = {}
        for mode in ("recent", "uniform"):
            ms = tm(lambda: B.sample_neighbors(g, rn, rc, k, mode, 1))
            E_s = int(B.sample_neighbors(g, rn, rc, k, mode, 1)[0].numel())
            out[mode] = {"ms": ms, "roots": n_roots, "k": k, "sampled_edges": E_s, "sampled_edges_per_s": E_s / (ms * 1e-3),
                         "output_bytes": 24 * E_s, "host_list_bytes_not_sent": 24 * E_s}
        out["tcsr_build"] = {"ms": t_build, "events": n_events, "nodes": n_nodes, "entries": int(g.indptr[-1].item())}
        out["note"] = ("device-side temporal neighbour sampler (PAPER.md:311, 412) on config 2's stream: 200 000 roots drawn from the stream's second half; "
                       "times include output allocation and the D2H of E")
        extras["sampler"] = out


def run_e2e_sampled(args, B, extras):
    """`--e2e-sampled` (configs 1 and 3): the step end to end the B200-first way: the event stream's T-CSR and
    the node feature tables live in HBM (config 3: 1 M nodes x 256 B x 2 tables = 0.5 GB of 180 GB), so per step the host
    sends only the batch's roots (node, cutoff) and the per-root tensors (Q, dO); the sampler, the block build, the
    K / V row gather (tg_cache_lookup + tg_feature_reconstruct, every row resident) and the fused forward + backward run
    on the device; O, dQ, dK, dV come back.  No sampled list and no feature row crosses PCIe."""
    import torch
    import workloads as W
    cid = args.config
    n_nodes, n_events, batch, k, mode = {1: (20_000, 200_000, 600, 10, "recent"), 3: (1_000_000, 50_000_000, 4000, 20, "uniform")}[cid]
    H, D, dt = {1: (2, 50, torch.float32), 3: (4, 32, torch.bfloat16)}[cid]
    u, v, t = W._event_stream(args.seed, cid, n_nodes, n_events)
    rn, rc = W._batch_roots(u, v, n_nodes, batch, args.seed, cid)
    g = B.tcsr_build(n_nodes, torch.from_numpy(u.astype(np.int64)).cuda(), torch.from_numpy(v.astype(np.int64)).cuda(), torch.from_numpy(t.astype(np.float32)).cuda())
    del u, v, t
    gen = torch.Generator(device="cuda").manual_seed(args.seed)
    Ktab = (torch.randn(n_nodes, H, D, device="cuda", generator=gen) / math.sqrt(D)).to(dt)      # resident node-level K / V rows
    Vtab = (torch.randn(n_nodes, H, D, device="cuda", generator=gen) / math.sqrt(D)).to(dt)
    slot = torch.arange(n_nodes, dtype=torch.int32, device="cuda")                               # every node resident: slot = id
    none_fresh = torch.empty(0, H, D, dtype=dt, device="cuda")
    R = len(rn)
    h_rn, h_rc = torch.from_numpy(rn.astype(np.int64)).pin_memory(), torch.from_numpy(rc.astype(np.int64)).pin_memory()
    h_q = (torch.randn(R, H, D) / math.sqrt(D)).to(dt).pin_memory()
    h_do = torch.randn(R, H, D).to(dt).pin_memory()
    d_rn, d_rc, d_q, d_do = (torch.empty_like(x, device="cuda") for x in (h_rn, h_rc, h_q, h_do))
    h_out = {}

    def step():
        for dst, src in ((d_rn, h_rn), (d_rc, h_rc), (d_q, h_q), (d_do, h_do)):
            dst.copy_(src, non_blocking=True)
        lists = B.sample_neighbors(g, d_rn, d_rc, k, mode, args.seed)
        blk = B.block_build(R, lists[0], lists[1], lists[2], lists[3], 1)
        m_, _ = B.cache_lookup(blk.uniq_node, slot)
        K = B.feature_reconstruct(None, m_, none_fresh, Ktab)
        V = B.feature_reconstruct(None, m_, none_fresh, Vtab)
        O, lse = B.attn_fused_fwd(blk, d_q, K, V, 1.0)
        dQ, dK, dV = B.attn_fused_bwd(blk, d_q, K, V, O, lse, d_do, 1.0)
        for n, x in (("O", O), ("dQ", dQ), ("dK", dK), ("dV", dV)):
            if n not in h_out or h_out[n].shape != x.shape:
                h_out[n] = torch.empty(x.shape, dtype=x.dtype).pin_memory()
            h_out[n].copy_(x, non_blocking=True)
        torch.cuda.synchronize()
        return blk

    blk = step()
    n = max(3, min(args.steps, 20))
    t0 = time.perf_counter()
    for _ in range(n):
        blk = step()
    ms = (time.perf_counter() - t0) * 1e3 / n
    h2d = sum(x.numel() * x.element_size() for x in (h_rn, h_rc, h_q, h_do))
    d2h = sum(x.numel() * x.element_size() for x in h_out.values())
    extras["e2e_sampled"] = {"ms_per_step": ms, "edges": blk.E, "unique_rows": blk.U, "edges_per_s": blk.E / (ms * 1e-3), "h2d_bytes_per_step": h2d,
                             "d2h_bytes_per_step": d2h, "resident_bytes": int(Ktab.numel() * Ktab.element_size() * 2 + g.nbr.numel() * 20),
                             "sampling": f"{mode}, k = {k}, on the device", "steps": n,
                             "note": "host sends roots + Q + dO, receives O, dQ, dK, dV; T-CSR and node-level K / V tables resident in HBM; synchronous steps (no overlap)"}


def step_spread(per_step_ms, how):
    """median / min / p10 / p90 of single-step device times ('report median, min, p10/p90')."""
    a = np.sort(np.asarray(per_step_ms, dtype=np.float64))
    if a.size == 0:
        return None
    return {"median": float(np.median(a)), "min": float(a[0]), "p10": float(np.percentile(a, 10)), "p90": float(np.percentile(a, 90)),
            "max": float(a[-1]), "n": int(a.size), "rank": 0, "how": how}


def relaunch_under_torchrun(n_gpus: int) -> int:
    """`python bench.py --gpus N` with N > 1 and no rendezvous in the environment: start the N ranks ourselves, exactly as the
    driver's launch line does (one process per GPU, 127.0.0.1 rendezvous), and pass the ranks' output through.  NCCL's
    communicator log is switched on (unless the caller set NCCL_DEBUG) so that the number of ranks in the barrier / all-reduce
    communicator can be read off; its lines go to stderr, stdout stays the one JSON line of rank 0."""
    import socket
    import subprocess
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    p = subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, text=True)
    for ln in p.stdout:
        (sys.stderr if " NCCL " in ln else sys.stdout).write(ln)
    return p.wait()


def other_configs_extras(args, B, peak):
    """Configs 1-3 (launch-bound: the working set fits in L2) in the default line: one CUDA-graph replay of the fused
    fwd + bwd step per config, warm (back-to-back replays) and cold (256 MB L2 flush before every replay, outside the events).
    Not the headline: the driver never runs these configs by themselves."""
    import torch
    TDT = {"f32": torch.float32, "bf16": torch.bfloat16}
    out = {}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for c in (1, 2, 3):
        if c == args.config:
            continue
        ws = make_workloads(c, args.seed)
        items, comp_bytes = [], 0
        for w in ws:
            dt = TDT[w.dtype]
            blk = B.block_build(w.R, torch.from_numpy(w.root_idx).cuda(), torch.from_numpy(w.nbr_node).cuda(), None, None, w.dedup_mode)
            q, k, v, do = (torch.from_numpy(x).to(dt).cuda() for x in w.features(blk.U))
            o = dict(O=torch.empty_like(q), lse=torch.empty(w.R, w.H, dtype=torch.float32, device="cuda"), dQ=torch.empty_like(q),
                     dK=torch.empty_like(k), dV=torch.empty_like(v))
            items.append((w, blk, q, k, v, do, o))
            comp_bytes += sum(call_bytes(w.R, w.E, blk.U, w.H, w.D, 2 if w.dtype == "bf16" else 4, w.dedup_mode).values())

        def step():
            for w, blk, q, k, v, do, o in items:
                B.attn_fused_fwd(blk, q, k, v, w.scale, out=(o["O"], o["lse"]))
                B.attn_fused_bwd_dst(blk, q, k, v, o["O"], o["lse"], do, w.scale, o["dQ"])
                B.attn_fused_bwd_src(blk, q, k, v, do, w.scale, o["dK"], o["dV"])

        for _ in range(3):
            step()
        g, cs = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        cs.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(cs):
            step()
        torch.cuda.current_stream().wait_stream(cs)
        with torch.cuda.graph(g, stream=cs):
            step()
        n = 50
        for _ in range(5):
            g.replay()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        torch.cuda.synchronize()
        ev[0].record()
        for i in range(n):
            g.replay()
            ev[i + 1].record()
        torch.cuda.synchronize()
        warm = [ev[i].elapsed_time(ev[i + 1]) for i in range(n)]
        ce = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
        for i, (a, b_) in enumerate(ce):
            flush.fill_(i & 255)
            a.record()
            g.replay()
            b_.record()
        torch.cuda.synchronize()
        cold = float(np.median([a.elapsed_time(b_) for a, b_ in ce]))
        E = sum(it[0].E for it in items)
        wm = float(np.median(warm))
        out[f"config{c}"] = {"workload": "+".join(it[0].name for it in items), "E": E, "graph_ms_per_step": wm, "min_ms": float(min(warm)),
                             "edges_per_s": E / (wm * 1e-3), "cold_l2_ms_per_step": cold, "compulsory_bytes": comp_bytes,
                             "cold_frac_of_measured_copy": comp_bytes / (cold * 1e-3) / 1e9 / peak,
                             "byte_time_us_at_measured_copy": comp_bytes / (peak * 1e9) * 1e6}
        del g, items
    del flush
    return out


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
        root_h, nbr_h = torch.from_numpy(w.root_idx).pin_memory(), torch.from_numpy(w.nbr_node).pin_memory()
        blk = B.block_build(w.R, root_h.cuda(), nbr_h.cuda(), None, None, w.dedup_mode)
        q, k, v, do = w.features(blk.U)                                          # K/V sized from the block's own U
        hostbuf = dict(root=root_h, nbr=nbr_h,
                       q=torch.from_numpy(q).to(dt).pin_memory(), k=torch.from_numpy(k).to(dt).pin_memory(),
                       v=torch.from_numpy(v).to(dt).pin_memory(), do=torch.from_numpy(do).to(dt).pin_memory())
        d = {n: hostbuf[n].cuda() for n in ("q", "k", "v", "do")}
        out = dict(O=torch.empty_like(d["q"]), lse=torch.empty(w.R, w.H, dtype=torch.float32, device="cuda"),
                   dQ=torch.empty_like(d["q"]), dK=torch.empty_like(d["k"]), dV=torch.empty_like(d["v"]))
        # --side-copy (bf16 storage): the forward also writes a float32 copy of O and the backward takes delta from it
        # (DESIGN.md §6.2).  Measured on config 4: fwd +0.024 ms, bwd_dst -0.020 ms: no gain, so it is off by default.
        out["o32"] = torch.empty(w.R, w.H, w.D, dtype=torch.float32, device="cuda") if (w.dtype == "bf16" and args.side_copy) else None
        blocks.append(dict(w=w, blk=blk, host=hostbuf, dev=d, out=out, info=blk.info()))
    cfg, comp = config_dict(args, ws, [b["blk"].U for b in blocks])
    small = comp <= 2.5e8                                      # configs 1-3: working set fits in L2, launch-bound
    use_graph = (args.launch == "graph") or (args.launch == "auto" and small)

    def step(ev=None):
        for bi, b in enumerate(blocks):
            w, blk, d, o = b["w"], b["blk"], b["dev"], b["out"]
            if ev is not None: ev[bi][0].record()
            B.attn_fused_fwd(blk, d["q"], d["k"], d["v"], w.scale, out=(o["O"], o["lse"]), o32=o["o32"])
            if ev is not None: ev[bi][1].record()
            B.attn_fused_bwd_dst(blk, d["q"], d["k"], d["v"], o["O"], o["lse"], d["do"], w.scale, o["dQ"], o32=o["o32"])
            if ev is not None: ev[bi][2].record()
            B.attn_fused_bwd_src(blk, d["q"], d["k"], d["v"], d["do"], w.scale, o["dK"], o["dV"])
            if ev is not None: ev[bi][3].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, n, sampler=None):
        """EXACTLY n calls of fn between barrier + synchronize on both sides; device time by CUDA events."""
        barrier()
        if sampler is not None:
            sampler.start()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        for i in range(n):
            fn(i)
        t1.record()
        barrier()
        return t0.elapsed_time(t1)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step()
    # ---- eager launches: per-call events (this is also the headline when no graph is used) ----
    evs = [[[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in blocks] for _ in range(args.steps)]
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = B.launch_count()
    eager_ms = timed(lambda i: step(evs[i]), args.steps, None if use_graph else sampler)
    launches_per_step = (B.launch_count() - launches0) / args.steps
    total_ms, launch_mode = eager_ms, "eager (one C-ABI call per pass, launched from Python)"
    # ---- CUDA graph replay of the same step (default for the launch-bound configs) ----
    graph_ms = None
    if use_graph:
        g = torch.cuda.CUDAGraph()
        cs = torch.cuda.Stream()
        cs.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(cs):
            step()
        torch.cuda.current_stream().wait_stream(cs)
        with torch.cuda.graph(g, stream=cs):
            step()
        for _ in range(warm):
            g.replay()
        graph_ms = timed(lambda i: g.replay(), args.steps, sampler)
        total_ms, launch_mode = graph_ms, "cuda_graph_replay (the step's C-ABI calls captured once; tg_* calls are capturable)"
    clocks = sampler.stop() if rank == 0 else None
    # spread of single steps (SURVEY.md §8(d) timing protocol), this rank: one event pair per step.  Eager: the events already
    # recorded inside the headline region (first call's start -> last call's end, so launch gaps BETWEEN steps are not in it);
    # graph: a separate pass of the same length with an event between replays (the headline region has none).
    if use_graph:
        se = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
        barrier()
        se[0].record()
        for i in range(args.steps):
            g.replay()
            se[i + 1].record()
        barrier()
        per_step = [se[i].elapsed_time(se[i + 1]) for i in range(args.steps)]
        spread_how = "separate pass: one event between consecutive graph replays"
    else:
        per_step = [evs[i][0][0].elapsed_time(evs[i][-1][3]) for i in range(args.steps)]
        spread_how = "events of the headline region: first call's start to last call's end of each step"
    step_ms = step_spread(per_step, spread_how)
    E_local = sum(b["w"].E for b in blocks)
    total_ms, E_all = reduce_over_ranks(total_ms, E_local, world, "cuda")
    ms_per_step = total_ms / args.steps
    value = E_all / (ms_per_step * 1e-3)

    # per-call durations (this rank, eager launches), averaged over the timed steps
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
    cb = call_bytes(w.R, w.E, b["blk"].U, w.H, w.D, eb, w.dedup_mode)
    gb = gathered_bytes(w.E, w.H, w.D, eb)
    dom = max(per_block[bi_dom], key=per_block[bi_dom].get)
    dom_ms = per_block[bi_dom][dom]
    achieved = cb[dom] / (dom_ms * 1e-3) / 1e9
    # the roof the kernels actually sit against: 256-byte row gathers that hit L1, measured in this process (tg_probe_gather)
    l1_peak = B.probe_gather(512)
    traffic, traffic_src = committed_traffic(args.config, build_stamp())
    big_side = w.E >= (1 << 20)
    opname = {"fwd": "FwdOp", "bwd_dst": "Bwd1Op", "bwd_src": "Bwd2Op"}[dom]
    kernels = (f"tg_warp_kernel + tg_hub_warp_kernel (+ tg_hub_kernel x2) + 2 x tg_group_kernel <{opname}>" if big_side
               else f"tg_small_side_kernel (+ tg_hub_kernel) <{opname}>")
    call_name = {"fwd": "tg_attn_fused_fwd", "bwd_dst": "tg_attn_fused_bwd_dst", "bwd_src": "tg_attn_fused_bwd_src"}[dom]
    roofline = {"bound": "issue / L1 gather (see `binding`); the HBM fraction is reported because BASELINE.json's metric is quoted against HBM",
                "kernel": f"{call_name} = {kernels}", "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic.get(dom), "traffic_source": traffic_src,
                "algorithmic_bytes_per_launch": cb[dom], "kernel_ms": dom_ms,
                "binding": {"kind": "l1_gather", "achieved": gb[dom] / (dom_ms * 1e-3) / 1e9, "peak": l1_peak, "unit": "GB/s",
                            "frac": gb[dom] / (dom_ms * 1e-3) / 1e9 / l1_peak, "gathered_bytes_per_launch": gb[dom],
                            "peak_source": "tg_probe_gather(512 rows, all L1 hits) in this process"},
                "per_call": {n: {"ms": per_block[bi_dom][n], "algorithmic_bytes": cb[n], "hbm_frac": cb[n] / (per_block[bi_dom][n] * 1e-3) / 1e9 / peak,
                                 "l1_gather_frac": gb[n] / (per_block[bi_dom][n] * 1e-3) / 1e9 / l1_peak, "traffic": traffic.get(n)}
                             for n in ("fwd", "bwd_dst", "bwd_src")}}
    comp_all = comp * (E_all / max(E_local, 1))               # every rank runs a block of the same recipe
    hbm_gbs = comp_all / (ms_per_step * 1e-3) / 1e9
    hbm = {"compulsory_bytes_per_step": comp, "achieved_gbs": hbm_gbs, "frac_of_8TBs": hbm_gbs / HBM_NOMINAL_GBS / world,
           "frac_of_measured_copy": hbm_gbs / peak / world,
           "fp32_side_copy_of_O": {"used": any(x["out"]["o32"] is not None for x in blocks),
                                   "extra_bytes_per_step_not_counted": sum(2 * x["out"]["o32"].numel() * 4 for x in blocks if x["out"]["o32"] is not None)},
           "sum_of_call_bytes": sum(sum(call_bytes(x["w"].R, x["w"].E, x["blk"].U, x["w"].H, x["w"].D,
                                                                                        2 if x["w"].dtype == "bf16" else 4, x["w"].dedup_mode).values()) for x in blocks)}

    extras = {"launch": {"mode": launch_mode, "eager_ms_per_step": eager_ms / args.steps,
                         "graph_ms_per_step": None if graph_ms is None else graph_ms / args.steps,
                         "kernel_launches_per_step": launches_per_step}}
    # cold-L2 protocol for the configs that fit in L2: a 256 MB flush before every step, outside the timed events
    if small:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        n_cold = min(args.steps, 50)
        ce = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_cold)]
        for i in range(n_cold):
            flush.fill_(i & 255)
            ce[i][0].record()
            if use_graph:
                g.replay()
            else:
                step()
            ce[i][1].record()
        torch.cuda.synchronize()
        cold = float(np.median([a.elapsed_time(b_) for a, b_ in ce]))
        extras["l2"] = {"warm_ms_per_step": ms_per_step, "cold_ms_per_step": cold, "flush_bytes": 256 << 20,
                        "cold_hbm_gbs": comp / (cold * 1e-3) / 1e9, "cold_frac_of_measured_copy": comp / (cold * 1e-3) / 1e9 / peak}
        del flush

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
        bb["dout"] = [{**{n: torch.empty_like(bb["out"][n]) for n in OUT + ("lse",)},
                       "o32": None if bb["out"]["o32"] is None else torch.empty_like(bb["out"]["o32"])} for _ in range(NB)]
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
                O, lse = B.attn_fused_fwd(blk, di["q"], di["k"], di["v"], ww.scale, out=(do_["O"], do_["lse"]), o32=do_["o32"])
                B.attn_fused_bwd(blk, di["q"], di["k"], di["v"], O, lse, di["do"], ww.scale, out=(do_["dQ"], do_["dK"], do_["dV"]), o32=do_["o32"])
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

    run_extras(args, B, blocks, bi_dom, extras, peak)
    if not args.no_unfused:
        run_next34(args, B, blocks, bi_dom, extras, peak)
    if args.e2e_sampled and args.config in (1, 3):
        run_e2e_sampled(args, B, extras)
    if not args.no_other_configs and not args.no_unfused:
        extras["other_configs"] = other_configs_extras(args, B, peak)
    extras["kernel_ms"] = kms
    extras["schedule"] = {**blocks[bi_dom]["info"], **blocks[bi_dom]["blk"].sched_info()}

    cpu = None if args.no_cpu else oracle_cpu_baseline([bb["w"] for bb in blocks], args.cpu_full_edges, args.cpu_edges)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms_per_step, "step_ms": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic", "config": cfg,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(round(launches_per_step * args.steps)), "roofline": roofline, "hbm": hbm,
        "cpu_baseline": cpu, "extras": extras,
    }
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--cpu-edges", type=int, default=1_000_000, help="cpu_baseline: edges of the 1-thread sample")
    ap.add_argument("--cpu-full-edges", type=int, default=12_000_000, help="cpu_baseline: the all-core leg runs the whole workload up to this many edges")
    ap.add_argument("--launch", default="auto", choices=["auto", "eager", "graph"],
                    help="auto: CUDA-graph replay for the launch-bound configs (working set fits in L2), eager launches otherwise")
    ap.add_argument("--ref-edges", type=int, default=1_000_000)
    ap.add_argument("--src-nodes", type=int, default=0, help="diagnostic (config 4): number of source nodes; not the headline workload")
    ap.add_argument("--probe-gather", action="store_true", help="diagnostic: print the measured L1 / L2 row-gather bandwidth and exit")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-unfused", action="store_true", help="skip the extras: unfused chain, edge term, SlimCache, plain AGG, sampler")
    ap.add_argument("--no-sampler", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip extras.other_configs (configs 1-3, graph-replayed; ~45 s of host-side input generation)")
    ap.add_argument("--e2e-sampled", action="store_true", help="configs 1, 3: extras.e2e_sampled = the step with the sampler and the feature rows on the device")
    ap.add_argument("--side-copy", action="store_true", help="bf16 storage: the forward writes a float32 side copy of O, the backward takes delta from it")
    args = ap.parse_args()
    if args.probe_gather:
        from paper_2607_05095_b200 import binding as B
        rows = {"l1_64rows_16KB": 64, "l1_512rows_128KB": 512, "l2_65536rows_16MB": 65536, "dram_8Mrows_2GB": 8 << 20}
        print(json.dumps({"probe": "256-byte row gathers, 8 lanes x 2 LDG.128 per row", "unit": "GB/s",
                          **{k: round(B.probe_gather(v), 1) for k, v in rows.items()}}))
        for stages in (2, 4, 8):
            res = {k: B.probe_gather_bulk(v, stages) for k, v in rows.items()}
            print(json.dumps({"probe": f"the same gathers as cp.async.bulk (256 bytes per row, one elected lane per group) into a ring of {stages} "
                                       "shared-memory stages per warp, mbarrier completion, 2 LDS.128 per lane",
                              "unit": "GB/s", "ctas_per_sm": next(iter(res.values()))[1], **{k: round(v[0], 1) for k, v in res.items()}}))
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(relaunch_under_torchrun(args.gpus))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:   # one line per rank, before any heavy import: who was started
        print(f"[bench.py] rank {os.environ.get('RANK', '?')}/{os.environ['WORLD_SIZE']} started", file=sys.stderr, flush=True)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
