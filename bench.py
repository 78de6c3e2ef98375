#!/usr/bin/env python
"""bench.py -- throughput of the IBP hot path (fused gather-and-decompress) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload gnn|dlrm|tiny] [--impl reference]

One "step" = one pass of the whole hot path (plus the ordering pre-pass when the handle uses it)
over one batch of synthetic ids: ibp_gather_decompress(handle, row_ids, n, out, stream).  A different seeded id batch
every step.  Default workload = BASELINE.json configs[1] (GNN node-feature gather, 10M x 128 fp32, 250k unique ids); the
default run also measures the other four BASELINE configs (Tiny, DLRM, KV with all 32 layers, weight streaming with all 32
layers, one layer per step) and reports them in `per_config`, and the headline step over a cudaHostAlloc store in
`value_pinned_store`.

Prints ONE JSON line (rank 0):
  value      effective (decompressed) GB/s, whole job, ids resident in HBM, the packed store in host memory (that the
             store is read over PCIe IS the method; nothing else is staged)
  e2e        same metric through ibp_gather_decompress_host: pinned HOST ids in, pinned HOST rows out, copies timed
  roofline   dominant kernel (ibp_decode_kernel): achieved = ALGORITHMIC link bytes of the launch (sum of ceil(k_g/8) over the
             batch's distinct rows) / its duration (CUDA events on the launch stream); peak = cudaMemcpy H2D
             ceiling measured in this run (BASELINE.json north_star: "measured cudaMemcpy H2D ceiling"); bound = "pcie"
             (DESIGN.md section 7); frac_stored = the same with rows rounded up to the declared alignment unit A; traffic =
             read from the committed ncu summary of this kernel build (profiles/r02_*_decode_ncu.md) or null
  cpu_baseline  the oracle (oracle/, as it stands, 1 thread) on a bounded sample of the same workload
Timing: CUDA events around every step on the launch stream, L2 flushed (256 MiB write) between steps outside the
events, >= 3 warm-up steps, barrier + synchronize on both sides, max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

def make_workload(name):
    from paper_2605_30728_b200 import workloads
    if name == "gnn":
        return workloads.GNN()
    if name == "gnn-interleaved":
        return workloads.GNN(interleaved=True)
    if name == "dlrm":
        return workloads.DLRM()
    if name == "dlrm-hot":
        return workloads.DLRM(hot_order=True)
    if name == "tiny":
        return workloads.Tiny()
    if name == "kv":
        return workloads.KV()
    raise SystemExit(f"unknown workload {name}")


def describe(w):
    if getattr(w, "hot_order", False):
        return ("configs[2] DLRM embedding lookup with the store laid out by sampling rank (slot = rank x 26 + table; the entries are i.i.d., so "
                "ratio and content are unchanged): 26 x 2M x 64 fp32 (13.3 GB), groups of 128, 16384 x 26 Zipf(1.05) ids per step (repeats kept)")
    if getattr(w, "interleaved", False):
        return ("configs[1] GNN node-feature gather, SECONDARY variant (reading R15): the 70% N(0,1)-in-2^-8-steps rows and the 30% sparse 0/1 rows are "
                "interleaved at random, so every group of 256 mixes both types; 10M x 128 fp32, 250k unique Zipf(0.9) ids per step")
    return {
        "gnn": "configs[1] GNN node-feature gather: 10M x 128 fp32 (5.12 GB), 70% N(0,1) in 2^-8 steps + 30% sparse 0/1 at 2%, groups of 256, 250k unique Zipf(0.9) ids per step",
        "dlrm": "configs[2] DLRM embedding lookup: 26 x 2M x 64 fp32 (13.3 GB), U(-0.05,0.05) in 2^-12 steps, groups of 128, 16384 x 26 Zipf(1.05) ids per step (repeats kept)",
        "tiny": "configs[0] Tiny: 4096 x 128 fp32, N(0,1) in 2^-6 steps clipped to 8, groups of 64, 1024 uniform ids per step",
        "kv": "configs[3] LLM KV-cache offload: bf16 K/V, 32 layers x 32 heads x head_dim 128, 16-token pages, 8 x 4096 tokens (17.2 GB); K~N(0,1), V~N(0,0.5); group = one page of one head; 64 random pages per layer fetched per step (4096 spans of 512 rows, 512 MiB out)",
    }[w.name]


# ------------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML; nvidia-smi as a fallback is not needed)."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self._stop = [], set(), None, threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "applications_clocks_setting": 0x2}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.01)

    def start(self):
        if self.nv:
            self.t.start()

    def stop(self):
        self._stop.set()
        if self.nv and self.t.is_alive():
            self.t.join(timeout=1)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------- oracle arm
class OracleSample:
    """The CPU oracle on a bounded sample of the workload: a few hundred groups of the table (built once with the
    oracle's own compressor), then ids of the workload's batch sampler that fall in those groups.  Single thread."""

    def __init__(self, w, thr=(1, 1)):
        import oracle
        self.oracle, self.w = oracle, w
        G = w.group_param
        n_groups = 96 if w.row_bytes >= 512 else 160
        ids_all = np.concatenate([w.ids(1000 + i) for i in range(2)])
        if w.index_span > 1:                                   # span ids -> row ids (first spans only: bounded sample)
            ids_all = (ids_all[:8, None] * w.index_span + np.arange(w.index_span)[None, :]).reshape(-1)
        groups = np.unique(ids_all // G)[:n_groups]
        blocks = [w.rows(int(g) * G, min(G, w.n_rows - int(g) * G)) for g in groups]
        self.X = np.concatenate(blocks)
        starts = np.cumsum([0] + [b.shape[0] for b in blocks])
        sel = ids_all[np.isin(ids_all // G, groups)]
        gi = np.searchsorted(groups, sel // G)
        self.local = (starts[gi] + sel % G).astype(np.int64)
        self.n_groups = len(groups)
        self.ds = oracle.Dataset(self.X, 0, G) if thr[0] == thr[1] else oracle.DatasetT(self.X, 0, G, thr[0], thr[1])
        reps = np.resize(self.local, 2000)
        t0 = time.perf_counter()
        self.ds.gather_decompress(reps)
        self.sec_per_row = (time.perf_counter() - t0) / len(reps)

    def run(self, seconds_target):
        w = self.w
        n = int(max(2000, min(4_000_000, seconds_target / self.sec_per_row)))
        reps = np.resize(self.local, n)
        t0 = time.perf_counter()
        out = self.ds.gather_decompress(reps)
        dt = time.perf_counter() - t0
        assert np.array_equal(out[:64], self.oracle.gather_plain(self.X, reps[:64]))
        desc = (f"{n} row decodes over {self.n_groups} groups ({self.X.shape[0]} rows) of the {w.name} table, ids from its "
                f"batch sampler, {dt:.1f} s")
        return n * w.row_bytes / dt * 1e-9, n / dt, desc


def oracle_sample(w, seconds_target=12.0, thr=(1, 1)):
    return OracleSample(w, thr).run(seconds_target)


def parse_threshold(text):
    num, den = (int(t) for t in text.split("/"))
    return num, den


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload)
    smp = OracleSample(w, parse_threshold(args.threshold))
    per_step = max(0.2, min(10.0, 90.0 / max(1, args.steps + args.warmup)))
    vals, desc = [], ""
    for s in range(args.warmup + args.steps):
        gbps, rps, desc = smp.run(per_step)
        if s >= args.warmup:
            vals.append((gbps, rps))
    v = float(np.mean([x[0] for x in vals]))
    rows_per_step = w.batch_rows
    line = {
        "impl": "reference", "metric": "effective decompressed GB/s (gather-decompress)", "value": v, "unit": "GB/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": rows_per_step * w.row_bytes / (v * 1e9) * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": bench_config(w, parse_threshold(args.threshold)),
        "note": "CPU oracle (oracle/ibp_oracle.cpp, single thread) on a bounded sample per step; ms_per_step is the time a full batch would take at that rate",
        "cpu_baseline": {"value": v, "unit": "GB/s", "cores": 1, "kind": "oracle", "sample": "per step: " + desc, "rows_per_s": float(np.mean([x[1] for x in vals]))},
        "e2e": {"value": v, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------- CUDA arm
def read_hbm_peak():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"], "MEASURED_PEAKS.json hbm_gbs (copy; read+write bytes)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def traffic_from_profile(name, matches_capture):
    """roofline.traffic comes from the committed ncu summary of THIS kernel build, by file name, never from a literal here:
    profiles/r02_<workload>_decode_ncu.md carries lines `dram_bytes_per_launch: N`, `sysmem_bytes_per_launch: N`, `kernel: ...`,
    `commit: ...`.  Emitted only when the run matches the captured configuration (default alignment, store, order, dedup, no
    cache, strict codec); otherwise null."""
    path = os.path.join(ROOT, "profiles", f"r02_{name}_decode_ncu.md")
    if not matches_capture or not os.path.exists(path):
        return None, None, None
    vals = {}
    for line in open(path):
        for key in ("dram_bytes_per_launch", "sysmem_bytes_per_launch", "kernel", "commit"):
            if line.strip().startswith(key + ":"):
                vals[key] = line.split(":", 1)[1].strip()
    to_int = lambda k: int(vals[k].replace(",", "")) if k in vals else None
    return to_int("dram_bytes_per_launch"), to_int("sysmem_bytes_per_launch"), {"file": os.path.relpath(path, ROOT), "kernel": vals.get("kernel"), "commit": vals.get("commit")}


class Ctx:
    """Per-process measurement context: device, streams, ceilings measured once in this run."""

    def __init__(self, args):
        import torch
        import torch.distributed as dist
        from paper_2605_30728_b200 import binding as ibp
        import oracle
        self.torch, self.dist, self.ibp, self.oracle, self.args = torch, dist, ibp, oracle, args
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device; the IBP hot path has no CPU fallback")
        torch.cuda.set_device(self.local)
        if self.world > 1:
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
        self.stream = torch.cuda.current_stream().cuda_stream
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        self.h2d = ibp.ibp_measure_h2d(self.local, 1 << 30, 8)
        self.zc = ibp.ibp_measure_zero_copy_read(self.local, 1 << 30, 3)
        self.hbm_peak, self.hbm_src = read_hbm_peak()
        self.launches = 0

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            self.dist.barrier()
            self.torch.cuda.synchronize()

    def max_over_ranks(self, v):
        t = self.torch.tensor([float(v)], dtype=self.torch.float64, device="cuda")
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def timed_loop(self, fn, count, first):
        """count steps, CUDA events around each on the launch stream, L2 flushed (256 MiB write) between steps outside the events"""
        torch = self.torch
        evs = []
        for j in range(count):
            self.flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn(first + j)
            b.record()
            evs.append((a, b))
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]


def measure_gather(ctx, w, K, W, full, X=None, store="managed", keep=False):
    """One row- or span-gather workload end to end: build, parity of a warm-up batch against the plain definition, K timed steps
    (value), the e2e entry point, the uncompressed baseline.  `full` adds the resident decode, all baseline variants and the
    random-span ceiling.  Returns (entry dict, extras dict)."""
    torch, ibp, oracle, args = ctx.torch, ctx.ibp, ctx.oracle, ctx.args
    align = args.align if args.align else w.align_bytes
    thr = parse_threshold(args.threshold)
    shared = ctx.world > 1
    t0 = time.perf_counter()
    if X is None and (not shared or ctx.rank == 0):
        X = w.table()
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    if not shared:
        h = ibp.ibp_build(X, w.row_bytes, w.group_kind, w.group_param, align_bytes=align, index_span=w.index_span,
                          flags=ibp.IBP_FLAG_HOSTALLOC_STORE if store == "pinned" else 0, threshold=thr)
    else:
        # N > 1: ONE store in host memory for all ranks: rank 0 builds and exports it into a shared-memory segment
        # (pages interleaved over the NUMA nodes), every rank opens that segment and maps it for its own GPU
        name = f"/ibp_bench_{os.environ.get('MASTER_PORT', '0')}_{w.name}"
        if ctx.rank == 0:
            h0 = ibp.ibp_build(X, w.row_bytes, w.group_kind, w.group_param, align_bytes=align, index_span=w.index_span,
                               flags=ibp.IBP_FLAG_PAGEABLE_STORE, threshold=thr)
            h0.export_shared(name, numa_policy=1)
            h0.destroy()
        ctx.barrier()
        h = ibp.ibp_open_shared(name)
        ctx.barrier()
        if ctx.rank == 0:
            ibp.ibp_unlink_shared(name)
    t_build = time.perf_counter() - t0
    h.upload_metadata(ctx.local)
    if args.order is not None:
        h.set_order_mode(args.order)
    if args.decode_ctas:
        h.configure(args.decode_ctas, 0)
    dedup = args.dedup if args.dedup is not None else (0 if w.ids_unique else -1)
    h.set_dedup_mode(dedup)
    info = h.info()
    stream = ctx.stream
    cache = cinfo = None
    if full and args.cache_frac > 0:                           # S8f NEXT #3: compressed GPU cache in front of the store
        if w.index_span != 1 or not hasattr(w, "hot_ids"):
            raise SystemExit("bench.py --cache-frac needs a row-gather workload with a hot set (gnn, dlrm)")
        cache = ibp.Cache(h, int(info.packed_bytes_stored * args.cache_frac), 1, max_entries=max(1024, int(w.n_rows * min(1.0, 2 * args.cache_frac))))
        cache.insert(w.hot_ids(int(w.n_rows * min(1.0, 2 * args.cache_frac))), stream)
        cinfo = cache.info()

    n, n_rows_out = w.batch_ids, w.batch_rows
    batches = [w.ids(ctx.rank * 100_000 + i) for i in range(W + K)]
    ids_dev = [torch.from_numpy(b).cuda() for b in batches]
    out = torch.empty((n_rows_out, w.row_bytes), dtype=torch.uint8, device="cuda")
    hit_rate = None
    if cache is not None:                                      # only the misses cross PCIe: account the link bytes over them
        ent = torch.empty(n, dtype=torch.int64, device="cuda")
        link, hits = [], []
        for b, bd in zip(batches, ids_dev):
            cache.lookup(bd.data_ptr(), n, ent.data_ptr(), stream)
            torch.cuda.synchronize()
            miss = ent.cpu().numpy() == -1
            hits.append(1.0 - miss.mean())
            link.append(h.batch_link_bytes(b[miss]) if miss.any() else (1, 1, 1))
        hit_rate = float(np.mean(hits[W:]))
    else:
        link = [h.batch_link_bytes(b) for b in batches]        # (distinct ids, stored bytes, byte-aligned bytes)
    order_on = w.index_span == 1 and ((args.order == 1) or (args.order is None and info.packed_bytes_stored > (64 << 20) and n >= 4096))
    dedup_on = w.index_span == 1 and (dedup == 1 or (dedup < 0 and n >= 16384))
    launches_per_step = 1 + (3 if order_on else 0) + (2 if dedup_on else 0)

    def step(i):
        if cache is not None:
            cache.gather_decompress(ids_dev[i].data_ptr(), n, out.data_ptr(), stream)
        else:
            h.gather_decompress(ids_dev[i].data_ptr(), n, out.data_ptr(), stream)

    for i in range(W):
        step(i)
    torch.cuda.synchronize()
    # parity of one warm-up batch against the plain definition (oracle c1), so that a fast wrong kernel cannot score
    chk = np.random.default_rng(0).choice(n_rows_out, size=min(4096, n_rows_out), replace=False)
    got = out[torch.from_numpy(chk).cuda()].cpu().numpy()
    want = None
    if X is not None:                                           # N > 1: rank 0 holds the table (the others read the shared store only)
        want = oracle.gather_plain(X, batches[W - 1], w.index_span)[chk]
        if not np.array_equal(got, want):
            raise SystemExit(f"bench.py: GPU output differs from the oracle on {w.name}; refusing to report a number")

    clocks = ClockSampler(ctx.local)
    ctx.barrier()
    clocks.start()
    ms = ctx.timed_loop(step, K, W)
    ctx.barrier()
    clk = clocks.stop()
    ctx.launches += K * launches_per_step
    t_job = ctx.max_over_ranks(float(np.sum(ms)))
    world = ctx.world
    bytes_step = n_rows_out * w.row_bytes
    value = world * K * bytes_step / (t_job * 1e-3) * 1e-9

    sec = float(np.sum(ms)) * 1e-3
    uniq = float(np.sum([link[W + j][0] for j in range(K)]))
    stored = float(np.sum([link[W + j][1] for j in range(K)]))
    alg = float(np.sum([link[W + j][2] for j in range(K)]))
    raw_unique = uniq * w.index_span * w.row_bytes
    rep = K * n / uniq                                          # every repeat of a distinct id is delivered for free
    if cache is not None:
        roof_alg = roof_st = min(ctx.h2d * K * n * w.row_bytes / stored, ctx.hbm_peak)
    else:
        roof_alg = min(ctx.h2d * raw_unique / alg * rep, ctx.hbm_peak)
        roof_st = min(ctx.h2d * raw_unique / stored * rep, ctx.hbm_peak)

    # ---- e2e through the C ABI host entry point: pinned host ids in, pinned host rows out
    ids_pin = ibp.PinnedBuffer(n * 8)
    out_pin = ibp.PinnedBuffer(bytes_step)
    ids_pin_np = ids_pin.view(np.int64)
    out_pin_np = out_pin.view(np.uint8, (n_rows_out, w.row_bytes))
    ids_stage = torch.empty(n, dtype=torch.int64, device="cuda")
    ids_pin_t, out_pin_t = torch.from_numpy(ids_pin_np), torch.from_numpy(out_pin_np)

    def step_e2e(i):
        ids_pin_np[:] = batches[i]
        if cache is not None:                                   # no host entry point for the cache: the same copies through torch
            ids_stage.copy_(ids_pin_t, non_blocking=True)
            cache.gather_decompress(ids_stage.data_ptr(), n, out.data_ptr(), stream)
            out_pin_t.copy_(out, non_blocking=True)
            torch.cuda.current_stream().synchronize()
        else:
            h.gather_decompress_host(ids_pin_np, n, out_pin_np, stream)

    for i in range(min(W, 3)):
        step_e2e(i)
    if X is not None and not np.array_equal(out_pin_np[chk], oracle.gather_plain(X, batches[min(W, 3) - 1], w.index_span)[chk]):
        raise SystemExit(f"bench.py: end-to-end output differs from the oracle on {w.name}")
    ctx.barrier()
    Ke = max(3, min(K, 30 if full else 10))
    ms_e = ctx.timed_loop(step_e2e, Ke, W)
    ctx.barrier()
    e2e_value = world * Ke * bytes_step / (ctx.max_over_ranks(float(np.sum(ms_e))) * 1e-3) * 1e-9
    ids_pin.free(); out_pin.free()

    # ---- uncompressed zero-copy gather baseline (N=1 only): same ids, same timing
    base = None
    if world == 1 and not args.no_baseline:
        res = {}
        for kind in (("managed", "pinned") if full else ("managed",)):
            buf = ibp.PinnedBuffer(X.nbytes, managed=(kind == "managed"), device=ctx.local)
            buf.view(X.dtype, X.shape)[:] = X
            for order in ((False, True) if (w.index_span == 1 and full) else (False,)):
                def step_b(i, buf=buf, order=order):
                    ibp.ibp_gather_uncompressed(buf.dev_ptr, w.row_bytes * w.index_span, ids_dev[i].data_ptr(), n, out.data_ptr(), stream,
                                                n_rows=w.n_rows // w.index_span, locality_order=order)
                for i in range(3):
                    step_b(i)
                mb = ctx.timed_loop(step_b, min(K, 20 if full else 8), W)
                res[f"{kind}{'_ordered' if order else ''}"] = bytes_step / (float(np.mean(mb)) * 1e-3) * 1e-9
            buf.free()
        base = {"unit": "GB/s", "what": "ibp_gather_uncompressed: zero-copy gather of the raw rows (PAPER.md:329 'GPU (Aligned)')", **{k: round(v, 2) for k, v in res.items()}}

    kernel = ("ibp_stream_t_kernel" if info.thresholded else "ibp_stream_kernel") if w.index_span > 1 else "ibp_decode_kernel"
    entry = {
        "name": w.name, "workload": describe(w), "value": round(value, 3), "unit": "GB/s", "rows_per_s": round(world * K * n_rows_out / (t_job * 1e-3), 1),
        "ms_per_step": round(t_job / K, 5), "steps": K, "rows_per_step": n_rows_out, "row_bytes": w.row_bytes,
        "link_GBps_bytealigned": round(alg / sec * 1e-9, 3), "link_GBps_stored": round(stored / sec * 1e-9, 3),
        "frac_bytealigned": round(value / world / roof_alg, 4), "frac_stored": round(value / world / roof_st, 4),
        "roofline_GBps_bytealigned": round(roof_alg, 2), "roofline_GBps_stored": round(roof_st, 2),
        "ratio_bytealigned": round(w.n_rows * w.row_bytes / info.packed_bytes_bytealigned, 4), "ratio_stored": round(w.n_rows * w.row_bytes / info.packed_bytes_rows, 4),
        "align_bytes": info.align_bytes, "distinct_rows_per_s": round(uniq * w.index_span / sec), "kernel": kernel,
        "dedup": bool(dedup_on), "locality_order": bool(order_on),
        "e2e": {"value": round(e2e_value, 3), "unit": "GB/s", "h2d_bytes_per_step": n * 8, "d2h_bytes_per_step": bytes_step, "steps": Ke,
                "api": "ibp_gather_decompress_host (pinned host ids in, pinned host rows out)"},
        "baseline_uncompressed": base,
        "parity": f"bit-exact: {len(chk)} sampled output rows of one warm-up batch and of one e2e batch == oracle.gather_plain",
        "store": {0: "pageable", 1: "pinned (cudaHostAlloc)", 2: "managed host-resident (preferred CPU, accessed-by GPU)"}[info.store_kind],
        "packed_store_GB": round(info.packed_bytes_stored * 1e-9, 3), "metadata_MB": round(info.metadata_bytes * 1e-6, 2),
        "build_s": round(t_build, 2), "datagen_s": round(t_gen, 2), "gpu_launches": K * launches_per_step,
    }
    extras = {"info": info, "clk": clk, "stored_per_launch": stored / K, "alg_per_launch": alg / K, "uniq": uniq, "sec": sec, "order_on": order_on,
              "dedup_on": dedup_on, "launches_per_step": launches_per_step, "thr": thr, "hit_rate": hit_rate, "cinfo": cinfo, "Ke": Ke, "t_job": t_job}

    if full:
        # the same step with the store kind BASELINE.json's north_star names literally: cudaHostAlloc pinned memory
        if world == 1 and store != "pinned" and cache is None and not args.no_pinned_store:
            hp = ibp.ibp_build(X, w.row_bytes, w.group_kind, w.group_param, align_bytes=align, index_span=w.index_span,
                               flags=ibp.IBP_FLAG_HOSTALLOC_STORE, threshold=thr).upload_metadata(ctx.local)
            hp.set_dedup_mode(dedup)
            if args.decode_ctas:
                hp.configure(args.decode_ctas, 0)
            stp = lambda i: hp.gather_decompress(ids_dev[i].data_ptr(), n, out.data_ptr(), stream)
            for i in range(W):
                stp(i)
            torch.cuda.synchronize()
            if not np.array_equal(out[torch.from_numpy(chk).cuda()].cpu().numpy(), want):
                raise SystemExit("bench.py: pinned-store output differs from the oracle")
            mp_ = ctx.timed_loop(stp, K, W)
            ctx.launches += K * launches_per_step
            vp = bytes_step / (float(np.mean(mp_)) * 1e-3) * 1e-9
            extras["value_pinned_store"] = {"value": round(vp, 3), "unit": "GB/s", "ms_per_step": round(float(np.mean(mp_)), 5), "store": "pinned (cudaHostAlloc, mapped): IBP_FLAG_HOSTALLOC_STORE",
                                            "frac_bytealigned": round(vp / roof_alg, 4), "frac_stored": round(vp / roof_st, 4),
                                            "note": "same table, ids, steps and launch path as `value`; 4 KB GPU pages make address translation the limit for random rows (DESIGN.md section 6), which is why the managed host-resident store is the default"}
            hp.destroy()
        # random-row gathers: the same link read as random, span-aligned spans of about one packed row over a managed host
        # buffer as large as the packed store -- the measured ceiling of any random gather of rows this small on this box
        if w.index_span == 1 and ctx.rank == 0 and info.packed_bytes_stored >= (64 << 20):
            mean_row = info.packed_bytes_rows / w.n_rows
            span = 128 if mean_row <= 128 else 256 if mean_row <= 256 else 512
            sps, gbs = ibp.ibp_measure_random_read(ctx.local, int(min(info.packed_bytes_stored, 8 << 30)), span, 3)
            extras["rand_ceiling"] = {"span_bytes": span, "footprint_GB": round(min(info.packed_bytes_stored, 8 << 30) * 1e-9, 2),
                                      "spans_per_s": round(sps), "GBps": round(gbs, 2),
                                      "what": "ibp_measure_random_read: LSU 16-byte loads of span-aligned random spans, managed host-resident buffer"}
        # S8: resident decode (ibp_decompress_resident) of a contiguous range staged in HBM beforehand
        if world == 1 and not args.no_resident:
            G = w.group_param
            nr = min(w.n_rows, 1 << 20) // G * G
            ptr, nb = h.packed_range(0, nr)
            staged = torch.from_numpy(h.packed_view(ptr, nb).copy()).cuda()
            outr = torch.empty((nr, w.row_bytes), dtype=torch.uint8, device="cuda")
            step_r = lambda i: h.decompress_resident(staged.data_ptr(), 0, nr, outr.data_ptr(), stream)
            for i in range(3):
                step_r(i)
            torch.cuda.synchronize()
            if not np.array_equal(outr[:4096].cpu().numpy(), X[:4096].view(np.uint8).reshape(4096, -1)):
                raise SystemExit("bench.py: resident decode differs from the original rows")
            t_r = float(np.mean(ctx.timed_loop(step_r, 20, 0)))
            ctx.launches += 20
            meta_bytes = (nr // G) * 2 * w.row_bytes
            extras["resident"] = {"rows": nr, "ms": round(t_r, 4), "out_GBps": round(nr * w.row_bytes / (t_r * 1e-3) * 1e-9, 1),
                                  "in_plus_out_GBps": round((nb + nr * w.row_bytes) / (t_r * 1e-3) * 1e-9, 1), "bound": "hbm", "peak": ctx.hbm_peak,
                                  "frac": round((nb + nr * w.row_bytes + meta_bytes) / (t_r * 1e-3) * 1e-9 / ctx.hbm_peak, 4),
                                  "algorithmic_bytes": int(nb + nr * w.row_bytes + meta_bytes),
                                  "kernel": ("ibp_stream_t_kernel" if info.thresholded else "ibp_stream_kernel") + " (ibp_decompress_resident)",
                                  "what": "packed bytes of the first rows of the table staged in HBM, decoded to HBM; L2 flushed between launches"}
            del staged, outr
    if cache is not None:
        cache.destroy()
    h.destroy()
    del ids_dev, out
    if not keep:
        X = None
    torch.cuda.empty_cache()
    return entry, extras


def tiny_latency_breakdown(ctx, entry):
    """configs[0] is one wave of 1,024 rows: the step is a sum of dependent latencies, not a bandwidth.
    Measured here: an event pair around an empty stream, a one-row zero-copy gather (launch + one PCIe round trip), the link
    time of the batch's packed bytes at the zero-copy ceiling."""
    torch, ibp = ctx.torch, ctx.ibp
    evs = []
    for _ in range(50):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); b.record(); evs.append((a, b))
    torch.cuda.synchronize()
    ev_us = float(np.median([a.elapsed_time(b) for a, b in evs])) * 1e3
    buf = ibp.PinnedBuffer(1 << 20, managed=True, device=ctx.local)
    ids1 = torch.zeros(1, dtype=torch.int64, device="cuda")
    o1 = torch.zeros(512, dtype=torch.uint8, device="cuda")
    one = lambda i: ibp.ibp_gather_uncompressed(buf.dev_ptr, 512, ids1.data_ptr(), 1, o1.data_ptr(), ctx.stream)
    for i in range(5):
        one(i)
    t1 = float(np.median(ctx.timed_loop(one, 30, 0))) * 1e3
    buf.free()
    link_us = entry["rows_per_step"] * entry["row_bytes"] / entry["ratio_stored"] / (ctx.zc * 1e9) * 1e6
    return {"step_us": round(entry["ms_per_step"] * 1e3, 2), "event_pair_on_an_idle_stream_us": round(ev_us, 2),
            "one_row_zero_copy_gather_us (launch + id load + one PCIe round trip + store)": round(t1, 2),
            "link_time_of_the_batch_at_the_zero_copy_ceiling_us": round(link_us, 2),
            "note": "a latency floor, not a kernel property: fetch engine, rows in flight, warps per CTA and store kind all give the same step time (DESIGN.md section 8)"}


def resident_thresholded(ctx, name, thr, steps=20):
    """ibp_decompress_resident of the first 2^20 rows of a workload's table built with tau = thr (the paper's codec): packed
    bytes staged in HBM, every decoded byte checked against the original rows, L2 flushed between the timed launches."""
    import oracle
    torch = ctx.torch
    ibp = ctx.ibp
    w = make_workload(name)
    nr = min(w.n_rows, 1 << 20) // w.group_param * w.group_param
    Xb = w.rows(0, nr).view(np.uint8).reshape(nr, -1)
    h = ibp.ibp_build(Xb, w.row_bytes, w.group_kind, w.group_param, align_bytes=w.align_bytes, threshold=thr, flags=ibp.IBP_FLAG_PAGEABLE_STORE).upload_metadata(ctx.local)
    info = h.info()
    stream = torch.cuda.current_stream().cuda_stream
    ptr, nb = h.packed_range(0, nr)
    staged = torch.from_numpy(h.packed_view(ptr, nb).copy()).cuda()
    out = torch.empty((nr, w.row_bytes), dtype=torch.uint8, device="cuda")
    step = lambda i: h.decompress_resident(staged.data_ptr(), 0, nr, out.data_ptr(), stream)
    for i in range(3):
        step(i)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    if not np.array_equal(got, Xb):
        raise SystemExit(f"bench.py: thresholded resident decode of {name} differs from the original rows")
    n_or = min(nr, 1 << 16) // w.group_param * w.group_param                            # the oracle's codec on the first 65,536 rows
    ids = np.random.default_rng(0).choice(n_or, 64, replace=False)
    ds = oracle.DatasetT(Xb[:n_or], w.group_kind, w.group_param, thr[0], thr[1])
    ok = np.array_equal(got[ids], ds.gather_decompress(ids))
    ds.close()
    if not ok:
        raise SystemExit(f"bench.py: thresholded resident decode of {name} differs from the oracle codec")
    t = float(np.mean(ctx.timed_loop(step, steps, 0)))
    ctx.launches += steps
    alg = nb + nr * w.row_bytes + info.n_groups * 2 * w.row_bytes
    e = {"workload": name, "rows": nr, "threshold": f"{thr[0]}/{thr[1]}", "ms": round(t, 4), "in_plus_out_GBps": round((nb + nr * w.row_bytes) / (t * 1e-3) * 1e-9, 1),
         "bound": "hbm", "peak": ctx.hbm_peak, "frac": round(alg / (t * 1e-3) * 1e-9 / ctx.hbm_peak, 4), "algorithmic_bytes": int(alg),
         "ratio_stored": round(nr * w.row_bytes / nb, 3), "rows_kept_raw": int(info.n_rows_raw), "kernel": "ibp_stream_t2_kernel (ibp_decompress_resident)",
         "parity": "every byte == the original rows; 64 sampled rows == the oracle's thresholded codec"}
    h.destroy()
    del staged, out
    return e


def run_cuda(args):
    ctx = Ctx(args)
    torch, ibp = ctx.torch, ctx.ibp
    W, K = max(3, args.warmup), args.steps
    w = make_workload(args.workload)
    entry, ex = measure_gather(ctx, w, K, W, full=True, store=args.store)
    info, thr = ex["info"], ex["thr"]
    world = ctx.world

    per_config = None
    if world == 1 and args.workload == "gnn" and not args.no_per_config and args.cache_frac == 0 and args.threshold == "1/1" and not args.align and args.store == "managed":
        Kc = max(3, min(K, 20))
        per_config = []
        for name in ("tiny", "gnn", "dlrm", "kv", "weights"):
            if name == "gnn":
                e = dict(entry)
            elif name == "weights":
                e = measure_weights(ctx, args, Kc, W, layers=args.layers, overlap=False, cpu=False)[0]
            else:
                e, _ = measure_gather(ctx, make_workload(name), Kc, W, full=False)
                if name == "tiny":
                    e["latency_breakdown"] = tiny_latency_breakdown(ctx, e)
            per_config.append(e)

    # S8 under the paper's own codec (tau = 4/5): resident decode of the first 2^20 rows of the three row-shaped configs
    resident_t = None
    if per_config is not None and not args.no_resident:
        resident_t = [resident_thresholded(ctx, name, (4, 5)) for name in ("gnn", "dlrm", "kv")]

    cpu = None
    if ctx.rank == 0 and world == 1 and not args.no_cpu:
        g, rps, desc = oracle_sample(w, seconds_target=12.0, thr=thr)
        cpu = {"value": round(g, 5), "unit": "GB/s", "cores": 1, "kind": "oracle", "sample": desc, "rows_per_s": round(rps, 1)}

    if ctx.rank == 0:
        default_cfg = (not args.align and args.store == "managed" and args.order is None and args.dedup is None and args.cache_frac == 0
                       and not info.thresholded and not getattr(w, "interleaved", False) and not args.decode_ctas)
        dram, sysmem, prof = traffic_from_profile(w.name, default_cfg)
        achieved = ex["alg_per_launch"] * K / ex["sec"] * 1e-9
        achieved_st = ex["stored_per_launch"] * K / ex["sec"] * 1e-9
        cinfo = ex["cinfo"]
        line = {
            "metric": "effective decompressed GB/s (gather-decompress)", "value": entry["value"], "unit": "GB/s",
            "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": entry["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic", "rows_per_s": entry["rows_per_s"],
            "config": bench_config(w, thr),
            "setup": {
                "align_bytes": info.align_bytes, "store": entry["store"], "locality_order": ex["order_on"], "dedup": ex["dedup_on"],
                "ids_unique_by_construction": bool(w.ids_unique),
                "l2": "flushed with a 256 MiB write between steps (outside the events); ids differ every step; the packed store is host memory and is never cached",
                "cache": None if cinfo is None else {"what": "compressed GPU software cache (P:349-357) holding the hottest rows of the sampler, static fill", "capacity_frac_of_packed_store": args.cache_frac,
                                                      "capacity_MB": round(cinfo.capacity_bytes * 1e-6, 1), "used_MB": round(cinfo.used_bytes * 1e-6, 1), "entries": cinfo.n_entries, "map_MB": round(cinfo.map_bytes * 1e-6, 1),
                                                      "hit_rate": round(ex["hit_rate"], 4), "equivalent_uncompressed_cache_rows": int(cinfo.capacity_bytes // w.row_bytes)},
                "ratio_stored": entry["ratio_stored"], "ratio_bytealigned": entry["ratio_bytealigned"],
                "packed_store_GB": entry["packed_store_GB"], "metadata_MB": entry["metadata_MB"], "build_s": entry["build_s"], "datagen_s": entry["datagen_s"],
                "n_rows_raw": int(info.n_rows_raw),
                "sharding": "ids sharded over ranks, no collective; ONE store in host memory (POSIX shared memory, pages interleaved over the NUMA nodes) read by every rank's GPU over its own PCIe link" if world > 1 else "single GPU",
            },
            "roofline": {
                "bound": "pcie", "achieved": round(achieved, 3), "peak": round(ctx.h2d, 3), "unit": "GB/s", "frac": round(achieved / ctx.h2d, 4),
                "achieved_def": "ALGORITHMIC link bytes of the launch = sum over the batch's distinct rows of ceil(k_g/8) (SURVEY 8(d)), / event-timed duration",
                "traffic": dram, "traffic_sysmem": sysmem, "traffic_from_profile": prof,
                "kernel": entry["kernel"], "peak_source": "cudaMemcpyAsync H2D of 1 GiB from pinned memory, best of 8, this run (ibp_measure_h2d)",
                "algorithmic_bytes_per_launch": int(ex["alg_per_launch"]),
                "stored_bytes_per_launch": int(ex["stored_per_launch"]), "achieved_stored": round(achieved_st, 3), "frac_stored": round(achieved_st / ctx.h2d, 4),
                "frac_stored_def": f"the same with each row rounded up to the declared alignment unit A = {info.align_bytes} B: what the layout stores and the kernel fetches",
                "zero_copy_read_ceiling": round(ctx.zc, 3), "frac_of_zero_copy_ceiling": round(achieved / ctx.zc, 4), "frac_stored_of_zero_copy_ceiling": round(achieved_st / ctx.zc, 4),
                "random_span_ceiling": ex.get("rand_ceiling"), "distinct_rows_per_s": entry["distinct_rows_per_s"],
                "effective_roofline_GBps": entry["roofline_GBps_bytealigned"], "frac_of_effective_roofline": entry["frac_bytealigned"],
                "effective_roofline_def": "min(H2D ceiling x raw bytes / byte-aligned packed bytes of the batch's distinct rows, HBM peak): BASELINE.json's min(PCIe x ratio, HBM) with the codec's own ratio",
                "effective_roofline_stored_GBps": entry["roofline_GBps_stored"], "frac_of_effective_roofline_stored": entry["frac_stored"],
                "hbm_peak": ctx.hbm_peak, "hbm_peak_source": ctx.hbm_src,
            },
            "e2e": entry["e2e"],
            "value_pinned_store": ex.get("value_pinned_store"),
            "gpu_launches": ctx.launches,
            "clocks": ex["clk"],
            "resident_decode": ex.get("resident"),
            "resident_decode_thresholded": resident_t,
            "baseline_uncompressed": entry["baseline_uncompressed"],
            "per_config": per_config,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        ctx.dist.destroy_process_group()


def bench_config(w, thr):
    """`config` of the JSON line: the same keys and values in the CUDA arm and in the --impl reference arm."""
    return {"workload": describe(w), "rows_per_step": w.batch_rows, "row_bytes": w.row_bytes,
            "codec": "group-strict (tau = 1)" if thr[0] == thr[1] else f"thresholded, tau = {thr[0]}/{thr[1]} per group, 4-byte chunks, participation bits"}


# ------------------------------------------------------------------------------------------------- weight streaming
WEIGHTS_DESC = ("configs[4] LLM weight streaming: bf16 N(0,0.02) matrices of a 7B-shaped decoder, 4 x 4096x4096 + 3 x 4096x11008 per layer, "
                "{L} layers in host memory ({gb:.2f} GB raw), groups = 128-column tiles (strided); one step = one whole layer "
                "(ONE launch: ibp_decode_ranges over the layer's 7 matrices, {mb:.1f} MB out)")


def measure_weights(ctx, args, K, W, layers, overlap, cpu):
    """BASELINE configs[4]: bf16 matrices of a 7B-shaped decoder held packed in host memory; one step = one whole layer
    streamed in order by ONE launch (ibp_decode_ranges over its 7 handles); with the overlap harness (S7), layer l+1's fetch
    against a consumer GEMM ([M,4096] activation x the 7 matrices) on layer l, every overlapped step checked."""
    torch, ibp, oracle = ctx.torch, ctx.ibp, ctx.oracle
    from paper_2605_30728_b200 import workloads
    from paper_2605_30728_b200.overlap import DoubleBufferedPipeline, summarize
    L = layers
    t0 = time.perf_counter()
    hs, raw_bytes, stored, bytealigned = [], 0, 0, 0
    keep_raw = {}                                               # raw matrices of a few layers, for the parity checks
    check_layers = sorted({0, L - 1, min(L - 1, 2), min(L - 1, W + 1)})
    for l in range(L):
        mats = []
        for wm in workloads.weight_layer(l):
            X = wm.table()
            h = ibp.ibp_build(X, 256, 1, wm.group_param, align_bytes=args.align if args.align else 16,
                              flags=ibp.IBP_FLAG_HOSTALLOC_STORE if args.store == "pinned" else 0,
                              threshold=parse_threshold(args.threshold)).upload_metadata(ctx.local)
            if args.decode_ctas:
                h.configure(args.decode_ctas, 0)
            info = h.info()
            raw_bytes += X.nbytes; stored += info.packed_bytes_rows; bytealigned += info.packed_bytes_bytealigned
            mats.append((h, wm.n_rows, wm.mat_rows, wm.mat_cols))
            if l in check_layers:
                keep_raw.setdefault(l, []).append(X.view(np.uint8).reshape(wm.n_rows, -1).copy())
        hs.append(mats)
    t_build = time.perf_counter() - t0
    layer_rows = sum(m[1] for m in hs[0])
    layer_bytes = layer_rows * 256
    bufs = [torch.empty((layer_rows, 256), dtype=torch.uint8, device="cuda") for _ in range(2)]
    stream = ctx.stream

    def ranges_of(l, base_ptr, packed=None):
        rs, off = [], 0
        for j, (h, n_rows, _, _) in enumerate(hs[l]):
            rs.append((h, None if packed is None else packed[j], 0, n_rows, base_ptr + off * 256))
            off += n_rows
        return rs

    def fetch(i, bi, stream_ptr):
        ibp.ibp_decode_ranges(ranges_of(i % L, bufs[bi].data_ptr()), stream_ptr)

    def check_layer(buf, l, what):
        want = np.concatenate(keep_raw[l])
        if not np.array_equal(buf.cpu().numpy(), want):
            raise SystemExit(f"bench.py: {what}: streamed layer {l} differs from the original matrices")

    for i in range(W):
        fetch(i, 0, stream)
    for l in check_layers:                                      # (c1) every byte of whole layers
        fetch(l, 1, stream)
        torch.cuda.synchronize()
        check_layer(bufs[1], l, "range gather")
    clocks = ClockSampler(ctx.local)
    clocks.start()
    ms = ctx.timed_loop(lambda i: fetch(i, i % 2, stream), K, W)
    clk = clocks.stop()
    ctx.launches += K
    t_step = float(np.mean(ms))
    value = layer_bytes / (t_step * 1e-3) * 1e-9
    stored_layer, alg_layer = stored / L, bytealigned / L

    # ---- S8: a layer decoded from HBM (packed bytes staged once, outside the timing), one launch per layer
    l0 = check_layers[0]
    staged = []
    for (h, n_rows, _, _) in hs[l0]:
        ptr, nb = h.packed_range(0, n_rows)
        staged.append((torch.from_numpy(h.packed_view(ptr, nb).copy()).cuda(), nb))
    res_ranges = ranges_of(l0, bufs[0].data_ptr(), [s_[0].data_ptr() for s_ in staged])
    resident = lambda i: ibp.ibp_decode_ranges(res_ranges, stream)
    for i in range(3):
        resident(i)
    torch.cuda.synchronize()
    check_layer(bufs[0], l0, "resident decode")
    t_res = float(np.mean(ctx.timed_loop(resident, 10, 0)))
    ctx.launches += 10
    meta_layer = sum(2 * 256 * (c // 128) for (_, _, _, c) in hs[l0])
    res_bytes = sum(s_[1] for s_ in staged) + layer_bytes + meta_layer
    del staged

    # ---- e2e: the layer into pinned HOST memory through the host entry point (7 calls, synchronous)
    out_pin = ibp.PinnedBuffer(layer_bytes)
    out_pin_np = out_pin.view(np.uint8, (layer_rows, 256))

    def step_e2e(i):
        rs, off = [], 0
        for (h, n_rows, _, _) in hs[i % L]:
            rs.append((h, None, 0, n_rows, out_pin_np[off:off + n_rows]))
            off += n_rows
        ibp.ibp_decode_ranges_host(rs, stream)                     # host destinations; synchronises the stream

    step_e2e(check_layers[-1])
    if not np.array_equal(out_pin_np, np.concatenate(keep_raw[check_layers[-1]])):
        raise SystemExit("bench.py: weights e2e output differs from the original matrices")
    Ke = max(3, min(K, 8))
    ms_e = ctx.timed_loop(step_e2e, Ke, W)
    e2e_value = layer_bytes / (float(np.mean(ms_e)) * 1e-3) * 1e-9
    out_pin.free()

    entry = {
        "name": "weights", "workload": WEIGHTS_DESC.format(L=L, gb=raw_bytes * 1e-9, mb=layer_bytes * 1e-6), "value": round(value, 3), "unit": "GB/s",
        "rows_per_s": round(layer_rows / (t_step * 1e-3), 1), "ms_per_step": round(t_step, 5), "steps": K, "rows_per_step": layer_rows, "row_bytes": 256, "layers": L,
        "link_GBps_bytealigned": round(alg_layer / (t_step * 1e-3) * 1e-9, 3), "link_GBps_stored": round(stored_layer / (t_step * 1e-3) * 1e-9, 3),
        "frac_bytealigned": round(value / min(ctx.h2d * raw_bytes / bytealigned, ctx.hbm_peak), 4), "frac_stored": round(value / min(ctx.h2d * raw_bytes / stored, ctx.hbm_peak), 4),
        "roofline_GBps_bytealigned": round(ctx.h2d * raw_bytes / bytealigned, 2), "roofline_GBps_stored": round(ctx.h2d * raw_bytes / stored, 2),
        "ratio_bytealigned": round(raw_bytes / bytealigned, 4), "ratio_stored": round(raw_bytes / stored, 4), "align_bytes": args.align if args.align else 16,
        "kernel": "ibp_stream_kernel (one launch per layer)",
        "e2e": {"value": round(e2e_value, 3), "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": layer_bytes, "steps": Ke,
                "api": "ibp_decode_ranges_host over the layer's 7 matrices (the packed rows are read in place from the host store; the decoded layer lands in pinned host memory; one launch, one synchronisation)"},
        "baseline_uncompressed": None,
        "resident_decode": {"ms_per_layer": round(t_res, 4), "in_plus_out_GBps": round(res_bytes / (t_res * 1e-3) * 1e-9, 1), "out_GBps": round(layer_bytes / (t_res * 1e-3) * 1e-9, 1),
                            "bound": "hbm", "peak": ctx.hbm_peak, "frac": round(res_bytes / (t_res * 1e-3) * 1e-9 / ctx.hbm_peak, 4), "launches_per_layer": 1,
                            "kernel": "ibp_stream_kernel (ibp_decode_ranges, resident, tile-block chunks)"},
        "parity": f"bit-exact: every byte of layers {check_layers} (range gather), of layer {l0} (resident) and of layer {check_layers[-1]} (e2e) == the original matrices (oracle c1)",
        "store": args.store, "build_s": round(t_build, 1), "gpu_launches": K,
    }
    extras = {"clk": clk, "stored_layer": stored_layer, "alg_layer": alg_layer, "raw_bytes": raw_bytes, "stored": stored, "bytealigned": bytealigned, "t_step": t_step}

    if overlap:
        # ---- S7: overlap with a consumer GEMM on the previous layer; EVERY overlapped step's buffer is checked: the consumer
        # folds the buffer into a per-step 64-bit checksum (sum of its int64 words) next to the GEMMs, and the sums of the layers
        # whose raw matrices were kept are compared with the originals'; a whole-buffer copy is compared for the kept layers.
        M = args.gemm_m
        act = torch.randn((M, 4096), dtype=torch.bfloat16, device="cuda")
        shapes = [(m[2], m[3]) for m in hs[0]]
        outs = [torch.empty((M, c), dtype=torch.bfloat16, device="cuda") for (_, c) in shapes]
        n_pipe = min(max(K, 8), 16)
        sums = torch.zeros(n_pipe, dtype=torch.int64, device="cuda")
        kept = {i: torch.empty_like(bufs[0]) for i in range(n_pipe) if (i % L) in keep_raw}
        check_on = [True]

        def consume(i, bi):
            off = 0
            for j, (r, c) in enumerate(shapes):
                wmat = bufs[bi][off:off + r * (c // 128)].view(torch.bfloat16).view(r, c)
                torch.matmul(act, wmat, out=outs[j])
                off += r * (c // 128)
            if check_on[0]:
                sums[i] = bufs[bi].view(torch.int64).sum()
                if i in kept:
                    kept[i].copy_(bufs[bi])

        pipe = DoubleBufferedPipeline(fetch, consume, n_pipe)
        for _ in range(2):
            pipe.run_overlapped()
        torch.cuda.synchronize()
        got_sums = sums.cpu().numpy()
        ref = {}
        for i in range(n_pipe):                                 # reference checksums from a serial fetch of the same layer
            l = i % L
            if l not in ref:
                fetch(l, 0, stream)
                ref[l] = int(bufs[0].view(torch.int64).sum().item())
            if int(got_sums[i]) != ref[l]:
                raise SystemExit(f"bench.py: overlapped step {i}: the consumer read a stale or half-written buffer")
        for i, t in kept.items():
            check_layer(t, i % L, f"overlapped step {i}")
        check_on[0] = False                                     # timing runs: the consumer is the GEMMs alone
        ov = summarize(pipe.run_fetch_only(), pipe.run_consume_only(), pipe.run_serial(), pipe.run_overlapped())
        ov.update({"steps": n_pipe, "consumer": f"torch.matmul [M={M},4096] bf16 x the 7 decoded matrices of the previous layer (cuBLAS)",
                   "decode_ctas": args.decode_ctas or "library default (host-store streams: 48 CTAs)",
                   "checked": f"all {n_pipe} overlapped steps: 64-bit checksum of the consumed buffer == that of a serial fetch of the same layer; whole-buffer bytes == the original matrices for steps {sorted(kept)}"})
        extras["overlap"] = ov
    if cpu:
        wm = workloads.WeightMatrix(1024, 4096, 0, 0)           # the first 1024 rows of layer 0's first matrix: same tiles, same values
        Xs = wm.table()
        ds = oracle.Dataset(Xs, 1, wm.group_param)
        sid = np.arange(wm.n_rows, dtype=np.int64)
        t0 = time.perf_counter()
        done = 0
        while time.perf_counter() - t0 < 10.0:
            o = ds.gather_decompress(sid)
            done += len(sid)
        dt = time.perf_counter() - t0
        assert np.array_equal(o, Xs.view(np.uint8).reshape(wm.n_rows, -1))
        ds.close()
        extras["cpu"] = {"value": round(done * 256 / dt * 1e-9, 5), "unit": "GB/s", "cores": 1, "kind": "oracle", "rows_per_s": round(done / dt, 1),
                         "sample": f"{done} row decodes by the oracle codec over the first 1024 matrix rows of layer 0's first 4096x4096 matrix (strided groups = 32 column tiles), {dt:.1f} s"}
    for mats in hs:
        for m in mats:
            m[0].destroy()
    del bufs
    torch.cuda.empty_cache()
    return entry, extras


def run_weights(args):
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py --workload weights runs on one GPU")
    ctx = Ctx(args)
    W, K = max(3, args.warmup), args.steps
    entry, ex = measure_weights(ctx, args, K, W, layers=args.layers, overlap=True, cpu=not args.no_cpu)
    L = args.layers
    achieved = ex["alg_layer"] / (ex["t_step"] * 1e-3) * 1e-9
    achieved_st = ex["stored_layer"] / (ex["t_step"] * 1e-3) * 1e-9
    line = {
        "metric": "effective decompressed GB/s (gather-decompress)", "value": entry["value"], "unit": "GB/s", "n_gpus": 1,
        "steps": K, "warmup": W, "ms_per_step": entry["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic", "rows_per_s": entry["rows_per_s"],
        "config": {"workload": entry["workload"], "rows_per_step": entry["rows_per_step"], "row_bytes": 256, "codec": "group-strict (tau = 1)" if args.threshold == "1/1" else f"thresholded, tau = {args.threshold}"},
        "setup": {"align_bytes": entry["align_bytes"], "store": args.store, "ratio_stored": entry["ratio_stored"], "ratio_bytealigned": entry["ratio_bytealigned"], "build_s": entry["build_s"],
                  "layers": L, "l2": "flushed with a 256 MiB write between steps (outside the events)"},
        "roofline": {"bound": "pcie", "achieved": round(achieved, 3), "peak": round(ctx.h2d, 3), "unit": "GB/s", "frac": round(achieved / ctx.h2d, 4), "traffic": None,
                     "kernel": "ibp_stream_kernel", "algorithmic_bytes_per_launch": int(ex["alg_layer"]), "stored_bytes_per_launch": int(ex["stored_layer"]),
                     "achieved_stored": round(achieved_st, 3), "frac_stored": round(achieved_st / ctx.h2d, 4),
                     "zero_copy_read_ceiling": round(ctx.zc, 3), "frac_of_zero_copy_ceiling": round(achieved / ctx.zc, 4),
                     "effective_roofline_GBps": entry["roofline_GBps_bytealigned"], "frac_of_effective_roofline": entry["frac_bytealigned"],
                     "effective_roofline_stored_GBps": entry["roofline_GBps_stored"], "frac_of_effective_roofline_stored": entry["frac_stored"]},
        "resident_decode": entry["resident_decode"],
        "overlap": ex.get("overlap"),
        "e2e": entry["e2e"],
        "gpu_launches": ctx.launches, "clocks": ex["clk"], "parity": entry["parity"],
        "cpu_baseline": ex.get("cpu"),
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------- Fig. 7 sweep
def run_sweep(args):
    """PAPER.md:399-401 (Fig. 7): decompression throughput versus space savings with synthetic masks, 100,000 tensors of
    256 B / 1 KB / 4 KB, every tensor fetched once in random order, normalised to a "mock" that moves the compressed bytes
    across PCIe without decoding (here: ibp_gather_uncompressed over the packed store with row size = packed stride)."""
    import torch
    from paper_2605_30728_b200 import binding as ibp, workloads
    import oracle

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py --workload sweep runs on one GPU")
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    W, K = max(3, args.warmup), max(5, min(args.steps, 20))
    h2d_ceiling = ibp.ibp_measure_h2d(0, 1 << 30, 8)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    points, launches = [], 0
    clocks = ClockSampler(0)
    clocks.start()
    for rb in (256, 1024, 4096):
        for sv in (0.1, 0.3, 0.5, 0.7, 0.9, 0.95):
            w = workloads.Sweep(row_bytes=rb, savings=sv)
            X = w.table()
            h = ibp.ibp_build(X, rb, 0, w.group_param, align_bytes=args.align if args.align else 32).upload_metadata(0)
            h.set_dedup_mode(0)                                  # every row exactly once
            info = h.info()
            stride = info.max_row_stride
            n = w.n_rows
            ids = [torch.from_numpy(w.ids(i)).cuda() for i in range(W + K)]
            out = torch.empty((n, rb), dtype=torch.uint8, device="cuda")
            store_dev = h.store_device_ptr()

            def timed(fn):
                for i in range(W):
                    fn(i)
                evs = []
                for j in range(K):
                    flush.zero_()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(); fn(W + j); b.record()
                    evs.append((a, b))
                torch.cuda.synchronize()
                return float(np.mean([a.elapsed_time(b) for a, b in evs]))

            t_ibp = timed(lambda i: h.gather_decompress(ids[i].data_ptr(), n, out.data_ptr(), stream))
            got = out[:2048].cpu().numpy()
            if not np.array_equal(got, oracle.gather_plain(X, w.ids(W + K - 1)[:2048])):
                raise SystemExit("bench.py: sweep output differs from the oracle")
            t_mock = timed(lambda i: ibp.ibp_gather_uncompressed(store_dev, stride, ids[i].data_ptr(), n, out.data_ptr(), stream, n_rows=n, locality_order=True))
            launches += 2 * K
            points.append({"row_bytes": rb, "space_saved_target": sv, "space_saved_stored": round(1 - stride / rb, 4), "packed_stride": stride,
                           "ibp_ms": round(t_ibp, 4), "mock_ms": round(t_mock, 4), "ibp_effective_GBps": round(n * rb / (t_ibp * 1e-3) * 1e-9, 2),
                           "link_GBps": round(n * stride / (t_ibp * 1e-3) * 1e-9, 2), "frac_of_mock": round(t_mock / t_ibp, 4),
                           "frac_of_pcie_ceiling": round(n * stride / (t_ibp * 1e-3) * 1e-9 / h2d_ceiling, 4)})
            h.destroy()
            del out, ids
    clk = clocks.stop()
    ref = [p_ for p_ in points if p_["row_bytes"] == 1024 and p_["space_saved_target"] == 0.5][0]
    line = {"metric": "effective decompressed GB/s (gather-decompress)", "value": ref["ibp_effective_GBps"], "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": W,
            "ms_per_step": ref["ibp_ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": "PAPER.md:399-401 (Fig. 7) sweep: 100,000 tensors of 256 B / 1 KB / 4 KB, synthetic Mask with a chosen popcount, uniformly random variant bits, one global group, every tensor fetched once in random order; value = the 1 KB / 50 % point",
                       "mock": "ibp_gather_uncompressed over the packed store (moves the compressed bytes, no decode), locality-ordered like the IBP gather",
                       "paper_curve": "P:401 on A100/PCIe Gen4: >= 95 % of the mock below 50 % savings; at 90 % savings 78 % (1 KB), 86 % (4 KB), about 50 % (256 B)",
                       "l2": "flushed with a 256 MiB write between steps"},
            "roofline": {"bound": "pcie", "achieved": ref["link_GBps"], "peak": round(h2d_ceiling, 3), "unit": "GB/s", "frac": ref["frac_of_pcie_ceiling"], "traffic": None, "kernel": "ibp_decode_kernel"},
            "sweep": points, "e2e": {"value": None, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": launches, "clocks": clk, "cpu_baseline": None}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------- GPU-side compressor
def run_build(args):
    """ibp_build_device on the workload's table, rows resident in HBM, the
    packed store written in place into host memory over PCIe.  One step = one whole build (mask kernel, [size kernel, scan,]
    pack kernel).  Kernel times are CUDA events recorded inside the library around each kernel (ibp_get_build_stats)."""
    import torch
    from paper_2605_30728_b200 import binding as ibp
    import oracle

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py --phase build runs on one GPU")
    torch.cuda.set_device(0)
    w = make_workload(args.workload)
    thr = parse_threshold(args.threshold)
    align = args.align if args.align else w.align_bytes
    X = w.table()
    Xb = X.view(np.uint8).reshape(w.n_rows, -1)
    xd = torch.from_numpy(Xb).cuda()
    stream = torch.cuda.current_stream().cuda_stream
    flags = ibp.IBP_FLAG_HOSTALLOC_STORE if args.store == "pinned" else 0
    W, K = min(max(1, args.warmup), 2), max(1, min(args.steps, 5))
    d2h_ceiling = ibp.ibp_measure_d2h(0, 1 << 30, 8)
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        hbm_peak = 6650.0

    def build():
        return ibp.ibp_build_device(xd.data_ptr(), w.n_rows, w.row_bytes, w.group_kind, w.group_param, align_bytes=align,
                                    index_span=w.index_span, flags=flags, threshold=thr, stream=stream)

    # parity of a sample against the oracle (groups are independent: the oracle compresses the sampled groups alone)
    h = build()
    G = w.group_param
    rng = np.random.default_rng(0)
    for g in rng.choice(w.n_rows // G, 6, replace=False):
        blk = Xb[g * G:(g + 1) * G]
        m, b, k = h.metadata_host(int(g))
        if thr[0] == thr[1]:
            ds = oracle.Dataset(blk, 0, G)
            ok = np.array_equal(m, ds.mask(0)) and np.array_equal(b, ds.bitval(0)) and k == ds.k_bits(0)
            for r in range(0, G, 7):
                data, _ = h.packed_row(int(g) * G + r)
                want = ds.packed_row(r)
                ok = ok and np.array_equal(data[:want.size], want) and not data[want.size:].any()
        else:
            ds = oracle.DatasetT(blk, 0, G, thr[0], thr[1])
            ok = np.array_equal(m, ds.mask(0)) and np.array_equal(b, ds.bitval(0))
            for r in range(0, G, 7):
                data, stored, comp = h.row_info(int(g) * G + r)
                want, want_comp = ds.row(r)
                ok = ok and comp == want_comp and np.array_equal(data, want)
        ds.close()
        if not ok:
            raise SystemExit("bench.py: the GPU-built store differs from the oracle; refusing to report a number")
    info = h.info()
    h.destroy()
    for _ in range(W - 1):
        build().destroy()
    clocks = ClockSampler(0)
    clocks.start()
    stats = []
    for _ in range(K):
        h = build()
        stats.append(h.build_stats())
        h.destroy()
    clk = clocks.stop()
    mean = lambda f: float(np.mean([getattr(s_, f) for s_ in stats]))
    raw = stats[0].raw_bytes
    k_ms = mean("mask_ms") + mean("size_ms") + mean("scan_ms") + mean("pack_ms")
    # host compressor (ibp_build, all cores) and the oracle's compressor (1 core, sample of groups) for comparison
    t0 = time.perf_counter()
    hh = ibp.ibp_build(Xb, w.row_bytes, w.group_kind, w.group_param, align_bytes=align, index_span=w.index_span, flags=flags, threshold=thr)
    t_host = time.perf_counter() - t0
    hh.destroy()
    cpu = None
    if not args.no_cpu:
        ng_s = 1
        t0 = time.perf_counter()
        done = 0
        while time.perf_counter() - t0 < 10.0:
            blk = Xb[done * G:(done + ng_s) * G]
            (oracle.Dataset(blk, 0, G) if thr[0] == thr[1] else oracle.DatasetT(blk, 0, G, thr[0], thr[1])).close()
            done += ng_s
            ng_s = min(ng_s * 2, 64)
        dt = time.perf_counter() - t0
        cpu = {"value": round(done * G * w.row_bytes / dt * 1e-9, 5), "unit": "GB/s", "cores": 1, "kind": "oracle",
               "sample": f"oracle compressor (masks + pack) on the first {done} groups ({done * G} rows) of the {w.name} table, {dt:.1f} s"}
    line = {
        "metric": "compression throughput, raw GB/s (ibp_build_device kernels)", "value": round(raw / (k_ms * 1e-3) * 1e-9, 3), "unit": "GB/s",
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": round(k_ms, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic",
        "config": {"workload": describe(w) + " -- whole table compressed, rows resident in HBM, packed store written to host memory", "align_bytes": info.align_bytes,
                   "codec": "group-strict (tau = 1)" if not info.thresholded else f"thresholded, tau = {thr[0]}/{thr[1]}",
                   "store": {1: "pinned (cudaHostAlloc)", 2: "managed host-resident"}[info.store_kind], "packed_store_GB": round(info.packed_bytes_stored * 1e-9, 3),
                   "slices_per_group": stats[0].slices_per_group},
        "kernels_ms": {"mask": round(mean("mask_ms"), 4), "size": round(mean("size_ms"), 4), "scan": round(mean("scan_ms"), 4), "pack": round(mean("pack_ms"), 4)},
        "roofline": {"bound": "pcie", "kernel": "ibp_pack_t_kernel" if info.thresholded else ("ibp_pack_bulk_kernel" if (w.group_kind == 0 and info.align_bytes >= 16) else "ibp_pack_kernel"), "achieved": round(stats[0].store_bytes / (mean("pack_ms") * 1e-3) * 1e-9, 3),
                     "peak": round(d2h_ceiling, 3), "unit": "GB/s", "frac": round(stats[0].store_bytes / (mean("pack_ms") * 1e-3) * 1e-9 / d2h_ceiling, 4), "traffic": None,
                     "peak_source": "cudaMemcpyAsync D2H of 1 GiB into pinned memory, best of 8, this run (ibp_measure_d2h)",
                     "algorithmic_bytes_per_launch": int(stats[0].store_bytes)},
        "roofline_mask_kernel": {"bound": "hbm", "kernel": "ibp_mask_kernel", "achieved": round(raw / (mean("mask_ms") * 1e-3) * 1e-9, 1), "peak": hbm_peak, "unit": "GB/s",
                                 "frac": round(raw / (mean("mask_ms") * 1e-3) * 1e-9 / hbm_peak, 4), "algorithmic_bytes_per_launch": int(raw)},
        "e2e": {"value": round(raw / (mean("total_ms") * 1e-3) * 1e-9, 3), "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": int(stats[0].store_bytes),
                "note": "whole ibp_build_device call: kernels + host-side store allocation and zero fill + metadata copies to the host"},
        "host_build": {"value": round(raw / t_host * 1e-9, 3), "unit": "GB/s", "what": f"ibp_build (host compressor, all {os.cpu_count()} cores), {t_host:.2f} s"},
        "gpu_launches": K * (2 if not info.thresholded else 6), "clocks": clk, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)


def run_masks(args):
    """the mask-quality tools on the workload's table resident in HBM (csrc/ibp_analysis.cu).
    Fig. 13's protocol (space saved for chunk sizes 1/2/4/8 B x T/N 70..100 %, one global Mask/Bitval), Table 5's
    (masks from a 1/10/50 % sample evaluated on all rows) and Fig. 15's (net space saved vs number of clusters of
    a bit-similarity k-means) on SYNTHETIC rows; one step = one counting pass + one size pass over the table."""
    import torch
    from paper_2605_30728_b200 import binding as ibp
    from oracle import mask_tools as mt

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py --phase masks runs on one GPU")
    torch.cuda.set_device(0)
    w = make_workload(args.workload)
    X = w.table()
    Xb = X.view(np.uint8).reshape(w.n_rows, -1)
    n, rb = Xb.shape
    xd = torch.from_numpy(Xb).cuda()
    st = torch.cuda.current_stream().cuda_stream
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        hbm_peak = 6650.0
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    glob = ibp.table_desc(n, rb, ibp.IBP_GROUP_BLOCKED, 1 << 30)
    W, K = max(3, min(args.warmup, 5)), max(1, min(args.steps, 10))
    counts = torch.zeros(8 * rb, dtype=torch.int32, device="cuda")
    gn = torch.zeros(1, dtype=torch.int32, device="cuda")
    mask = torch.zeros(rb, dtype=torch.uint8, device="cuda")
    bitval = torch.zeros(rb, dtype=torch.uint8, device="cuda")
    totals = torch.zeros(2, dtype=torch.int64, device="cuda")
    t_cnt, t_sz = [], []
    clocks = ClockSampler(0)
    for it in range(W + K):
        if it == W:
            clocks.start()
        flush.zero_()
        counts.zero_(); gn.zero_(); totals.zero_()
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        ibp.ibp_bit_counts_device(xd.data_ptr(), glob, None, 0, counts.data_ptr(), gn.data_ptr(), st)
        e[1].record()
        ibp.ibp_masks_from_counts_device(counts.data_ptr(), gn.data_ptr(), 1, rb, 4, 5, mask.data_ptr(), bitval.data_ptr(), None, st)
        ibp.ibp_compressed_size_device(xd.data_ptr(), glob, mask.data_ptr(), bitval.data_ptr(), 4, None, totals.data_ptr(), st)
        e[2].record()
        torch.cuda.synchronize()
        if it >= W:
            t_cnt.append(e[0].elapsed_time(e[1])); t_sz.append(e[1].elapsed_time(e[2]))
    clk = clocks.stop()
    ms_cnt, ms_sz = float(np.mean(t_cnt)), float(np.mean(t_sz))
    raw = n * rb
    # parity of a sample against the oracle: counters of 3,000 rows, masks and sizes from them
    sample = np.sort(np.random.default_rng(1).choice(n, 3000, replace=False))
    sd = torch.from_numpy(sample.astype(np.int64)).cuda()
    counts.zero_(); gn.zero_()
    ibp.ibp_bit_counts_device(xd.data_ptr(), glob, sd.data_ptr(), len(sample), counts.data_ptr(), gn.data_ptr(), st)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    oc, on = mt.bit_counters(Xb, np.zeros(n, np.int64), 1, sample)
    t_or = time.perf_counter() - t0
    if not (np.array_equal(counts.cpu().numpy().astype(np.uint64), oc[0]) and int(gn.item()) == int(on[0])):
        raise SystemExit("bench.py: GPU bit counters differ from the oracle; refusing to report a number")
    # Fig. 13: chunk size x T/N, one global Mask/Bitval
    taus = [(70, 100), (75, 100), (80, 100), (85, 100), (90, 100), (95, 100), (1, 1)]
    css = [1, 2, 4, 8]
    tot, _ = ibp.ibp_mask_sweep_device(xd.data_ptr(), glob, None, 0, taus, css, st)
    fig13 = {f"{c}B": [round(100.0 * (1 - int(tot[i, j]) / raw), 2) for i in range(len(taus))] for j, c in enumerate(css)}
    # the build's per-group masks for comparison
    grp = ibp.table_desc(n, rb, w.group_kind, w.group_param)
    ng = ibp.ibp_table_groups(grp)
    totg, _ = ibp.ibp_mask_sweep_device(xd.data_ptr(), grp, None, 0, [(4, 5), (1, 1)], [4], st)
    per_group = {"groups": ng, "space_saved_pct_tau_0.8": round(100.0 * (1 - (int(totg[0, 0]) + 2 * rb * ng) / raw), 2),
                 "space_saved_pct_tau_1": round(100.0 * (1 - (int(totg[1, 0]) + 2 * rb * ng) / raw), 2), "note": "net of 2*row_bytes metadata per group"}
    # Table 5: sampled masks evaluated on the whole table
    sampling = {}
    for pct in (1, 10, 50, 100):
        ids = np.sort(np.random.default_rng(pct).choice(n, n * pct // 100, replace=False)).astype(np.int64)
        idd = torch.from_numpy(ids).cuda()
        ts, _ = ibp.ibp_mask_sweep_device(xd.data_ptr(), glob, idd.data_ptr(), len(ids), [(4, 5)], [4], st)
        sampling[f"{pct}%"] = round(raw / int(ts[0, 0]), 4)
    # Fig. 15: k-means on 250,000 rows (the paper's dataset size), net space saved vs k
    nk = min(n, 250_000)
    first = max(0, min(n - nk, 7_000_000 - nk // 2)) if args.workload == "gnn" else 0     # GNN: half dense, half sparse rows
    xs = xd[first:first + nk]
    rng = np.random.default_rng(15)
    fig15 = {}
    for k in (1, 2, 16, 128, 1024):
        init = torch.from_numpy(np.sort(rng.choice(nk, k, replace=False)).astype(np.int64)).cuda()
        assign = torch.zeros(nk, dtype=torch.int32, device="cuda")
        cent = torch.zeros((k, rb), dtype=torch.uint8, device="cuda")
        cost = torch.zeros(4, dtype=torch.int64, device="cuda")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ibp.ibp_kmeans_bits_device(xs.data_ptr(), nk, rb, k, init.data_ptr(), 4, assign.data_ptr(), cent.data_ptr(), cost.data_ptr(), st)
        e1.record()
        torch.cuda.synchronize()
        used = int(torch.unique(assign).numel())
        tk, _ = ibp.ibp_mask_sweep_device(xs.data_ptr(), ibp.table_desc(nk, rb, ibp.IBP_GROUP_MAP, 0, k, assign.data_ptr()), None, 0, [(4, 5)], [4], st)
        extra = {}
        if k == 2:
            # clustered compression with this library's positional groups: reorder the rows so that clusters are runs of
            # consecutive rows (ibp_order_by_group_device), then strict blocked groups of 256 over either order
            order = torch.zeros(nk, dtype=torch.int64, device="cuda")
            ibp.ibp_order_by_group_device(assign.data_ptr(), nk, k, order.data_ptr(), None, st)
            xo = xs.index_select(0, order)
            g256 = ibp.table_desc(nk, rb, ibp.IBP_GROUP_BLOCKED, 256)
            ng256 = ibp.ibp_table_groups(g256)
            t_a, _ = ibp.ibp_mask_sweep_device(xs.data_ptr(), g256, None, 0, [(1, 1)], [4], st)
            t_b, _ = ibp.ibp_mask_sweep_device(xo.data_ptr(), g256, None, 0, [(1, 1)], [4], st)
            extra = {"groups_of_256_net_space_saved_pct": {"original_order": round(100.0 * (1 - (int(t_a[0, 0]) + 2 * rb * ng256) / (nk * rb)), 2),
                                                            "cluster_order": round(100.0 * (1 - (int(t_b[0, 0]) + 2 * rb * ng256) / (nk * rb)), 2)}}
        fig15[str(k)] = {**extra, "net_space_saved_pct": round(100.0 * (1 - (int(tk[0, 0]) + 2 * rb * used) / (nk * rb)), 2), "clusters_used": used,
                         "ms_4_iterations": round(e0.elapsed_time(e1), 2), "cost": [int(c) for c in cost.cpu().tolist()]}
    cpu = None
    if not args.no_cpu:                                                # the oracle's counting pass on successive slices, about 12 s
        t0 = time.perf_counter()
        done = 0
        while time.perf_counter() - t0 < 12.0 and done + 20000 <= n:
            mt.bit_counters(Xb[done:done + 20000], np.zeros(20000, np.int64), 1)
            done += 20000
        dt = time.perf_counter() - t0
        cpu = {"value": round(done * rb / dt * 1e-9, 6), "unit": "GB/s", "cores": 1, "kind": "oracle",
               "sample": f"oracle/mask_tools.bit_counters (P:229, one row at a time) on the first {done} rows of the {w.name} table, {dt:.1f} s"}
    line = {
        "metric": "preprocessing throughput, raw GB/s (per-bit counters + compressed sizes of the whole table)", "value": round(raw / ((ms_cnt + ms_sz) * 1e-3) * 1e-9, 1),
        "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": round(ms_cnt + ms_sz, 4), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": describe(w) + " -- whole table resident in HBM, one global Mask/Bitval (P:231), tau = 4/5, 4-byte chunks",
                   "l2": "flushed with a 256 MiB write between steps (outside the events)"},
        "kernels_ms": {"ibp_count_kernel": round(ms_cnt, 4), "ibp_masks_kernel + ibp_csize_kernel": round(ms_sz, 4)},
        "roofline": {"bound": "hbm", "kernel": "ibp_count_kernel", "achieved": round(raw / (ms_cnt * 1e-3) * 1e-9, 1), "peak": hbm_peak, "unit": "GB/s",
                     "frac": round(raw / (ms_cnt * 1e-3) * 1e-9 / hbm_peak, 4), "traffic": None, "algorithmic_bytes_per_launch": int(raw),
                     "peak_source": "MEASURED_PEAKS.json hbm_gbs"},
        "roofline_csize_kernel": {"bound": "hbm", "kernel": "ibp_csize_kernel<4>", "achieved": round(raw / (ms_sz * 1e-3) * 1e-9, 1), "peak": hbm_peak, "unit": "GB/s",
                                  "frac": round(raw / (ms_sz * 1e-3) * 1e-9 / hbm_peak, 4), "algorithmic_bytes_per_launch": int(raw)},
        "fig13_space_saved_pct": {"tau_pct": [70, 75, 80, 85, 90, 95, 100], **fig13, "what": "one global Mask/Bitval; rows: chunk size; P:525-537 protocol on synthetic rows"},
        "per_group_masks": per_group, "table5_ratio_from_sampled_masks": sampling,
        "fig15_kmeans": {"rows": nk, "first_row": first, **fig15},
        "e2e": {"value": round(raw / ((ms_cnt + ms_sz) * 1e-3) * 1e-9, 1), "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 16,
                "note": "the table is resident in HBM by design (preprocessing of a dataset already staged); only the totals come back"},
        "gpu_launches": K * 3, "clocks": clk, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)


def run_resident(args):
    """SURVEY 8(a) S8 alone: ibp_decompress_resident of a contiguous range whose packed bytes were staged in HBM beforehand
    (what a compressed GPU cache or a DMA-staged block decodes).  One step = one launch over the range: the first
    2^20 rows of the workload's table, or one 4096 x 11008 bf16 matrix for `weights`.  HBM-bound: algorithmic bytes = packed
    in + rows out + Mask/Bitval of the groups touched."""
    import torch
    from paper_2605_30728_b200 import binding as ibp, workloads
    import oracle

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py --phase resident runs on one GPU")
    torch.cuda.set_device(0)
    thr = parse_threshold(args.threshold)
    if args.workload == "weights":
        w = workloads.WeightMatrix(rows=4096, cols=11008)
        nr = w.n_rows
        label = "configs[4] one 4096 x 11008 bf16 matrix N(0,0.02), 128-column tiles as strided groups (86 tiles)"
    else:
        w = make_workload(args.workload)
        nr = min(w.n_rows, 1 << 20)
        label = describe(w) + f" -- the first {nr} rows"
    align = args.align if args.align else w.align_bytes
    X = w.rows(0, nr)
    Xb = X.view(np.uint8).reshape(nr, -1)
    h = ibp.ibp_build(Xb, w.row_bytes, w.group_kind, w.group_param, align_bytes=align, threshold=thr, flags=ibp.IBP_FLAG_PAGEABLE_STORE).upload_metadata(0)
    if args.stream_mode is not None:
        h.set_stream_mode(args.stream_mode)
    info = h.info()
    stream = torch.cuda.current_stream().cuda_stream
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        hbm_peak = 6650.0
    ptr, nb = h.packed_range(0, nr)
    staged = torch.from_numpy(h.packed_view(ptr, nb).copy()).cuda()
    out = torch.empty((nr, w.row_bytes), dtype=torch.uint8, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    W, K = max(3, args.warmup), max(1, args.steps)
    for _ in range(W):
        h.decompress_resident(staged.data_ptr(), 0, nr, out.data_ptr(), stream)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    if not np.array_equal(got, Xb):                                            # (c1): the original rows, every byte
        raise SystemExit("bench.py: resident decode differs from the original rows; refusing to report a number")
    ids = np.random.default_rng(0).choice(nr, 256, replace=False)
    ds = (oracle.Dataset(Xb, w.group_kind, w.group_param) if thr[0] == thr[1] else oracle.DatasetT(Xb, w.group_kind, w.group_param, thr[0], thr[1])) if nr * w.row_bytes <= (64 << 20) else None
    if ds is not None:
        if not np.array_equal(got[ids], ds.gather_decompress(ids)):
            raise SystemExit("bench.py: resident decode differs from the oracle codec")
        ds.close()
    clocks = ClockSampler(0)
    clocks.start()
    ms = []
    for _ in range(K):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        h.decompress_resident(staged.data_ptr(), 0, nr, out.data_ptr(), stream)
        b.record()
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
    clk = clocks.stop()
    t = float(np.mean(ms))
    meta_bytes = info.n_groups * 2 * w.row_bytes
    alg = nb + nr * w.row_bytes + meta_bytes
    # e2e: the packed bytes come from pinned host memory (DMA staging, P:357 cache fill path) and the rows go back to the host
    pk_pin = ibp.PinnedBuffer(nb)
    pk_pin.view(np.uint8)[:] = h.packed_view(ptr, nb)
    out_pin = ibp.PinnedBuffer(nr * w.row_bytes)
    pin_t = torch.from_numpy(pk_pin.view(np.uint8))
    out_t = torch.from_numpy(out_pin.view(np.uint8, (nr, w.row_bytes)))
    te = []
    for i in range(5):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        staged.copy_(pin_t, non_blocking=True)
        h.decompress_resident(staged.data_ptr(), 0, nr, out.data_ptr(), stream)
        out_t.copy_(out, non_blocking=True)
        b.record()
        torch.cuda.synchronize()
        if i >= 2:
            te.append(a.elapsed_time(b))
    cpu = None
    if not args.no_cpu:
        sample = Xb[: 96 * w.group_param] if w.group_kind == 0 else Xb
        dsb = oracle.Dataset(sample, w.group_kind, w.group_param) if thr[0] == thr[1] else oracle.DatasetT(sample, w.group_kind, w.group_param, thr[0], thr[1])
        t0 = time.perf_counter()
        done = 0
        sid = np.arange(min(len(sample), 20000), dtype=np.int64)
        while time.perf_counter() - t0 < 10.0:
            dsb.gather_decompress(sid)
            done += len(sid)
        dt = time.perf_counter() - t0
        dsb.close()
        cpu = {"value": round(done * w.row_bytes / dt * 1e-9, 5), "unit": "GB/s", "cores": 1, "kind": "oracle",
               "sample": f"{done} row decodes of the first {len(sid)} rows by the oracle codec, {dt:.1f} s"}
    kernel = "ibp_stream_t_kernel" if info.thresholded else "ibp_stream_kernel"
    line = {
        "metric": "resident decode, decompressed GB/s (ibp_decompress_resident)", "value": round(nr * w.row_bytes / (t * 1e-3) * 1e-9, 1), "unit": "GB/s",
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": round(t, 5), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic", "rows_per_s": round(nr / (t * 1e-3)),
        "config": {"workload": label + "; packed bytes staged in HBM, decoded to HBM", "rows": nr, "row_bytes": w.row_bytes, "align_bytes": info.align_bytes,
                   "codec": "group-strict (tau = 1)" if not info.thresholded else f"thresholded, tau = {thr[0]}/{thr[1]}",
                   "packed_MB": round(nb * 1e-6, 2), "ratio_stored": round(nr * w.row_bytes / nb, 4),
                   "l2": "flushed with a 256 MiB write between steps (outside the events)"},
        "roofline": {"bound": "hbm", "kernel": kernel, "achieved": round(alg / (t * 1e-3) * 1e-9, 1), "peak": hbm_peak, "unit": "GB/s",
                     "frac": round(alg / (t * 1e-3) * 1e-9 / hbm_peak, 4), "traffic": None, "algorithmic_bytes_per_launch": int(alg),
                     "algorithmic_bytes_def": "packed bytes in + rows out + 2*row_bytes of Mask/Bitval per group", "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy; read+write bytes)"},
        "e2e": {"value": round(nr * w.row_bytes / (float(np.mean(te)) * 1e-3) * 1e-9, 2), "unit": "GB/s", "h2d_bytes_per_step": int(nb), "d2h_bytes_per_step": int(nr * w.row_bytes),
                "api": "cudaMemcpyAsync of the packed range from pinned memory, ibp_decompress_resident, cudaMemcpyAsync of the rows to pinned memory"},
        "gpu_launches": K, "clocks": clk, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)


def run_probes(args):
    """The link ceilings every roofline in this file is read against, and the levers that were tried on the random-row path
    (DESIGN.md section 6): copy-engine H2D / D2H, SM-issued contiguous zero-copy reads, and random span reads over host memory of
    every kind the library can map -- the span rate of a large footprint follows the GPU-side page size of the mapping."""
    import torch
    from paper_2605_30728_b200 import binding as ibp
    torch.cuda.set_device(0)
    fp = 6 << 30
    kinds = [("managed host-resident (default store)", ibp.IBP_MEM_MANAGED_HOST), ("cudaHostAlloc", ibp.IBP_MEM_HOSTALLOC),
             ("mmap 4 KB pages + cudaHostRegister", ibp.IBP_MEM_MALLOC_REGISTERED), ("mmap + MADV_HUGEPAGE + cudaHostRegister", ibp.IBP_MEM_THP_REGISTERED),
             ("hugetlbfs 2 MB pages + cudaHostRegister", ibp.IBP_MEM_HUGETLB_2M_REGISTERED)]
    table = []
    for name, k in kinds:
        row = {"memory": name}
        for span in (128, 256):
            try:
                sps, gbs = ibp.ibp_measure_random_read_kind(0, fp, span, k, 3)
                row[f"span_{span}B"] = {"M_spans_per_s": round(sps * 1e-6, 1), "GBps": round(gbs, 2)}
            except ibp.IbpError as e:
                row[f"span_{span}B"] = {"unavailable": str(e)[:160]}
        table.append(row)
    scan = []
    for mb in (32, 256, 1024, 2048, 6144):
        sps, gbs = ibp.ibp_measure_random_read_kind(0, mb << 20, 128, ibp.IBP_MEM_MANAGED_HOST, 3)
        scan.append({"footprint_MiB": mb, "M_spans_per_s": round(sps * 1e-6, 1), "GBps": round(gbs, 2)})
    line = {"metric": "link probes", "unit": "GB/s", "n_gpus": 1,
            "h2d_memcpy_GBps": round(ibp.ibp_measure_h2d(0, 1 << 30, 8), 2), "d2h_memcpy_GBps": round(ibp.ibp_measure_d2h(0, 1 << 30, 8), 2),
            "zero_copy_contiguous_read_GBps": round(ibp.ibp_measure_zero_copy_read(0, 1 << 30, 3), 2),
            "random_span_reads_6GiB_footprint": table, "random_128B_spans_managed_by_footprint": scan,
            "hugepages": {k: open(f).read().strip() for k, f in (("nr_hugepages", "/proc/sys/vm/nr_hugepages"), ("thp", "/sys/kernel/mm/transparent_hugepage/enabled")) if os.path.exists(f)}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="gnn", choices=["gnn", "gnn-interleaved", "dlrm", "dlrm-hot", "tiny", "kv", "weights", "sweep"])
    ap.add_argument("--align", type=int, default=0, help="packed-row alignment unit A; 0 = the workload's default")
    ap.add_argument("--layers", type=int, default=32, help="weights workload: decoder layers held in host memory (32 = BASELINE's 12.95 GB)")
    ap.add_argument("--gemm-m", type=int, default=16384, help="weights workload: rows of the consumer GEMM's activation")
    ap.add_argument("--decode-ctas", type=int, default=0, help="limit the decode grid (SM share of the fetch); 0 = library default")
    ap.add_argument("--store", default="managed", choices=["managed", "pinned"])
    ap.add_argument("--threshold", default="1/1", help="tau = T/N as a fraction: 1/1 = group-strict (BASELINE.json), 4/5 = the paper's thresholded codec")
    ap.add_argument("--order", type=int, default=None, choices=[0, 1])
    ap.add_argument("--dedup", type=int, default=None, choices=[0, 1], help="default: off when the workload's sampler guarantees distinct ids, else the library's automatic mode")
    ap.add_argument("--phase", default="gather", choices=["gather", "build", "masks", "resident", "probes"],
                    help="gather = the hot path (default); build = the GPU-side compressor ibp_build_device; masks = the mask-quality tools (tau / chunk-size sweep, sampled masks, k-means); resident = ibp_decompress_resident alone (S8)")
    ap.add_argument("--cache-frac", type=float, default=0.0, help="gnn/dlrm: put a compressed GPU cache of this fraction of the packed store in front of the host store")
    ap.add_argument("--stream-mode", type=int, default=None, choices=[0, 1, 2], help="--phase resident: ibp_set_stream_mode (test/compare hook)")
    ap.add_argument("--no-baseline", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-resident", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="default gnn run: skip the per_config entries for the other four BASELINE configs")
    ap.add_argument("--no-pinned-store", action="store_true", help="skip value_pinned_store (the same step over a cudaHostAlloc store)")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.workload in ("weights", "sweep"):
            args.workload = "kv"      # the oracle arm samples row decodes; bf16 256-byte rows either way
        run_reference(args)
    elif args.workload == "sweep":
        run_sweep(args)
    elif args.phase == "build":
        run_build(args)
    elif args.phase == "masks":
        run_masks(args)
    elif args.phase == "resident":
        run_resident(args)
    elif args.phase == "probes":
        run_probes(args)
    elif args.workload == "weights":
        run_weights(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
