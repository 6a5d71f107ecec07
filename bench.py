#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv 2402.00665 on B200.

A "step" is one pass of the whole hot path over one batch of synthetic input: linear-BVH build (scene
bounds, Morton codes, one-sweep radix sort, modified-Apetrei bottom-up pass with ropes and boxes) followed
by stackless sphere range search to CSR.  The query part of the step is the single-pass form of
count-then-fill (order, collect = one traversal that counts and stores rows, scan, rows -> CSR, overflow
rows) as ONE call of the C ABI (bvh_query_csr); the same stages as separate calls give the per-kernel breakdown, and
the two-traversal form (count, scan, fill) is timed beside it as `query_two_pass`.  The row capacity of the single-pass
query is learned from ANOTHER batch of the same workload (other seeds; an untimed count pass), never from the batch
that is timed: rows that do not fit are traversed again inside the timed call (`query.overflow_rows`), and
`query_small_capacity` times the same call with 1.25 x the other batch's mean row as capacity.  Workload at N=1: BASELINE.json configs[2]
("C3": 10,000,000 Gaussian-mixture points, 30-bit Morton, 1,000,000 sphere queries of radius 0.002), the
config `north_star` quotes its target on.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
  torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N --steps K --warmup W

`value` = build throughput (Mprims/s) with inputs resident in HBM, CUDA-event time of the build part of the
step; the query part is reported beside it (`query`), `ms_per_step` covers both.  N > 1 runs N independent
replicas (one per GPU, different seeds, no collective on the data path: DESIGN.md "Multi-GPU"), timed as
the max over ranks; `--multi shard` instead builds the same hierarchy on every rank and splits ONE query batch
over the ranks (NEXT-4: strong scaling of the query part, one all-gather of result sizes).  `--impl reference` times the CPU oracle (oracle/) on a bounded sample: for this tier
the oracle is the reference arm.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2402_00665_b200 import workloads  # noqa: E402  (numpy only; loads nothing native)

METRIC = "bvh_build_throughput"
UNIT = "Mprims/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
NOMINAL_HBM_GBS = 8000.0   # the denominator BASELINE.json north_star names

# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of a kernel from the `ncu --set full` captures
# summarised in profiles/, keyed by (workload, n, q): `roofline.traffic` is null for any other workload or size.
NCU_TRAFFIC_BYTES = {
    # profiles/r03_ncu.md, one step each: collect, rows_to_csr, level 1 of the hierarchy (DRAM read + write);
    # profiles/r02b_ncu.md, two-pass leg, rows 0 (count), 1 (fill)
    ("C3", 10_000_000, 1_000_000): {"collect": 3_180_537_000, "rows_to_csr": 4_829_984_000, "count": 241_363_000,
                                    "fill": 3_220_800_000, "hierarchy": 1_333_382_000},
    ("C4", 4_000_000, 4_000_000): {"collect": 948_331_008, "rows_to_csr": 313_999_616,
                                   "hierarchy": 605_211_136},
    ("C5", 1 << 24, 1 << 24): {"collect": 6_883_123_000, "rows_to_csr": 5_561_789_000,
                               "hierarchy": 2_681_882_000},
}


# ---- byte model (restated in DESIGN.md "Roofline") ---------------------------------------

def byte_model(n: int, q: int, nnz: int, prim_floats: int, query_floats: int, bits: int) -> dict:
    S, K, P, Sq = 4 * prim_floats, (4 if bits == 30 else 8), (4 if bits == 30 else 8), 4 * query_floats
    per_kernel = {
        "init": 4 * n,                                   # store memset (status words are implementation overhead)
        "bounds": S * n,
        "morton": (S + K) * n,                           # + digit histograms, fused (the model's "histogram read K" is saved)
        "sort_pass0": (K + K + 4) * n,                   # read code, write code + index (iota synthesised)
        **{f"sort_pass{p}": 2 * (K + 4) * n for p in range(1, P)},
        "hierarchy": (4 + S + 32 + K + 4 + 32 + 24) * n,  # perm, input, leaf record, codes, CAS, internal record, sibling box
        "order": (Sq + 4) * q + (4 + 4 + 4) * q + 3 * 16 * q,   # query Morton codes + 4 sort passes of (code, index)
        "count": (Sq + 4 + 4) * q,
        "scan": (4 + 8) * q,
        "fill": (Sq + 8 + 4) * q + 4 * nnz,
        "collect": (Sq + 4 + 4) * q + 4 * nnz,           # query, order, count out, every hit stored once
        "rows_to_csr": (4 + 8) * q + 8 * nnz,            # counts, offsets, every hit read and written once
        "overflow": 4 * q,                               # counts (no row overflows when the capacity holds the largest row)
    }
    per_kernel["tie_fixup"] = K * n                  # 63-bit two-stage sort: one read of the sorted codes
    per_kernel["second_sort"] = 0                    # ... and one cooperative launch that returns at once unless a run did not fit a block
    per_kernel["front"] = sum(v for k, v in per_kernel.items() if k in ("init", "bounds", "morton") or k.startswith("sort_pass"))
    build_total = (3 * S + 4 * K + (2 * P - 1) * (K + 4) + 100) * n      # SURVEY.md B_build
    query_total = (2 * Sq + 24) * q + 4 * nnz                            # SURVEY.md B_query
    return {"per_kernel": per_kernel, "build_total": build_total, "query_total": query_total}


def measured_peak() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ---- clocks ---------------------------------------------------------------------------------------------------

class ClockSampler:
    """nvidia-smi sampling of SM clocks and throttle reasons while the timed region runs."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "50", "-f", self.path], stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        try:
            rows = [r.split(",") for r in open(self.path).read().strip().splitlines() if r.strip()]
            os.unlink(self.path)
            sm = [float(r[0]) for r in rows]
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            reasons = [nm for k, nm in enumerate(names) if any(r[3 + k].strip().lower() == "active" for r in rows)]
            if sm:
                # "under load": the upper half of the samples (idle gaps between steps pull the clock down)
                load = sorted(sm)[len(sm) // 2:]
                out.update(sm_mhz=float(np.median(load)), sm_max_mhz=float(rows[0][1]), reasons=reasons,
                           samples=len(sm), power_w_max=max(float(r[2]) for r in rows))
        except Exception as e:  # never let telemetry kill the bench
            out["error"] = repr(e)
        return out


# ---- distributed plumbing (one process per GPU; nothing on the data path) ---------------------------------------

def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    import torch.distributed as dist

    rank, local_rank, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def dist_barrier(world: int, device=None):
    if world > 1:
        import torch.distributed as dist

        if device is not None and device.type == "cuda":
            dist.barrier(device_ids=[device.index])
        else:
            dist.barrier()


def reduce_max_sum(values_max, values_sum, world: int, device):
    """Max over ranks of `values_max` and sum over ranks of `values_sum` (lists of floats)."""
    import torch

    if world == 1:
        return list(values_max), list(values_sum)
    import torch.distributed as dist

    tm = torch.tensor(values_max, dtype=torch.float64, device=device)
    ts = torch.tensor(values_sum, dtype=torch.float64, device=device)
    dist.all_reduce(tm, op=dist.ReduceOp.MAX)
    dist.all_reduce(ts, op=dist.ReduceOp.SUM)
    return tm.cpu().tolist(), ts.cpu().tolist()


# ---- the two arms ---------------------------------------------------------------------------------------------------

def make_workload(args, rank: int):
    n = args.n if args.n else None
    q = args.q if args.q else None
    w = workloads.make(args.workload, n=n, q=q, seed_offset=rank)
    return w


def config_dict(args, w, world: int, extra=None) -> dict:
    c = {
        "workload": f"{w.name}: {w.n} {w.prim_kind} ({w.note}), {w.morton_bits}-bit Morton; {w.q} {w.query_kind} queries"
                    + (" [BASELINE.json configs[2]]" if (w.name == "C3" and not args.n and not args.q) else " [non-default size]"),
        "n": w.n, "q": w.q, "morton_bits": w.morton_bits, "replicas": world,
        "l2": "flushed between timed steps (512 MiB device write) and step working set >> 126 MB L2",
    }
    if extra:
        c.update(extra)
    return c


def run_ours(args) -> dict | None:
    import torch

    from paper_2402_00665_b200 import binding, sharded

    rank, local_rank, world = dist_init("nccl")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU path); use --impl reference for the oracle")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    binding.load_library()

    shard = args.multi == "shard" and world > 1
    w = make_workload(args, 0 if shard else rank)           # shard: every rank holds the same scene and the same batch
    n, bits = w.n, w.morton_bits
    is_box = int(w.prim_kind == "boxes")
    kind = binding.QUERY_KINDS[w.queries.shape[1]]
    q_lo, q_hi = sharded.block_bounds(w.q, rank, world) if shard else (0, w.q)
    q = q_hi - q_lo                                         # queries this rank serves
    h_prims = torch.from_numpy(w.prims).pin_memory()
    h_queries = torch.from_numpy(np.ascontiguousarray(w.queries[q_lo:q_hi])).pin_memory()
    d_prims = h_prims.to(device)
    d_queries = h_queries.to(device)
    bvh = binding.Bvh(n, bits, device)
    ws = binding.QueryWorkspace(q, device)
    order_fn = (binding.bvh_query_order_spheres, binding.bvh_query_order_boxes, binding.bvh_query_order_rays)[kind]
    count_fn = (binding.bvh_query_spheres_count, binding.bvh_query_boxes_count, binding.bvh_query_rays_count)[kind]
    fill_fn = (binding.bvh_query_spheres_fill, binding.bvh_query_boxes_fill, binding.bvh_query_rays_fill)[kind]
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)

    # Row capacity of the single-pass query.  A caller cannot know the rows of the batch it is about to serve, so the
    # capacity is NOT taken from this batch: it comes from an untimed count pass over ANOTHER batch of the same workload
    # (other seeds: "the previous batch"), rounded up to 8.  Rows of the timed batch that are longer overflow and are
    # traversed a second time inside the timed query; how many do is reported.  A second capacity, 1.25 x the previous
    # batch's mean row, is timed beside it (less scratch, more overflow).
    bvh.build(d_prims)
    cap, cap_small, prev_q = 8, 8, min(q, 1 << 20)
    if prev_q > 0:
        d_prev = torch.from_numpy(np.ascontiguousarray(
            workloads.previous_queries(args.workload, prev_q, seed_offset=0 if shard else rank))).to(device)
        count_fn(bvh.nodes, n, d_prev, prev_q, None, ws.counts)
        prev_counts = ws.counts[:prev_q]
        cap = max(8, (int(prev_counts.max().item()) + 7) // 8 * 8)
        cap_small = max(8, (int(np.ceil(1.25 * float(prev_counts.double().mean().item()))) + 7) // 8 * 8)
        del d_prev
    # one untimed pass over the batch itself: nnz sizes the result buffer (same inputs every step -> same counts)
    order_fn(bvh.nodes, n, d_queries, q, ws.order, ws.order_scratch)
    count_fn(bvh.nodes, n, d_queries, q, ws.order, ws.counts)
    binding.bvh_scan_counts(ws.counts, q, ws.offsets, ws.scan_scratch)
    nnz = int(ws.offsets[q].item())
    max_row = int(ws.counts[:q].max().item()) if q > 0 else 0
    overflow_rows = int((ws.counts[:q] > cap).sum().item()) if q > 0 else 0
    overflow_rows_small = int((ws.counts[:q] > cap_small).sum().item()) if q > 0 else 0
    d_indices = torch.empty(max(nnz, 1), dtype=torch.int32, device=device)
    d_rows = torch.empty(max(q, 1) * cap, dtype=torch.int32, device=device)

    def ev():
        e = torch.cuda.Event(enable_timing=True)
        e.record()  # materialise the cudaEvent_t so its handle can cross the C ABI
        return e

    stage = [ev() for _ in range(binding.NUM_STAGE_EVENTS)]
    e_b0, e_b1, e_order, e_collect, e_scan, e_rows, e_over = (ev() for _ in range(7))
    t_c0, t_c1, t_c2, t_c3 = (ev() for _ in range(4))
    P = 4 if bits == 30 else 8
    stage_for_call = [stage[k] if (k < 4 + P or k == 12) else None for k in range(binding.NUM_STAGE_EVENTS)]
    build_fn = binding.bvh_build_boxes if is_box else binding.bvh_build_points

    def step():
        """One pass of the hot path through the public entry points: the build as ONE call and the single-pass query
        as ONE call (bvh_query_csr), no events inside either."""
        e_b0.record()
        build_fn(d_prims, n, bits, bvh.nodes, bvh.scratch)
        e_b1.record()
        binding.bvh_query_csr(bvh.nodes, n, d_queries, kind, q, cap, d_rows, ws.order, ws.counts, ws.offsets, d_indices,
                              d_indices.numel(), ws.order_scratch)
        e_over.record()

    def staged_query():
        """The same query through its separate entry points, an event after each stage (per-kernel breakdown)."""
        e_b1.record()
        order_fn(bvh.nodes, n, d_queries, q, ws.order, ws.order_scratch)
        e_order.record()
        binding.bvh_query_collect(bvh.nodes, n, d_queries, kind, q, ws.order, cap, d_rows, ws.counts)
        e_collect.record()
        binding.bvh_scan_counts(ws.counts, q, ws.offsets, ws.scan_scratch)
        e_scan.record()
        binding.bvh_rows_to_csr(d_rows, cap, ws.counts, ws.offsets, q, d_indices)
        e_rows.record()
        binding.bvh_query_fill_overflow(bvh.nodes, n, d_queries, kind, q, ws.order, cap, ws.counts, ws.offsets, d_indices)
        e_over.record()

    def two_pass():
        """The two-traversal form of the same query (count, scan, fill), on the hierarchy the last step left."""
        t_c0.record()
        count_fn(bvh.nodes, n, d_queries, q, ws.order, ws.counts)
        t_c1.record()
        binding.bvh_scan_counts(ws.counts, q, ws.offsets, ws.scan_scratch)
        t_c2.record()
        fill_fn(bvh.nodes, n, d_queries, q, ws.order, ws.offsets, d_indices)
        t_c3.record()

    small_build = n <= 16384          # bounds + Morton + sort in one launch (csrc/small_build.cu), no memset
    two_stage = bits == 63 and not small_build   # 63-bit codes: 4 passes over the upper bits + tie fix-up (csrc/tie_fixup.cu)
    sort_names = [f"sort_pass{p}" for p in range(4)] + ["tie_fixup", "second_sort"] if two_stage else \
        [f"sort_pass{p}" for p in range(P)]
    build_names = ["front", "hierarchy"] if small_build else ["init", "bounds", "morton"] + sort_names + ["hierarchy"]
    query_names = ["order", "collect", "scan", "rows_to_csr", "overflow"]
    names = build_names + query_names
    # kernels of this library per stage when the stages are called one by one (the staged legs) ...
    launches_per_step = {**({"front": 1} if small_build else
                            {"init": 0, "bounds": 1, "morton": 1, **{k: 1 for k in sort_names},
                             **({"tie_fixup": 2, "second_sort": 1} if two_stage else {})}),
                         "hierarchy": 2 if n > 256 else 1, "order": 5 if q > 8192 else 1, "collect": 1,
                         "scan": 3 if q > 4096 else 1, "rows_to_csr": 1, "overflow": 1}
    # ... and in the timed step, where the query is one call: no identity order for q <= 8192, scan + row copy fused for q <= 4096
    step_launches = (sum(launches_per_step[k] for k in build_names)
                     + (5 if q > 8192 else 0) + 1 + (4 if q > 4096 else 1) + 1)

    def read_times() -> dict:
        return {"_build": e_b0.elapsed_time(e_b1), "_query": e_b1.elapsed_time(e_over), "_step": e_b0.elapsed_time(e_over)}

    def read_query_stage_times() -> dict:
        return {"order": e_b1.elapsed_time(e_order), "collect": e_order.elapsed_time(e_collect),
                "scan": e_collect.elapsed_time(e_scan), "rows_to_csr": e_scan.elapsed_time(e_rows),
                "overflow": e_rows.elapsed_time(e_over), "_query_staged": e_b1.elapsed_time(e_over)}

    def read_stage_times() -> dict:
        if small_build:   # bounds + Morton + sort are one launch (and there is no memset): one stage, "front"
            return {"front": stage[0].elapsed_time(stage[3 + P]), "hierarchy": stage[3 + P].elapsed_time(stage[12]),
                    "_build_staged": stage[0].elapsed_time(stage[12])}
        t = {"init": stage[0].elapsed_time(stage[1]), "bounds": stage[1].elapsed_time(stage[2]),
             "morton": stage[2].elapsed_time(stage[3])}
        prev = stage[3]
        for p in range(4 if two_stage else P):
            t[f"sort_pass{p}"] = prev.elapsed_time(stage[4 + p])
            prev = stage[4 + p]
        if two_stage:   # [8] after the fix-up, [11] after the (normally idle) kernels of the conditional second sort
            t["tie_fixup"] = stage[7].elapsed_time(stage[8])
            t["second_sort"] = stage[8].elapsed_time(stage[11])
            prev = stage[11]
        t["hierarchy"] = prev.elapsed_time(stage[12])
        t["_build_staged"] = stage[0].elapsed_time(stage[12])
        return t

    for _ in range(args.warmup):
        flush.fill_(1)
        step()
    torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    dist_barrier(world, device)
    torch.cuda.synchronize()
    acc = {}
    per_step_build = []
    for _ in range(args.steps):
        flush.fill_(1)          # evict L2 between timed steps (outside the events)
        step()
        torch.cuda.synchronize()
        t = read_times()
        per_step_build.append(t["_build"])
        for k, v in t.items():
            acc[k] = acc.get(k, 0.0) + v
    torch.cuda.synchronize()
    dist_barrier(world, device)
    clocks = sampler.stop() if rank == 0 else None

    # ---- per-stage breakdown of the single-pass query: the same stages as separate calls, an event after each ----------
    for _ in range(args.steps):
        flush.fill_(1)
        staged_query()
        torch.cuda.synchronize()
        for k, v in read_query_stage_times().items():
            acc[k] = acc.get(k, 0.0) + v

    # ---- the one-call query again with the small capacity (1.25 x the previous batch's mean row): its own rows buffer ----
    e_s0, e_s1 = ev(), ev()
    d_rows_small = torch.empty(max(q, 1) * cap_small, dtype=torch.int32, device=device)
    for it in range(args.steps + 1):
        flush.fill_(1)
        e_s0.record()
        binding.bvh_query_csr(bvh.nodes, n, d_queries, kind, q, cap_small, d_rows_small, ws.order, ws.counts, ws.offsets,
                              d_indices, d_indices.numel(), ws.order_scratch)
        e_s1.record()
        torch.cuda.synchronize()
        if it > 0:   # the first one is a warm-up
            acc["small_cap_query"] = acc.get("small_cap_query", 0.0) + e_s0.elapsed_time(e_s1)
    del d_rows_small

    # ---- the two-traversal query, same inputs, same hierarchy (not part of `value` / `ms_per_step`) ------------------
    for _ in range(args.steps):
        flush.fill_(1)
        two_pass()
        torch.cuda.synchronize()
        for k, v in (("tp_count", t_c0.elapsed_time(t_c1)), ("tp_scan", t_c1.elapsed_time(t_c2)),
                     ("tp_fill", t_c2.elapsed_time(t_c3))):
            acc[k] = acc.get(k, 0.0) + v

    # ---- per-kernel breakdown of the build: the same build through bvh_build_staged, which records an event after
    # every kernel.  Separate steps, not part of `value`: an event between two kernels keeps the second from being
    # set up while the first still runs (programmatic dependent launch), so the staged build is a little slower.
    for _ in range(args.steps):
        flush.fill_(1)
        binding.bvh_build_staged(d_prims, is_box, n, bits, bvh.nodes, bvh.scratch, stage_for_call)
        torch.cuda.synchronize()
        for k, v in read_stage_times().items():
            acc[k] = acc.get(k, 0.0) + v

    # ---- end to end: pinned host inputs -> device -> build -> query -> CSR back on the host, public API ----------
    e2e_steps = max(1, min(args.steps, 5))
    h_root = torch.empty(32, dtype=torch.uint8).pin_memory()
    host_out = binding.HostCsr(q, nnz)

    def e2e_step():
        t0 = time.perf_counter()
        dp = h_prims.to(device, non_blocking=True)
        bvh.build(dp)
        h_root.copy_(bvh.nodes[64:96], non_blocking=True)   # root record (after the 64-byte header)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        # queries H2D, single-pass search in chunks, each chunk's rows copied to the host while the next one is searched
        binding.query_to_host(bvh, h_queries, host_out, row_capacity=cap, chunks=args.e2e_chunks)
        t2 = time.perf_counter()
        return t1 - t0, t2 - t1

    e2e_step()
    dist_barrier(world, device)
    e2e_b, e2e_q = 0.0, 0.0
    for _ in range(e2e_steps):
        b, qq = e2e_step()
        e2e_b += b
        e2e_q += qq
    dist_barrier(world, device)

    # ---- NEXT-1: operations at the leaf through the same traversal kernel (rank 0) -----------------------------------
    next1 = {}
    if rank == 0 and not args.no_extras:
        def timed(fn, reps=4):
            ts = []
            for _ in range(reps):
                flush.fill_(1)
                a0 = ev()
                fn()
                a1 = ev()
                torch.cuda.synchronize()
                ts.append(a0.elapsed_time(a1))
            return float(np.median(ts[1:]))

        if kind == 0:
            idx_n = torch.empty(max(q, 1), dtype=torch.int32, device=device)
            key_n = torch.empty(max(q, 1), dtype=torch.float32, device=device)
            ms_near = timed(lambda: binding.bvh_query_spheres_nearest(bvh.nodes, n, d_queries, q, ws.order, idx_n, key_n))
            found = int((idx_n[:q] >= 0).sum().item())
            ms_any = timed(lambda: binding.bvh_query_any_hit(bvh.nodes, n, d_queries, 0, q, ws.order, idx_n))
            next1["nearest_within_radius"] = {"ms": round(ms_near, 4), "mqueries_per_s": round(q / (ms_near * 1e-3) / 1e6, 2),
                                              "found": found}
            next1["any_hit"] = {"ms": round(ms_any, 4), "mqueries_per_s": round(q / (ms_any * 1e-3) / 1e6, 2)}
            next1["what"] = "same queries, Morton order from the step; no CSR (PAPER.md:56 'perform an operation')"
        if is_box:
            qr = int(min(max(q, 1), 1 << 20))
            lo, hi = w.prims[:, :3].min(axis=0), w.prims[:, 3:].max(axis=0)
            origins = workloads.uniform_cube(qr, seed=2001) * (hi - lo) * np.float32(1.2) + lo - (hi - lo) * np.float32(0.1)
            h_rays = workloads.rays_at(origins.astype(np.float32), workloads.sphere_surface(qr, seed=2002), 0.0,
                                       float(np.linalg.norm(hi - lo)))
            d_rays = torch.from_numpy(h_rays).to(device)
            wr = binding.QueryWorkspace(qr, device)
            off_r, idx_r = binding.query(bvh, d_rays, wr)          # sizes the result
            ridx = torch.empty(max(int(idx_r.numel()), 1), dtype=torch.int32, device=device)
            rms = timed(lambda: binding.query(bvh, d_rays, wr, indices=ridx))
            fi = torch.empty(qr, dtype=torch.int32, device=device)
            ft = torch.empty(qr, dtype=torch.float32, device=device)
            fms = timed(lambda: binding.bvh_query_rays_first_hit(bvh.nodes, n, d_rays, qr, wr.order, fi, ft))
            next1["rays"] = {"q": qr, "csr_ms": round(rms, 4), "csr_mrays_per_s": round(qr / (rms * 1e-3) / 1e6, 3),
                             "hits_per_ray": round(int(off_r[qr].item()) / qr, 3), "first_hit_ms": round(fms, 4),
                             "first_hit_mrays_per_s": round(qr / (fms * 1e-3) / 1e6, 3),
                             "what": "segments through the scene box, random directions: order + count + scan + fill, "
                                     "and first hit alone on the same order"}

    # ---- NEXT-2: the constructions the paper compares itself with, same bounds / Morton / sort -----------------------
    variant_info = None
    if rank == 0 and not args.no_variant:
        common = sum(acc[k] for k in build_names if k != "hierarchy") / args.steps     # staged: everything but the last step
        variant_info = {"alg4_build_ms": round(acc["_build"] / args.steps, 4),
                        "alg4_last_step_ms": round(acc["_build"] / args.steps - common, 4),
                        "what": "whole build as one call, median of 5; last step = build minus the staged times of memset, "
                                "bounds, Morton and sort (rank 0)"}
        for variant, label in ((1, "karras_topdown + algorithm2 ropes + separate box pass"),
                               (2, "algorithm3 (apetrei numbering, global atomics) + separate rope pass"),
                               (3, "algorithm4 as written (one thread per leaf, global store + ATOMICCAS, ropes and boxes "
                                   "in the same pass): the paper's modification without the windowed organisation")):
            vscratch = torch.empty(binding.bvh_variant_sizes(n, bits, variant), dtype=torch.uint8, device=device)
            vnodes = torch.empty_like(bvh.nodes)
            vt = []
            for _ in range(6):
                flush.fill_(1)
                v0 = ev()
                binding.bvh_build_variant(d_prims, is_box, n, bits, vnodes, vscratch, variant)
                v1 = ev()
                torch.cuda.synchronize()
                vt.append(v0.elapsed_time(v1))
            vms = float(np.median(vt[1:]))
            variant_info[f"variant{variant}"] = {"what": label, "build_ms": round(vms, 4), "last_step_ms": round(vms - common, 4)}
            del vscratch, vnodes

    # ---- reduce over ranks: time = max, units = sum -----------------------------------------------------------------
    keys = sorted(acc)
    mx, sm = reduce_max_sum([acc[k] for k in keys] + [e2e_b, e2e_q], [float(n), float(q), float(nnz)], world, device)
    acc = dict(zip(keys, mx[: len(keys)]))
    e2e_b, e2e_q = mx[len(keys)], mx[len(keys) + 1]
    n_all, q_all, nnz_all = sm
    if shard:
        n_all = float(n)                                    # one scene, replicated: the build does not scale in this mode
    if rank != 0:
        return None

    K = args.steps
    ms = {k: v / K for k, v in acc.items()}
    model = byte_model(n, q, nnz, w.prims.shape[1], w.queries.shape[1], bits)
    peak, peak_src = measured_peak()
    kernels = {}
    for k in names:
        b = model["per_kernel"][k]
        gbs = b / (ms[k] * 1e-3) / 1e9 if ms[k] > 0 else 0.0
        kernels[k] = {"ms": round(ms[k], 5), "alg_bytes": int(b), "gbs": round(gbs, 1), "frac": round(gbs / peak, 4),
                      "launches": launches_per_step[k]}
    dominant = max((k for k in names if launches_per_step[k] == 1), key=lambda k: ms[k])
    dk = kernels[dominant]
    build_gbs = model["build_total"] / (ms["_build"] * 1e-3) / 1e9
    query_gbs = model["query_total"] / (ms["_query"] * 1e-3) / 1e9
    tp_ms = ms["order"] + ms["tp_count"] + ms["tp_scan"] + ms["tp_fill"]
    value = n_all / (ms["_build"] * 1e-3) / 1e6
    full = not args.n and not args.q
    traffic = NCU_TRAFFIC_BYTES.get((w.name, w.n, w.q), {}).get(dominant) if full and world == 1 else None
    line = {
        "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": round(ms["_step"], 4), "higher_is_better": True, "scaling": "strong" if shard else "weak",
        "vs_baseline": None,
        "dtype": "u32 Morton codes / f32 boxes" if bits == 30 else "u64 Morton codes / f32 boxes", "data": "synthetic",
        "config": config_dict(args, w, world, {"hits_per_query": round(nnz_all / max(q_all, 1), 2), "nnz": int(nnz_all),
                                               "row_capacity": cap,
                                               "row_capacity_source": f"largest row of another batch of the workload ({prev_q} "
                                                                      "queries, other seeds), untimed count pass, rounded up to 8",
                                               "multi": args.multi if world > 1 else "single"}),
        "build": {"ms": round(ms["_build"], 4), "mprims_per_s": round(value, 2), "alg_bytes": int(model["build_total"]),
                  "gbs": round(build_gbs, 1), "frac_of_measured_peak": round(build_gbs / peak, 4),
                  "frac_of_8TBs": round(build_gbs / NOMINAL_HBM_GBS, 4),
                  "ms_min": round(min(per_step_build), 4), "ms_median": round(float(np.median(per_step_build)), 4)},
        "query": {"ms": round(ms["_query"], 4), "mqueries_per_s": round(q_all / (ms["_query"] * 1e-3) / 1e6, 3),
                  "alg_bytes": int(model["query_total"]), "gbs": round(query_gbs, 1),
                  "frac_of_measured_peak": round(query_gbs / peak, 4), "frac_of_8TBs": round(query_gbs / NOMINAL_HBM_GBS, 4),
                  "path": "bvh_query_csr, one call: order + collect + scan + rows_to_csr + fill_overflow (byte-identical CSR)",
                  "staged_ms": round(ms["_query_staged"], 4),
                  "row_capacity": cap, "rows_bytes": int(max(q, 1) * cap * 4), "largest_row": max_row,
                  "overflow_rows": overflow_rows,
                  "excluded": "nnz read-back and indices allocation (included in e2e)"},
        "query_two_pass": {"ms": round(tp_ms, 4), "mqueries_per_s": round(q_all / (tp_ms * 1e-3) / 1e6, 3),
                           "count_ms": round(ms["tp_count"], 4), "scan_ms": round(ms["tp_scan"], 4),
                           "fill_ms": round(ms["tp_fill"], 4), "path": "order + count + scan + fill"},
        "query_small_capacity": {"ms": round(ms["small_cap_query"], 4),
                                 "mqueries_per_s": round(q_all / (ms["small_cap_query"] * 1e-3) / 1e6, 3),
                                 "row_capacity": cap_small, "rows_bytes": int(max(q, 1) * cap_small * 4),
                                 "overflow_rows": overflow_rows_small,
                                 "path": "bvh_query_csr, one call, capacity = 1.25 x mean row of the other batch: the rows that "
                                         "overflow are traversed again by the fill inside the call (byte-identical CSR)"},
        "roofline": {"bound": "hbm", "kernel": dominant, "achieved": dk["gbs"], "peak": peak, "unit": "GB/s",
                     "frac": dk["frac"], "traffic": traffic, "peak_source": peak_src,
                     "alg_bytes_per_launch": dk["alg_bytes"], "ms_per_launch": dk["ms"]},
        "kernels": kernels,
        "build_staged_ms": round(ms["_build_staged"], 4),
        "gpu_launches": K * step_launches,
        "e2e": {"value": round(n_all / (e2e_b / e2e_steps) / 1e6, 2), "unit": UNIT,
                "h2d_bytes_per_step": int(h_prims.numel() * 4 + h_queries.numel() * 4),
                "d2h_bytes_per_step": int(32 + (q + 1) * 8 + nnz * 4), "steps": e2e_steps,
                "build_ms": round(e2e_b / e2e_steps * 1e3, 3), "query_ms": round(e2e_q / e2e_steps * 1e3, 3),
                "query_mqueries_per_s": round(q_all / (e2e_q / e2e_steps) / 1e6, 3), "query_chunks": args.e2e_chunks,
                "what": "pinned host prims -> H2D -> build -> root record D2H | pinned queries -> H2D -> single-pass search in "
                        "chunks, each chunk's CSR rows copied D2H on a second stream while the next chunk is searched -> "
                        "offsets + indices in pinned host memory; wall clock, through binding.Bvh / binding.query_to_host"},
        "clocks": clocks,
    }
    if next1:
        line["next1_operations"] = next1
    if variant_info:
        line["next2_variant"] = variant_info
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w)
    return line


def cpu_baseline(w) -> dict:
    """The oracle as it stands, one core, on a bounded sample of the same workload."""
    import oracle

    oracle.build()
    qs = min(w.q, 50_000)
    t0 = time.perf_counter()
    o = oracle.build_bvh(w.prims, w.morton_bits)
    t1 = time.perf_counter()
    if w.query_kind == "spheres":
        off, _ = oracle.query_spheres_tree(o, w.queries[:qs])
    else:
        off, _ = oracle.query_boxes_tree(o, w.queries[:qs])
    t2 = time.perf_counter()
    return {"value": round(w.n / (t1 - t0) / 1e6, 3), "unit": UNIT, "cores": 1, "kind": "oracle",
            "host_cores": os.cpu_count(),
            "sample": f"build: all {w.n} primitives once ({t1 - t0:.2f} s); queries: first {qs} of {w.q} against that tree "
                      f"({t2 - t1:.2f} s, {int(off[-1])} hits)",
            "query_mqueries_per_s": round(qs / (t2 - t1) / 1e6, 4)}


def run_reference(args) -> dict | None:
    """Reference arm for this tier = the CPU oracle, timed as it stands on the host cores (rank 0 only)."""
    rank, _, world = dist_env()
    if rank != 0:
        return None
    import oracle

    oracle.build()
    w = make_workload(args, 0)
    ns, qs = w.n, min(w.q, 10_000)          # the whole build (a few seconds for 10^7 primitives); a bounded query sample
    prims, queries = w.prims[:ns], w.queries[:qs]

    def step():
        t0 = time.perf_counter()
        o = oracle.build_bvh(prims, w.morton_bits)
        t1 = time.perf_counter()
        if w.query_kind == "spheres":
            oracle.query_spheres_tree(o, queries)
        else:
            oracle.query_boxes_tree(o, queries)
        return t1 - t0, time.perf_counter() - t1

    for _ in range(args.warmup):
        step()
    tb = tq = 0.0
    for _ in range(args.steps):
        b, qq = step()
        tb += b
        tq += qq
    value = round(ns / (tb / args.steps) / 1e6, 3)
    sample = (f"each step: oracle build of all {ns} primitives + the first {qs} of {w.q} queries on that tree; "
              f"serial, 1 of {os.cpu_count()} host cores")
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round((tb + tq) / args.steps * 1e3, 3), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "u32 Morton codes / f32 boxes" if w.morton_bits == 30 else "u64 Morton codes / f32 boxes", "data": "synthetic",
        "config": config_dict(args, w, world, {"sample": sample}),
        "query": {"mqueries_per_s": round(qs / (tq / args.steps) / 1e6, 4)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default="C3", choices=sorted(workloads.FULL_SIZES))
    ap.add_argument("--n", type=int, default=0, help="override the primitive count (non-default: for quick checks)")
    ap.add_argument("--q", type=int, default=0, help="override the query count")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-variant", action="store_true", help="skip the NEXT-2 comparison builds (Karras top-down, Algorithm 3)")
    ap.add_argument("--no-extras", action="store_true", help="skip the NEXT-1 operation timings (nearest, any hit, rays)")
    ap.add_argument("--multi", choices=["replicas", "shard"], default="replicas",
                    help="N > 1: independent replicas (weak scaling, default) or one query batch sharded over a replicated tree")
    ap.add_argument("--e2e-chunks", type=int, default=8, help="query chunks of the end-to-end leg (search / D2H overlap)")
    args = ap.parse_args(argv)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    line = run_reference(args) if args.impl == "reference" else run_ours(args)
    if line is not None:
        print(json.dumps(line), flush=True)
    try:
        import torch.distributed as dist

        if dist.is_available() and dist.is_initialized():
            dist.destroy_process_group()
    except Exception:
        pass


if __name__ == "__main__":
    main()
