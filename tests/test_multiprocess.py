"""N > 1 plumbing of bench.py on CPU: world_size 2, gloo, launched the way the driver launches it
(torch.distributed.run, 127.0.0.1).  The data path has no collective (replicas
only); what is covered here is the part that is shared between ranks: rendezvous, barrier, the
max-over-ranks / sum-over-ranks reduction of timings and units, per-rank seeds, and the reference arm
printing exactly one line from rank 0."""
from __future__ import annotations

import json
import os
import subprocess
import sys
import textwrap

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(script_args, port, timeout=600):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), *script_args]
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_reduce_over_two_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(textwrap.dedent(f"""
        import json, os, sys
        sys.path.insert(0, {ROOT!r})
        import torch
        import bench
        from paper_2402_00665_b200 import workloads
        rank, local_rank, world = bench.dist_init("gloo")
        assert world == 2
        bench.dist_barrier(world, torch.device("cpu"))
        w = workloads.make("C3", n=1000, q=10, seed_offset=rank)
        # times: rank r reports (r + 1) ms and (5 - r) ms; units: 1000 * (r + 1) primitives
        mx, sm = bench.reduce_max_sum([1.0 + rank, 5.0 - rank], [1000.0 * (rank + 1), float(w.q)], world,
                                      torch.device("cpu"))
        bench.dist_barrier(world, torch.device("cpu"))
        out = dict(rank=rank, mx=mx, sm=sm, first=w.prims[0].tolist())
        open(os.path.join({str(tmp_path)!r}, f"rank{{rank}}.json"), "w").write(json.dumps(out))
        torch.distributed.destroy_process_group()
    """))
    r = _torchrun([str(script)], port=29617)
    assert r.returncode == 0, r.stderr[-2000:]
    outs = [json.load(open(tmp_path / f"rank{k}.json")) for k in range(2)]
    for o in outs:
        assert o["mx"] == [2.0, 5.0]          # max over ranks
        assert o["sm"] == [3000.0, 20.0]      # sum over ranks
    # independent replicas: different seeds per rank
    assert not np.allclose(outs[0]["first"], outs[1]["first"])


def test_reference_arm_prints_one_line_from_rank0():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--workload", "C1"], port=29618)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0


def test_sharded_query_two_ranks_gloo_equals_single_rank_csr(tmp_path):
    """NEXT-4: one query batch split over 2 ranks against a replicated tree; the blocks of the global CSR (local CSR
    shifted by the results of the earlier rank, one all-gather of sizes) concatenate to the single-rank CSR.  The
    local range search is the CPU oracle here (the plumbing under test is device-agnostic); q is odd so the blocks
    differ in length, and one rank's block has queries without results."""
    script = tmp_path / "shard_worker.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys
        sys.path.insert(0, {ROOT!r})
        import numpy as np, torch, torch.distributed as dist
        import oracle
        from paper_2402_00665_b200 import sharded, workloads
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        w = workloads.make("C2", n=20000, q=1001, radius=0.03)
        queries = w.queries.copy()
        queries[:300, 3] = 0.0                                   # rank 0's block starts with empty rows
        o = oracle.build_bvh(w.prims, w.morton_bits)             # replicated tree: same deterministic build on both ranks
        def local_query(block):
            off, idx = oracle.query_spheres_tree(o, block.numpy())
            return torch.from_numpy(off), torch.from_numpy(idx)
        csr = sharded.sharded_query(local_query, torch.from_numpy(queries))
        lo, hi = sharded.block_bounds(1001, rank, world)
        assert (csr.q_lo, csr.q_hi) == (lo, hi) and csr.offsets.numel() == hi - lo + 1
        goff, gidx = sharded.gather_global(csr, 1001)
        ooff, oidx = oracle.query_spheres_tree(o, queries)       # single rank, whole batch
        assert np.array_equal(goff.numpy(), ooff) and np.array_equal(gidx.numpy(), oidx)
        assert int(csr.offsets[0]) == int(ooff[lo]) and int(csr.offsets[-1]) == int(ooff[hi])
        assert np.array_equal(csr.indices.numpy(), oidx[ooff[lo]:ooff[hi]])
        assert csr.nnz_total == int(ooff[-1]) and sum(csr.nnz_per_rank) == csr.nnz_total
        nodes = torch.full((64,), float(rank + 1))
        sharded.replicate_nodes(nodes, src=0)
        assert float(nodes[0]) == 1.0
        open(os.path.join({str(tmp_path)!r}, f"ok{{rank}}"), "w").write("ok")
        dist.destroy_process_group()
    """))
    r = _torchrun([str(script)], port=29619)
    assert r.returncode == 0, r.stderr[-3000:]
    assert (tmp_path / "ok0").exists() and (tmp_path / "ok1").exists()


def test_block_bounds_cover_the_batch():
    from paper_2402_00665_b200 import sharded

    for q in (0, 1, 7, 8, 1001, 1 << 20):
        for world in (1, 2, 3, 8):
            b = [sharded.block_bounds(q, r, world) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == q
            assert all(b[r][1] == b[r + 1][0] for r in range(world - 1))
            assert max(hi - lo for lo, hi in b) - min(hi - lo for lo, hi in b) <= 1
