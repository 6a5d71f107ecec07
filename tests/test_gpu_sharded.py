"""NEXT-4 on the GPU (Algorithm 1 keeps no state across queries): one batch of queries
split over ranks against a replicated hierarchy, with the CUDA range search as the local search and CUDA tensors through
``sharded.assemble`` / ``gather_global``.  World size 1 in this process, and world size 2 as two processes that share
cuda:0 (gloo carries the two all-gathers; NCCL cannot put two ranks on one device).  The global CSR must equal the
oracle's CSR of the whole batch: uneven blocks, a block that starts with empty rows, fewer queries than ranks."""
from __future__ import annotations

import os
import subprocess
import sys
import textwrap

import numpy as np
import pytest

from paper_2402_00665_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_sharded_query_world_size_one_cuda(oracle_lib):
    from paper_2402_00665_b200 import binding, sharded

    w = W.make("C2", n=30_000, q=2_001, radius=0.03)
    queries = w.queries.copy()
    queries[:250, 3] = 0.0
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    bvh = binding.Bvh(w.n, w.morton_bits).build(torch.from_numpy(w.prims).cuda())
    csr = sharded.sharded_query(lambda blk: binding.query(bvh, blk), torch.from_numpy(queries).cuda())
    goff, gidx = sharded.gather_global(csr, queries.shape[0])
    ooff, oidx = oracle_lib.query_spheres_tree(o, queries)
    assert goff.is_cuda and gidx.is_cuda
    assert (csr.q_lo, csr.q_hi, csr.nnz_before, csr.nnz_total) == (0, queries.shape[0], 0, int(ooff[-1]))
    assert np.array_equal(goff.cpu().numpy(), ooff) and np.array_equal(gidx.cpu().numpy(), oidx)


def test_sharded_query_two_processes_one_gpu(tmp_path):
    script = tmp_path / "shard_gpu_worker.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys
        sys.path.insert(0, {ROOT!r})
        import numpy as np, torch, torch.distributed as dist
        import oracle
        from paper_2402_00665_b200 import binding, sharded, workloads
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        torch.cuda.set_device(0)
        w = workloads.make("C2", n=30000, q=1001, radius=0.03)
        queries = w.queries.copy()
        queries[:300, 3] = 0.0                                   # rank 0's block starts with rows without results
        o = oracle.build_bvh(w.prims, w.morton_bits)
        bvh = binding.Bvh(w.n, w.morton_bits).build(torch.from_numpy(w.prims).cuda())   # replicated: the same build on each rank
        for q in (1001, 1, 0):                                   # uneven blocks; fewer queries than ranks; an empty batch
            qs = torch.from_numpy(queries[:q]).cuda()
            csr = sharded.sharded_query(lambda blk: binding.query(bvh, blk), qs)
            lo, hi = sharded.block_bounds(q, rank, world)
            assert (csr.q_lo, csr.q_hi) == (lo, hi) and csr.offsets.numel() == hi - lo + 1 and csr.offsets.is_cuda
            goff, gidx = sharded.gather_global(csr, q)
            ooff, oidx = oracle.query_spheres_tree(o, queries[:q])
            assert np.array_equal(goff.cpu().numpy(), ooff), q
            assert np.array_equal(gidx.cpu().numpy(), oidx), q
            assert int(csr.offsets[0]) == int(ooff[lo]) and int(csr.offsets[-1]) == int(ooff[hi])
            assert np.array_equal(csr.indices.cpu().numpy(), oidx[ooff[lo]:ooff[hi]])
            assert csr.nnz_total == int(ooff[-1]) and sum(csr.nnz_per_rank) == csr.nnz_total
        # the hierarchy received from rank 0 instead of built locally: same bytes
        mine = bvh.nodes.clone()
        recv = torch.zeros_like(bvh.nodes) if rank else bvh.nodes
        host = recv.cpu()                                        # (gloo: through the host; under nccl the device buffer goes as is)
        sharded.replicate_nodes(host, src=0)
        assert torch.equal(host.cuda(), mine)
        open(os.path.join({str(tmp_path)!r}, f"ok{{rank}}"), "w").write("ok")
        dist.destroy_process_group()
    """))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29631", OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29631", str(script)]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert (tmp_path / "ok0").exists() and (tmp_path / "ok1").exists()
