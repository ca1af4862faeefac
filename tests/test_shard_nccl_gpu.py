"""Row shards of ONE image over two GPUs with the real data plane: NCCL all-gathers between the kernels of
fitrig_shard_export / fitrig_shard_import (and the eta pair of the frequency branch), one process per GPU.

Needs two CUDA devices; on a one-GPU box the test is skipped (the protocol's host side is covered over gloo in
test_shard_gloo.py, the kernels by the one-GPU shard tests of test_parity_gpu*.py).
"""
import os
import socket

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, H, W, L, tile, tau, branch, ret):
    import torch.distributed as dist

    import paper_2509_21754_b200 as fitrig
    import synth
    from paper_2509_21754_b200 import shard

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        dev = f"cuda:{rank}"
        cfg = synth.scaled(synth.CONFIGS["imgfreq" if branch else "tiny"], H, W, L=L)
        full = synth.make_stack(cfg, device=dev)[0] if rank == 0 else torch.empty((L, H, W), dtype=torch.float32, device=dev)
        dist.broadcast(full, 0)  # the same image on every rank, whatever the devices' generators do
        side = torch.cuda.Stream(device=dev)  # a stream other than the one the collective runs on
        with shard.ShardedContext(H, W, L, rank, world, device=rank, tile=tile, branch=branch) as sc:
            rows = full[:, sc.r0:sc.r1].contiguous()
            torch.cuda.synchronize()
            sc.tlisi(rows, None, side)
            cands, n = sc.detect(tau, 1 << 16, side)
            merged = sc.gather(cands, dev) if branch == 0 else np.concatenate(shard.gather_candidates(cands, dev))
            q = sc.ctx.get_map(0)
            M, mu, sd = sc.ctx.get_stats()
            r0, r1 = sc.r0, sc.r1
            # the same image from (pinned) host memory: every rank streams its own rows of the whole snapshots
            host = full.cpu().pin_memory()
            sc.stream([host[s] for s in range(L)], None, side)
            cands_s, n_s = sc.detect(tau, 1 << 16, side)
            assert n_s == n and np.array_equal(cands_s, cands) and np.array_equal(sc.ctx.get_map(0), q)
        with fitrig.Context(H, W, L, device=rank, tile=tile, branch=branch) as ctx:
            ctx.tlisi(full)
            ref_c, ref_n = ctx.detect(tau)
            ref_q = ctx.get_map(0)
            ref_M, ref_mu, ref_sd = ctx.get_stats()
        ty0 = r0 // tile
        assert np.array_equal(q, ref_q[:, ty0:ty0 + q.shape[1]])  # the shard's map: bit-identical rows of the whole map
        assert M == ref_M
        np.testing.assert_allclose(mu, ref_mu, rtol=1e-6)
        np.testing.assert_allclose(sd, ref_sd, rtol=1e-5)
        key = lambda c: {(int(r["snapshot"]), int(r["y"]), int(r["x"])) for r in c if abs(float(r["score"]) - tau) > 2e-4}
        assert key(merged) == key(ref_c) and ref_n > 0
        ret[rank] = len(merged)
    finally:
        dist.destroy_process_group()


@pytest.mark.skipif(not torch.cuda.is_available() or torch.cuda.device_count() < 2, reason="needs two CUDA devices")
@pytest.mark.parametrize("branch,H,W,tile,tau", [(0, 256, 256, 32, 3.0), (0, 250, 252, 16, 3.0), (1, 256, 256, 16, 2.0)])
def test_row_shards_over_nccl(branch, H, W, tile, tau):
    import torch.multiprocessing as mp
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), H, W, 12 if branch else 8, tile, tau, branch, ret), nprocs=2, join=True)
    assert len(ret) == 2 and len(set(ret.values())) == 1
