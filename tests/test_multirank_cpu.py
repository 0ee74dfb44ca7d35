"""World-size-2 test (gloo, CPU) of the multi-GPU host logic: elements shard into
contiguous ranges with NO data-path collective, every rank's shard result equals the corresponding slice of
the single-process result, and the reported time is the max over ranks."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import nk_oracle as o
from workloads import configs as cfgs
from workloads import synthetic as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        title, op, blocks = cfgs.config_blocks(2, scale=0.1)          # 3^3 deformed hexes, P4
        b = cfgs.shard(blocks[0], rank, world)
        lo, hi = b["range"]
        el = o.Element(b["shape"], b["P"], b["P"] + 2)
        A, J = cfgs.block_factors(b, torch.tensor(el.xi))
        x = wl.coefficients(b["seed"], blocks[0]["v0"].shape[0], el.Nm)[lo:hi]
        y = o.helmholtz(el, A.numpy(), J.numpy(), b["lam"], x.numpy())
        # bench.py's reduction: max over ranks of the per-rank time, sum over ranks of the DoF
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        n = torch.tensor([float(y.size)], dtype=torch.float64)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
        dist.barrier()
        np.save(os.path.join(out, "y%d.npy" % rank), y)
        np.save(os.path.join(out, "m%d.npy" % rank), np.array([lo, hi, t.item(), n.item()]))
    finally:
        dist.destroy_process_group()


def test_shards_cover_the_block_and_reduce(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    title, op, blocks = cfgs.config_blocks(2, scale=0.1)
    b = blocks[0]
    el = o.Element(b["shape"], b["P"], b["P"] + 2)
    A, J = cfgs.block_factors(b, torch.tensor(el.xi))
    ne = J.shape[0]
    x = wl.coefficients(b["seed"], ne, el.Nm)
    ref = o.helmholtz(el, A.numpy(), J.numpy(), b["lam"], x.numpy())
    got = np.concatenate([np.load(tmp_path / ("y%d.npy" % r)) for r in range(world)])
    meta = [np.load(tmp_path / ("m%d.npy" % r)) for r in range(world)]
    assert meta[0][0] == 0 and meta[0][1] == meta[1][0] and meta[1][1] == ne        # contiguous cover
    assert all(m[2] == 10.0 + world - 1 for m in meta)                              # max over ranks
    assert all(m[3] == ref.size for m in meta)                                      # whole-job DoF
    np.testing.assert_array_equal(got, ref)       # element-local work: bit-identical to the unsharded run


def test_shard_ranges_ragged():
    title, op, blocks = cfgs.config_blocks(3, scale=0.1)
    ne = blocks[0]["v0"].shape[0]
    for world in (2, 3, 8):
        r = [cfgs.shard(blocks[0], k, world)["range"] for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == ne
        assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
        assert max(h - l for l, h in r) - min(h - l for l, h in r) <= 1
