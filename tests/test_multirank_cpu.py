"""World-size-2 tests (gloo, CPU) of the multi-GPU host logic: elements shard into
contiguous ranges with NO data-path collective, every rank's shard result equals the corresponding slice of
the single-process result, and the reported time is the max over ranks; for the ASSEMBLED system the partition
bookkeeping (shared dofs, interface slots, multiplicities) that feeds nk_part_create drives a partitioned CG over
torch.distributed whose solution equals the dense solve of the whole mesh."""
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


def _cg_worker(rank, world, port, out):
    """partitioned CG in numpy with the algorithm of nk_part_cg_solve (include/nk.h): local operator = the oracle's dense
    matrix of the rank's elements, interface sum and weighted dot products over gloo all-reduces."""
    from workloads import assembly as asm
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, P, lam = 2, 2, 1.5
        el = o.Element(o.HEX, P, P + 2)
        v0, E = wl.hex_mesh(n)
        A, J = wl.sinusoidal_factors(v0, E, torch.tensor(el.xi))
        l2g, ng = asm.hex_l2g(n, P)
        p = asm.partition_l2g(l2g, ng, world)[rank]
        lo, hi = p["range"]
        nr = p["glob"].numel()
        Ar = o.assembled_matrix(el, A[lo:hi].numpy(), J[lo:hi].numpy(), lam, p["l2g"].numpy(), nr)
        sd, ss, ni = p["shared_dof"].numpy(), p["shared_slot"].numpy(), p["n_interface"]
        w = np.ones(nr)
        w[sd] = 1.0 / p["shared_mult"].numpy()

        def exchange(v):
            buf = torch.zeros(ni, dtype=torch.float64)
            buf[torch.from_numpy(ss)] = torch.from_numpy(v[sd])
            dist.all_reduce(buf)
            v[sd] = buf.numpy()[ss]
            return v

        def dot(a, b_):
            t = torch.tensor([float(np.sum(w * a * b_))], dtype=torch.float64)
            dist.all_reduce(t)
            return t.item()

        def apply(v):
            return exchange(Ar @ v)
        b = np.random.Generator(np.random.Philox(3)).standard_normal(ng)[p["glob"].numpy()]     # consistent on shared dofs
        x = np.zeros(nr)
        r = b - apply(x)
        pvec, rr, bn = r.copy(), dot(r, r), dot(b, b)
        it = 0
        while np.sqrt(rr / bn) > 1e-12 and it < 10 * ng:
            Ap = apply(pvec)
            alpha = rr / dot(pvec, Ap)
            x += alpha * pvec
            r -= alpha * Ap
            rn = dot(r, r)
            pvec = r + (rn / rr) * pvec
            rr = rn
            it += 1
        np.save(os.path.join(out, "x%d.npy" % rank), x)
        np.save(os.path.join(out, "g%d.npy" % rank), p["glob"].numpy())
    finally:
        dist.destroy_process_group()


def test_partitioned_cg_over_gloo_equals_the_dense_solve(tmp_path):
    from workloads import assembly as asm
    world, port = 2, _free_port()
    mp.spawn(_cg_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    n, P, lam = 2, 2, 1.5
    el = o.Element(o.HEX, P, P + 2)
    v0, E = wl.hex_mesh(n)
    A, J = wl.sinusoidal_factors(v0, E, torch.tensor(el.xi))
    l2g, ng = asm.hex_l2g(n, P)
    G = o.assembled_matrix(el, A.numpy(), J.numpy(), lam, l2g.numpy(), ng)
    b = np.random.Generator(np.random.Philox(3)).standard_normal(ng)
    xs = np.linalg.solve(G, b)
    seen = np.zeros(ng, dtype=bool)
    for r in range(world):
        x, glob = np.load(tmp_path / ("x%d.npy" % r)), np.load(tmp_path / ("g%d.npy" % r))
        assert np.abs(x - xs[glob]).max() <= 1e-9 * np.abs(xs).max()
        seen[glob] = True
    assert seen.all()


def test_partition_bookkeeping():
    from workloads import assembly as asm
    l2g, ng = asm.hex_l2g(3, 2)
    for world in (1, 2, 3, 5):
        parts = asm.partition_l2g(l2g, ng, world)
        held = np.zeros(ng, dtype=int)
        for p in parts:
            glob = p["glob"].numpy()
            held[glob] += 1
            lo, hi = p["range"]
            assert np.array_equal(glob[p["l2g"].numpy()], l2g[lo:hi].numpy())           # the rank's map, renumbered
        for p in parts:
            glob, sd = p["glob"].numpy(), p["shared_dof"].numpy()
            assert np.array_equal(held[glob[sd]], p["shared_mult"].numpy()) and (held[glob[sd]] >= 2).all()
            assert np.array_equal(np.sort(glob[sd]), glob[held[glob] > 1])              # exactly the dofs on the cuts
            assert p["n_interface"] == int((held > 1).sum())
        # the same global dof has the same slot on every rank
        slot = {}
        for p in parts:
            for gdof, sl in zip(p["glob"].numpy()[p["shared_dof"].numpy()], p["shared_slot"].numpy()):
                assert slot.setdefault(int(gdof), int(sl)) == int(sl)
        assert sorted(slot.values()) == list(range(parts[0]["n_interface"]))
