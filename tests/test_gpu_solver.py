"""GPU parity of SURVEY 8(f) item 3 (include/nk.h "assembly and solver"): gather / scatter against their
definition, the assembled Helmholtz apply against the oracle's dense assembled matrix, and the conjugate-gradient
solve against a direct solve of that matrix."""
import numpy as np
import pytest
import torch

import nk_cases as K
from oracle import nk_oracle as o
from workloads import assembly as asm
from workloads import synthetic as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nk():
    import paper_2606_20917_b200 as nk
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return nk


def setup(nk, n, P, deformed):
    el = K.element(o.HEX, P)
    A, J = K.geometry(o.HEX, P, n, deformed)
    basis = nk.Basis(o.HEX, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    l2g, ng = asm.hex_l2g(n, P)
    return el, A, J, basis, geom, l2g, ng


def test_gather_scatter_definition(nk):
    n, P = 3, 3
    l2g, ng = asm.hex_l2g(n, P)
    rng = np.random.Generator(np.random.Philox(7))
    sign = torch.from_numpy(rng.choice(np.array([-1, 1], dtype=np.int8), size=tuple(l2g.shape)))
    for sg in (None, sign):
        gs = nk.GatherScatter(l2g, ng, sg)
        u = torch.from_numpy(rng.standard_normal(ng)).cuda()
        loc = torch.full(tuple(l2g.shape), float("nan"), dtype=torch.float64, device="cuda")
        nk.gs_gather(gs, u, loc)
        s = np.ones(l2g.shape) if sg is None else sg.numpy().astype(np.float64)
        assert np.array_equal(loc.cpu().numpy(), s * u.cpu().numpy()[l2g.numpy()])            # bit-exact
        v = torch.from_numpy(rng.standard_normal(tuple(l2g.shape))).cuda()
        out = torch.full((ng,), float("nan"), dtype=torch.float64, device="cuda")
        nk.gs_scatter_add(gs, v, out)
        ref = np.zeros(ng)
        flat, vals = l2g.numpy().ravel(), (s * v.cpu().numpy()).ravel()
        for i in range(flat.size):          # the definition, in the library's (increasing local index) order: bit-exact
            ref[flat[i]] += vals[i]
        assert np.array_equal(out.cpu().numpy(), ref)
        # adjointness <Q u, v> = <u, Q^T v>
        assert abs(float((loc * v).sum()) - float((u * out).sum())) <= 1e-12 * float(loc.abs().sum())


@pytest.mark.parametrize("precond", [0, 1])
@pytest.mark.parametrize("P,deformed", [(2, False), (3, True), (4, True)])
def test_assembled_apply_and_cg_against_dense_oracle(nk, P, deformed, precond):
    n, lam = 2, 1.75
    el, A, J, basis, geom, l2g, ng = setup(nk, n, P, deformed)
    G = o.assembled_matrix(el, A.numpy(), J.numpy(), lam, l2g.numpy(), ng)
    gs = nk.GatherScatter(l2g, ng)
    rng = np.random.Generator(np.random.Philox(11 + P))
    u = rng.standard_normal(ng)
    out = torch.full((ng,), float("nan"), dtype=torch.float64, device="cuda")
    nk.assembled_helmholtz_apply(basis, geom, gs, lam, torch.from_numpy(u).cuda(), out)
    ref = G @ u
    assert np.abs(out.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
    # CG against the direct solve of the oracle's matrix
    b = rng.standard_normal(ng)
    x = torch.zeros(ng, dtype=torch.float64, device="cuda")
    rtol = 1e-10      # unpreconditioned CG on the modified basis (cond ~ 1e3..1e5 here): the recursive residual stalls near 1e-12
    iters, rel = nk.cg_solve(basis, geom, gs, lam, torch.from_numpy(b).cuda(), x, rtol=rtol, maxit=20 * ng, precond=precond)
    assert rel <= rtol and 0 < iters < 20 * ng
    if precond:    # the cached diagonal is the diagonal of the oracle's matrix
        it1, _ = nk.cg_solve(basis, geom, gs, lam, torch.from_numpy(np.diag(G).copy()).cuda(), torch.zeros_like(x), rtol=0.5, maxit=1,
                             precond=precond)
        assert it1 <= 1
    xs = np.linalg.solve(G, b)
    cond = np.linalg.cond(G)
    assert np.abs(x.cpu().numpy() - xs).max() <= 10 * cond * rtol * np.abs(xs).max(), (iters, rel, cond)
    # the returned residual is the true residual (computed with the oracle's matrix)
    r = b - G @ x.cpu().numpy()
    assert np.linalg.norm(r) <= 10 * rtol * np.linalg.norm(b)
    # reproducible bit for bit, and a converged start returns at once
    x2 = torch.zeros(ng, dtype=torch.float64, device="cuda")
    it2, rel2 = nk.cg_solve(basis, geom, gs, lam, torch.from_numpy(b).cuda(), x2, rtol=rtol, maxit=20 * ng, precond=precond)
    assert it2 == iters and torch.equal(x, x2)
    it3, _ = nk.cg_solve(basis, geom, gs, lam, torch.from_numpy(b).cuda(), x2, rtol=1e-8, maxit=10)
    assert it3 == 0


@pytest.mark.parametrize("P", [2, 4])
def test_poisson_with_dirichlet_boundary(nk, P):
    """lambda = 0 with the boundary dofs constrained (nk_gs_set_constrained): the assembled apply and the CG solve against
    the oracle's constrained matrix; removing the constraints restores the plain operator."""
    n = 2
    el, A, J, basis, geom, l2g, ng = setup(nk, n, P, True)
    bd = asm.hex_boundary_dofs(n, P)
    L = o.assembled_matrix(el, A.numpy(), J.numpy(), 0.0, l2g.numpy(), ng)
    Lc = o.constrained_matrix(L, bd.numpy())
    gs = nk.GatherScatter(l2g, ng)
    gs.set_constrained(bd)
    rng = np.random.Generator(np.random.Philox(31 + P))
    u = rng.standard_normal(ng)
    out = torch.full((ng,), float("nan"), dtype=torch.float64, device="cuda")
    nk.assembled_helmholtz_apply(basis, geom, gs, 0.0, torch.from_numpy(u).cuda(), out)
    ref = Lc @ u
    assert np.abs(out.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
    b = rng.standard_normal(ng)
    b[bd.numpy()] = 0.0                                             # homogeneous conditions
    for precond in (0, 1):
        x = torch.zeros(ng, dtype=torch.float64, device="cuda")
        iters, rel = nk.cg_solve(basis, geom, gs, 0.0, torch.from_numpy(b).cuda(), x, rtol=1e-10, maxit=20 * ng, precond=precond)
        xs = np.linalg.solve(Lc, b)
        assert rel <= 1e-10 and float(x[bd.cuda()].abs().max()) == 0.0
        assert np.abs(x.cpu().numpy() - xs).max() <= 10 * np.linalg.cond(Lc) * 1e-10 * np.abs(xs).max()
    gs.set_constrained(torch.zeros(0, dtype=torch.int64))
    nk.assembled_helmholtz_apply(basis, geom, gs, 0.0, torch.from_numpy(u).cuda(), out)
    ref = L @ u
    assert np.abs(out.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
    with pytest.raises(nk.NkError):
        gs.set_constrained(torch.tensor([ng], dtype=torch.int64))


def test_cg_larger_mesh_residual(nk):
    """a mesh the dense oracle cannot hold (16^3 deformed hexes, P4, 2.7e5 dofs): CG converges and the residual,
    recomputed through the parity-tested assembled apply, matches the one the solver reports."""
    n, P, lam = 16, 4, 1.0
    dev = torch.device("cuda", 0)
    basis = nk.Basis(o.HEX, P)
    v0, E = wl.hex_mesh(n, device=dev)
    A, J = wl.sinusoidal_factors(v0, E, basis.points().to(dev))
    geom = nk.Geom(basis, A, J, True, streams=nk.Geom.METRIC)
    l2g, ng = asm.hex_l2g(n, P)
    gs = nk.GatherScatter(l2g, ng)
    b = wl.coefficients(5, 1, ng).reshape(ng).to(dev)
    x = torch.zeros_like(b)
    iters, rel = nk.cg_solve(basis, geom, gs, lam, b, x, rtol=1e-8, maxit=20000, precond=nk.PRECOND_JACOBI)
    assert rel <= 1e-8 and iters < 3000
    Ax = torch.empty_like(b)
    nk.assembled_helmholtz_apply(basis, geom, gs, lam, x, Ax)
    assert float((b - Ax).norm() / b.norm()) <= 2e-8
    print("CG 16^3 deformed hex P4, %d dofs: %d iterations, relative residual %.2e" % (ng, iters, rel))


def test_solver_errors(nk):
    el, A, J, basis, geom, l2g, ng = setup(nk, 2, 2, False)
    with pytest.raises(nk.NkError) as ei:                        # entry out of range
        bad = l2g.clone()
        bad[0, 0] = ng
        nk.GatherScatter(bad, ng)
    assert ei.value.code == 1
    gs = nk.GatherScatter(l2g, ng)
    other = nk.Basis(o.HEX, 3)
    x = torch.zeros(ng, dtype=torch.float64, device="cuda")
    y = torch.ones(ng, dtype=torch.float64, device="cuda")
    code = nk.lib.nk_cg_solve(other.h, geom.h, gs.h, 1.0, y.data_ptr(), x.data_ptr(), 0, 1e-8, 10, None, None, None)
    assert code == 3                                             # NK_ERR_SHAPE_MISMATCH: map of another block
    code = nk.lib.nk_cg_solve(basis.h, geom.h, gs.h, 1.0, x.data_ptr(), x.data_ptr(), 0, 1e-8, 10, None, None, None)
    assert code == 1                                             # rhs and x alias
    code = nk.lib.nk_cg_solve(basis.h, geom.h, gs.h, 1.0, y.data_ptr(), x.data_ptr(), 7, 1e-8, 10, None, None, None)
    assert code == 1                                             # unknown preconditioner
    it, rel = nk.cg_solve(basis, geom, gs, 1.0, torch.zeros_like(x), y, rtol=1e-8, maxit=10)
    assert it == 0 and float(y.abs().max()) == 0.0               # rhs = 0 -> x = 0


# ---- the assembled system on a mesh split over ranks (include/nk.h: nk_part_*) ----
import threading


def _run_ranks(world, fn):
    """runs fn(rank) on `world` host threads (the library calls release the GIL; the all-reduce callbacks meet at a
    barrier) and re-raises the first exception.  The ranks' KERNELS never wait for one another: each thread synchronises
    its stream before the host-side rendezvous."""
    err, th = [None] * world, []

    def body(r):
        try:
            torch.cuda.set_device(0)
            fn(r)
        except BaseException as e:      # noqa: BLE001 -- reported in the main thread
            err[r] = e
    for r in range(world):
        th.append(threading.Thread(target=body, args=(r,)))
        th[-1].start()
    for t in th:
        t.join(timeout=300)
    assert not any(t.is_alive() for t in th), "a rank did not finish"
    for e in err:
        if e is not None:
            raise e


class _HostAllreduce:
    """in-process all-reduce over `world` threads: every rank hands in its tensor, the last one to arrive sums them in a
    fixed order and writes the sum back to all; calls are matched by a barrier (all ranks make the same sequence)."""

    def __init__(self, world):
        self.world, self.bar, self.t, self.calls = world, threading.Barrier(world), [None] * world, 0

    def make(self, rank):
        def f(t):
            torch.cuda.current_stream().synchronize()      # my contribution is complete
            self.t[rank] = t
            if self.bar.wait(timeout=120) == 0:
                s = self.t[0].clone()
                for k in range(1, self.world):
                    s += self.t[k]
                for k in range(self.world):
                    self.t[k].copy_(s)
                torch.cuda.synchronize()
                self.calls += 1
            self.bar.wait(timeout=120)
        return f


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("precond,dirichlet", [(0, False), (1, False), (1, True)])
def test_partitioned_apply_and_cg_against_the_whole_mesh(nk, world, precond, dirichlet):
    """a 3^3 deformed hex mesh at P3 cut into `world` element ranges (workloads.assembly.partition_l2g): the partitioned
    operator and CG solve of every rank against the oracle's dense matrix of the WHOLE mesh and against nk_cg_solve on
    one rank; Jacobi uses the whole mesh's diagonal; Dirichlet dofs on the cut stay fixed."""
    n, P = 3, 3
    lam = 0.0 if dirichlet else 1.75
    el, A, J, basis, geom, l2g, ng = setup(nk, n, P, True)
    G = o.assembled_matrix(el, A.numpy(), J.numpy(), lam, l2g.numpy(), ng)
    bd = asm.hex_boundary_dofs(n, P)
    if dirichlet:
        G = o.constrained_matrix(G, bd.numpy())
    rng = np.random.Generator(np.random.Philox(77 + world))
    u, b = rng.standard_normal(ng), rng.standard_normal(ng)
    if dirichlet:
        b[bd.numpy()] = 0.0
    xs = np.linalg.solve(G, b)
    rtol = 1e-10
    # one rank, whole mesh: the iteration count to reproduce
    gs1 = nk.GatherScatter(l2g, ng)
    if dirichlet:
        gs1.set_constrained(bd)
    x1 = torch.zeros(ng, dtype=torch.float64, device="cuda")
    it1, _ = nk.cg_solve(basis, geom, gs1, lam, torch.from_numpy(b).cuda(), x1, rtol=rtol, maxit=20 * ng, precond=precond)
    parts = asm.partition_l2g(l2g, ng, world)
    assert sum(p["range"][1] - p["range"][0] for p in parts) == n ** 3 and parts[0]["n_interface"] > 0
    comm = _HostAllreduce(world)
    ranks = []
    for r, p in enumerate(parts):
        lo, hi = p["range"]
        g_r = nk.Geom(basis, A[lo:hi].contiguous().cuda(), J[lo:hi].contiguous().cuda(), True)
        gs_r = nk.GatherScatter(p["l2g"], p["glob"].numel())
        if dirichlet:
            isbd = torch.zeros(ng, dtype=torch.bool)
            isbd[bd] = True
            gs_r.set_constrained(torch.nonzero(isbd[p["glob"]]).reshape(-1).contiguous())
        part = nk.Partition(gs_r, p["shared_dof"], p["shared_slot"], p["shared_mult"], p["n_interface"], comm.make(r))
        ranks.append((g_r, gs_r, part, p["glob"].numpy()))
    out, sol, its = [None] * world, [None] * world, [None] * world

    def rank_body(r):
        g_r, gs_r, part, glob = ranks[r]
        y = torch.full((glob.size,), float("nan"), dtype=torch.float64, device="cuda")
        nk.part_assembled_helmholtz_apply(basis, g_r, part, lam, torch.from_numpy(u[glob]).cuda(), y)
        out[r] = y.cpu().numpy()
        x = torch.zeros(glob.size, dtype=torch.float64, device="cuda")
        its[r] = nk.part_cg_solve(basis, g_r, part, lam, torch.from_numpy(b[glob]).cuda(), x, rtol=rtol, maxit=20 * ng, precond=precond)
        sol[r] = x.cpu().numpy()
    _run_ranks(world, rank_body)
    ref = G @ u
    cond = np.linalg.cond(G)
    for r in range(world):
        glob = ranks[r][3]
        assert np.abs(out[r] - ref[glob]).max() <= 1e-12 * np.abs(ref).max(), r
        assert its[r] == its[0] and its[r][1] <= rtol                      # identical on every rank
        assert np.abs(sol[r] - xs[glob]).max() <= 10 * cond * rtol * np.abs(xs).max(), (r, its[r], cond)
        if dirichlet:
            assert np.abs(sol[r][np.isin(glob, bd.numpy())]).max() == 0.0
    # same Krylov iteration as the one-rank solve (sums in another order: the count may differ by a step or two)
    assert abs(its[0][0] - it1) <= max(3, it1 // 20), (its[0], it1)
    assert comm.calls > 3 * its[0][0]                                      # interface + two scalar all-reduces per iteration


def test_partition_of_one_rank_equals_cg_solve(nk):
    """world = 1: no shared dofs, the all-reduce is the identity: nk_part_cg_solve reproduces nk_cg_solve's iteration."""
    el, A, J, basis, geom, l2g, ng = setup(nk, 2, 3, True)
    gs = nk.GatherScatter(l2g, ng)
    p = asm.partition_l2g(l2g, ng, 1)[0]
    assert p["n_interface"] == 0 and torch.equal(p["l2g"], l2g)
    calls = []
    part = nk.Partition(gs, p["shared_dof"], p["shared_slot"], p["shared_mult"], 0, lambda t: calls.append(t.numel()))
    b = torch.from_numpy(np.random.Generator(np.random.Philox(5)).standard_normal(ng)).cuda()
    x0, x1 = torch.zeros_like(b), torch.zeros_like(b)
    it0, rel0 = nk.cg_solve(basis, geom, gs, 1.0, b, x0, rtol=1e-10, maxit=5000, precond=1)
    it1, rel1 = nk.part_cg_solve(basis, geom, part, 1.0, b, x1, rtol=1e-10, maxit=5000, precond=1)
    assert abs(it1 - it0) <= 2 and rel1 <= 1e-10
    assert float((x1 - x0).abs().max()) <= 1e-8 * float(x0.abs().max())
    assert set(calls) <= {1, 2}                                            # only the scalar reductions were called
    with pytest.raises(nk.NkError):                                        # a slot listed twice
        nk.Partition(gs, torch.tensor([0, 1]), torch.tensor([0, 0]), torch.tensor([2, 2], dtype=torch.int32), 2, lambda t: None)
