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
