"""GPU parity of the RUN-TIME SPECIALISED sum-factorised kernels (the paper's JIT):
bases outside the prebuilt Q = P+2 table -- other quadrature orders, tets and prisms of order 9 -- whose kernels NVRTC
instantiates on first use (csrc/nk_jit.cu) from the same template as the prebuilt ones.  Same gate as every other
parity test: normwise relative error per element <= 1e-12 against the plain CPU oracle, through the C-ABI."""
import numpy as np
import pytest
import torch

import nk_cases as K
from oracle import nk_oracle as o
from workloads import synthetic as wl

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def nk():
    import paper_2606_20917_b200 as nk
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return nk


def run_case(nk, shape, P, Q, n, deformed, ops, lam, take=None, zhi=None, seed=wl.SEED0 + 21, form=1):
    el = K.element(shape, P, Q)
    A, J = K.geometry(shape, P, n, deformed, take=take, zhi=zhi, xi=el.xi)
    ne = J.shape[0]
    basis = nk.Basis(shape, P, Q)
    assert basis.num_modes == el.Nm and basis.num_points == el.Nq == Q ** 3
    assert np.abs(basis.points().numpy() - el.xi).max() <= 1e-14
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    old = nk.get_affine_simplex_form()
    nk.set_affine_simplex_form(form)      # 1: the sum-factorised kernel also on affine simplices
    try:
        errs = {}
        for op in ops:
            x = K.make_input(op, seed, ne, el)
            ref = K.oracle_op(op, el, A, J, lam, x)
            got = K.gpu_op(nk, op, basis, geom, lam, x)
            assert np.isfinite(got).all(), (op, "non-finite output")
            errs[op] = K.op_err(op, got, ref)
    finally:
        nk.set_affine_simplex_form(old)
    bad = {k: v for k, v in errs.items() if not v <= TOL}
    assert not bad, "shape %d P %d Q %d def %d: %r" % (shape, P, Q, deformed, errs)


# (shape, P, Q): under-integrated (Q = P+1), over-integrated (Q = P+3, P+4) and a long line on a low order
CASES = [(o.HEX, 4, 5), (o.HEX, 4, 7), (o.HEX, 2, 6), (o.HEX, 7, 8), (o.TET, 3, 6), (o.TET, 4, 5), (o.PRISM, 3, 4), (o.PRISM, 4, 7)]


@pytest.mark.parametrize("shape,P,Q", CASES)
@pytest.mark.parametrize("deformed", [False, True])
def test_every_operator_at_other_quadrature_orders(nk, shape, P, Q, deformed):
    """all seven operators on several groups plus a ragged tail; the kernel counter shows that they were specialised at
    run time."""
    k0, _ = nk.jit_stats()
    full = K.mesh(shape, 3)[0].shape[0]
    run_case(nk, shape, P, Q, 3, deformed, K.OPS, lam=1.75, take=torch.arange(full - 5))
    k1, ms = nk.jit_stats()
    assert k1 >= k0, (k0, k1)
    print("shape %d P %d Q %d deformed %d: %d kernels specialised, %.0f ms in NVRTC so far" % (shape, P, Q, deformed, k1, ms))


def test_run_time_kernels_are_counted(nk):
    """a basis no other test uses: its first Helmholtz apply compiles exactly one kernel, the second none."""
    k0, _ = nk.jit_stats()
    run_case(nk, o.HEX, 3, 7, 2, True, ("helmholtz",), lam=0.5)
    k1, _ = nk.jit_stats()
    run_case(nk, o.HEX, 3, 7, 2, True, ("helmholtz",), lam=0.25)
    k2, _ = nk.jit_stats()
    assert k1 == k0 + 1 and k2 == k1, (k0, k1, k2)


@pytest.mark.parametrize("shape", [o.TET, o.PRISM])
def test_tet_and_prism_orders_9_and_10(nk, shape):
    """orders beyond the prebuilt simplex table (P <= 8; SURVEY section 5 asked for 1..10): P = 9 with
    Q = 11 and P = 10 with Q = 12 (one copy of the psi^b tables there: two do not fit the kernel-parameter space), affine
    (sum-factorised form) and deformed."""
    for deformed in (False, True):
        run_case(nk, shape, 9, 11, 2, deformed, ("helmholtz", "bwdtrans", "iprod", "physderiv", "iprod_deriv"), lam=10.0, zhi=1)
        run_case(nk, shape, 10, 12, 2, deformed, ("helmholtz", "bwdtrans", "iprod_deriv"), lam=10.0, zhi=1)


def test_specialised_equals_prebuilt_template(nk):
    """Q = P+3 and Q = P+2 integrate the affine hex mass and Laplacian exactly (degree 2P <= 2Q-3): the specialised
    kernel at Q = P+3 must reproduce the prebuilt one at Q = P+2 to rounding -- two instantiations of one template."""
    P = 3
    el = K.element(o.HEX, P)
    A, J = K.geometry(o.HEX, P, 3, False)
    x = K.make_input("helmholtz", wl.SEED0 + 22, J.shape[0], el)
    out = []
    for Q in (P + 2, P + 3):
        basis = nk.Basis(o.HEX, P, Q)
        geom = nk.Geom(basis, A.cuda(), J.cuda(), False)
        out.append(K.gpu_op(nk, "helmholtz", basis, geom, 2.0, x))
    assert K.normwise_err(out[1], out[0]) <= 1e-13


def test_unsupported_triples_are_refused(nk):
    for shape, P, Q in ((o.HEX, 3, 3), (o.HEX, 11, 13), (o.TET, 10, 13), (o.HEX, 4, 13), (o.PRISM, 11, 12)):
        with pytest.raises(nk.NkError) as ei:
            nk.Basis(shape, P, Q)
        assert ei.value.code == 2      # NK_ERR_UNSUPPORTED


def test_hp_mixed_batch_in_one_call(nk):
    """SURVEY 8(f) item 2, second half: a batch whose blocks differ in shape, order, quadrature order and geometry kind, as in
    hp-adaptivity, applied by ONE nk_helmholtz_apply_blocks call -- prebuilt sum-factorised, Kronecker, reference-matrix
    (DMMA) and run-time specialised kernels side by side on forked streams; every block against the oracle."""
    lam = 2.5
    spec = [(o.HEX, 2, 4, True, 3), (o.HEX, 5, 7, False, 2), (o.TET, 3, 5, True, 2), (o.PRISM, 4, 7, True, 2),
            (o.TET, 6, 8, False, 2), (o.HEX, 3, 6, True, 2), (o.PRISM, 1, 3, False, 3)]
    blocks, refs = [], []
    for i, (shape, P, Q, deformed, n) in enumerate(spec):
        el = K.element(shape, P, Q)
        A, J = K.geometry(shape, P, n, deformed, xi=el.xi)
        basis = nk.Basis(shape, P, Q)
        geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
        x = wl.coefficients(wl.SEED0 + 40 + i, J.shape[0], el.Nm)
        y = torch.full_like(x, float("nan")).cuda()
        blocks.append((basis, geom, x.cuda(), y))
        refs.append(o.helmholtz(el, A.numpy(), J.numpy(), lam, x.numpy()))
    nk.helmholtz_apply_blocks(blocks, lam)
    torch.cuda.synchronize()
    for (shape, P, Q, deformed, n), (b, g, x, y), ref in zip(spec, blocks, refs):
        assert K.normwise_err(y.cpu().numpy(), ref) <= TOL, (shape, P, Q, deformed)


@pytest.mark.parametrize("shape,P,Q,deformed", [(o.HEX, 4, 7, True), (o.HEX, 3, 4, False), (o.PRISM, 3, 6, True)])
def test_every_entry_point_serves_a_specialised_basis(nk, shape, P, Q, deformed):
    """the other entries of include/nk.h on a run-time specialised basis: the multi-field call (one launch, bit-identical
    to the single-field one), the host entry (chunked launches over group ranges), repeatability, and, on hexes, the
    assembled apply and CG solve; the entry that must not allocate refuses such a basis."""
    from workloads import assembly as asm
    lam = 1.25
    el = K.element(shape, P, Q)
    full = K.mesh(shape, 3)[0].shape[0]
    take = torch.arange(full - (0 if shape == o.HEX else 3))
    A, J = K.geometry(shape, P, 3, deformed, take=take, xi=el.xi)
    ne = J.shape[0]
    basis = nk.Basis(shape, P, Q)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    xs = [wl.coefficients(300 + f, ne, el.Nm) for f in range(3)]
    refs = [o.helmholtz(el, A.numpy(), J.numpy(), lam, x.numpy()) for x in xs]
    dx = [x.cuda() for x in xs]
    dy = [torch.full_like(x, float("nan")) for x in dx]
    nk.helmholtz_apply_fields(basis, geom, lam, dx, dy)          # compiles the multi-field instantiation
    n0 = nk.launch_count()
    nk.helmholtz_apply_fields(basis, geom, lam, dx, dy)
    assert nk.launch_count() == n0 + 1
    torch.cuda.synchronize()
    for f in range(3):
        assert K.normwise_err(dy[f].cpu().numpy(), refs[f]) <= TOL
        y1 = torch.empty_like(dx[f])
        nk.helmholtz_apply(basis, geom, lam, dx[f], y1)
        y2 = torch.empty_like(dx[f])
        nk.helmholtz_apply(basis, geom, lam, dx[f], y2)
        assert torch.equal(y1, dy[f]) and torch.equal(y1, y2)
    xh = xs[0].pin_memory()
    yh = torch.full_like(xh, float("nan")).pin_memory()
    nk.helmholtz_apply_host(basis, geom, lam, xh, yh)
    assert K.normwise_err(yh.numpy(), refs[0]) <= TOL
    if shape == o.HEX:
        l2g, ng = asm.hex_l2g(3, P)
        G = o.assembled_matrix(el, A.numpy(), J.numpy(), lam, l2g.numpy(), ng)
        gs = nk.GatherScatter(l2g, ng)
        rng = np.random.Generator(np.random.Philox(9))
        u, b = rng.standard_normal(ng), rng.standard_normal(ng)
        out = torch.full((ng,), float("nan"), dtype=torch.float64, device="cuda")
        nk.assembled_helmholtz_apply(basis, geom, gs, lam, torch.from_numpy(u).cuda(), out)
        ref = G @ u
        assert np.abs(out.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
        x = torch.zeros(ng, dtype=torch.float64, device="cuda")
        iters, rel = nk.cg_solve(basis, geom, gs, lam, torch.from_numpy(b).cuda(), x, rtol=1e-10, maxit=20 * ng, precond=1)
        xsol = np.linalg.solve(G, b)
        assert rel <= 1e-10 and np.abs(x.cpu().numpy() - xsol).max() <= 10 * np.linalg.cond(G) * 1e-10 * np.abs(xsol).max()
        with pytest.raises(nk.NkError) as ei:
            nk.assembled_helmholtz_apply_static(basis, geom, gs, lam, torch.from_numpy(u).cuda(), out)
        assert ei.value.code == 2
