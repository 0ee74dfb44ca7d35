"""GPU parity: every operator of include/nk.h, called through the C-ABI binding, against the
plain CPU oracle on the same seeded inputs.  Gate (north_star; A18): normwise relative
error per element <= 1e-12 in fp64."""
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


import contextlib


@contextlib.contextmanager
def simplex_form(nk, form):
    """forces the form of the affine simplex operators (nk_set_affine_simplex_form) for the duration of a block"""
    old = nk.get_affine_simplex_form()
    nk.set_affine_simplex_form(form)
    try:
        yield
    finally:
        nk.set_affine_simplex_form(old)


def run_case(nk, shape, P, n, deformed, ops, lam=1.0, take=None, seed=wl.SEED0, zhi=None):
    el = K.element(shape, P)
    A, J = K.geometry(shape, P, n, deformed, take=take, zhi=zhi)
    ne = J.shape[0]
    basis = nk.Basis(shape, P)
    assert basis.num_modes == el.Nm and basis.num_points == el.Nq
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    errs = {}
    for op in ops:
        x = K.make_input(op, seed, ne, el)
        ref = K.oracle_op(op, el, A, J, lam, x)
        got = K.gpu_op(nk, op, basis, geom, lam, x)
        assert np.isfinite(got).all(), (op, "non-finite output")
        errs[op] = K.op_err(op, got, ref)
    bad = {k: v for k, v in errs.items() if not v <= TOL}
    assert not bad, "shape %d P %d def %d: %r" % (shape, P, deformed, errs)
    return errs


def test_config1_hex_affine_P3_64_elements(nk):
    """BASELINE config 1 in full: BwdTrans, IProductWRTBase, Helmholtz lambda=1 (plus the rest)."""
    run_case(nk, o.HEX, 3, 4, False, K.OPS, lam=1.0, seed=wl.SEED0 + 1)


@pytest.mark.parametrize("shape", [o.HEX, o.TET, o.PRISM])
@pytest.mark.parametrize("deformed", [False, True])
def test_all_ops_P4_ragged(nk, shape, deformed):
    """several groups plus a ragged tail (nelem not a multiple of the interleave width)."""
    full = K.mesh(shape, 3)[0].shape[0]
    take = torch.arange(full - 5)
    run_case(nk, shape, 4, 3, deformed, K.OPS, lam=1.0, take=take, seed=wl.SEED0 + 2)


@pytest.mark.parametrize("shape", [o.TET, o.PRISM])
def test_all_ops_P4_ragged_sum_factorised_form(nk, shape):
    """the same on affine simplices with the sum-factorised kernels forced (form 1; the default on affine tets
    is the reference-matrix kernel)."""
    full = K.mesh(shape, 3)[0].shape[0]
    with simplex_form(nk, 1):
        run_case(nk, shape, 4, 3, False, K.OPS, lam=1.0, take=torch.arange(full - 5), seed=wl.SEED0 + 2)


@pytest.mark.parametrize("P", range(1, 11))
def test_config4_hex_psweep_mass_laplacian(nk, P):
    run_case(nk, o.HEX, P, 3 if P < 8 else 2, False, ("mass", "laplacian"), seed=wl.SEED0 + 4)


@pytest.mark.parametrize("P", range(1, 11))
def test_hex_affine_all_orders_helmholtz_bwd_iprod(nk, P):
    """Helmholtz (lambda != 1) on AFFINE hexes at every order: the coefficient-space kernel (nk_stage_lapkron.inc)
    with its lambda |J| term on both sides of the NK_LAPKRON_MAXNM switch, plus BwdTrans / IProduct at every order."""
    run_case(nk, o.HEX, P, 3 if P < 8 else 2, False, ("helmholtz", "bwdtrans", "iprod"), lam=2.75, seed=wl.SEED0 + 14)


@pytest.mark.parametrize("P", range(1, 11))
def test_hex_deformed_all_orders(nk, P):
    run_case(nk, o.HEX, P, 2, True, ("helmholtz", "physderiv", "iprod_deriv"), lam=0.7, seed=wl.SEED0 + 4)


@pytest.mark.parametrize("shape", [o.TET, o.PRISM])
@pytest.mark.parametrize("P", range(1, 9))
def test_simplex_all_orders(nk, shape, P):
    for deformed in (False, True):
        run_case(nk, shape, P, 2, deformed, ("bwdtrans", "iprod", "helmholtz", "physderiv", "iprod_deriv"),
                 lam=10.0, seed=wl.SEED0 + 5, zhi=1)


@pytest.mark.parametrize("shape", [o.TET, o.PRISM])
@pytest.mark.parametrize("P", [1, 2, 3])
def test_simplex_low_order_full_groups_and_tail(nk, shape, P):
    """low orders have wide interleaves (32 at P1 affine): at least two full groups plus a ragged tail."""
    full = K.mesh(shape, 4)[0].shape[0]          # 384 tets / 128 prisms
    take = torch.arange(full - 3)
    for deformed in (False, True):
        for form in ((1, 0) if not deformed else (0,)):
            with simplex_form(nk, form):
                run_case(nk, shape, P, 4, deformed, ("bwdtrans", "iprod", "mass", "laplacian", "helmholtz"), lam=0.3,
                         take=take, seed=wl.SEED0 + 15)


@pytest.mark.parametrize("P", range(1, 9))
def test_affine_tet_reference_matrix_form(nk, P):
    """the reference-matrix (DMMA) kernels of nk_dense.cuh against the oracle: mass, Laplacian, Helmholtz with
    lambda != 1 on several tiles of 8 elements plus a ragged tail, and against the sum-factorised form."""
    if not _dense_available(nk, o.TET, P):
        pytest.skip("no reference-matrix kernel instantiated for tet P%d" % P)
    el = K.element(o.TET, P)
    full = K.mesh(o.TET, 3)[0].shape[0]        # 162 tets: several tiles of 8 (and of 32 / 64 at P >= 6) plus a tail
    for ne in (full - 3, 8, 1):
        A, J = K.geometry(o.TET, P, 3, False, take=torch.arange(ne))
        basis = nk.Basis(o.TET, P)
        geom = nk.Geom(basis, A.cuda(), J.cuda(), False)
        for op in ("mass", "laplacian", "helmholtz"):
            x = K.make_input(op, wl.SEED0 + 16, ne, el)
            ref = K.oracle_op(op, el, A, J, 3.25, x)
            with simplex_form(nk, 2):
                got = K.gpu_op(nk, op, basis, geom, 3.25, x)
            with simplex_form(nk, 1):
                sf = K.gpu_op(nk, op, basis, geom, 3.25, x)
            assert K.normwise_err(got, ref) <= TOL, (P, ne, op)
            assert K.normwise_err(sf, ref) <= TOL, (P, ne, op)
            assert K.normwise_err(got, sf) <= 1e-13, (P, ne, op)


@pytest.mark.parametrize("shape,P", [(o.PRISM, 1), (o.PRISM, 2), (o.PRISM, 3), (o.PRISM, 4), (o.HEX, 2), (o.HEX, 3)])
def test_runtime_specialised_reference_matrix_kernel(nk, shape, P):
    """form 2 on prisms and on hexes of order >= 2.  Prisms P1..P3 have prebuilt reference-matrix kernels; prism P4 (Nm =
    75), hex P2 (27) and hex P3 (64) have none: the kernel is specialised at run time by NVRTC (csrc/nk_jit.cu), resident
    (27) or streamed (64, 75).  Against the oracle and against the sum-factorised / Kronecker form, several tiles plus a
    tail."""
    el = K.element(shape, P)
    full = K.mesh(shape, 3)[0].shape[0]
    A, J = K.geometry(shape, P, 3, False, take=torch.arange(full - 3))
    ne = J.shape[0]
    basis = nk.Basis(shape, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), False)
    k0, _ = nk.jit_stats()
    for op in ("mass", "laplacian", "helmholtz"):
        x = K.make_input(op, wl.SEED0 + 17, ne, el)
        ref = K.oracle_op(op, el, A, J, 0.75, x)
        with simplex_form(nk, 2):
            got = K.gpu_op(nk, op, basis, geom, 0.75, x)
        with simplex_form(nk, 1):
            other = K.gpu_op(nk, op, basis, geom, 0.75, x)
        assert K.normwise_err(got, ref) <= TOL, (shape, P, op)
        assert K.normwise_err(other, ref) <= TOL, (shape, P, op)
        assert K.normwise_err(got, other) <= 1e-13, (shape, P, op)
    k1, ms = nk.jit_stats()
    if (shape, P) in ((o.PRISM, 4), (o.HEX, 2), (o.HEX, 3)):      # no prebuilt kernel for 75, 27, 64 modes
        assert k1 - k0 == 3 and ms > 0.0            # three operators specialised, once per process and mode count
    else:                                          # prisms P1..P3 have prebuilt kernels (and take them by default)
        assert k1 == k0


def _dense_available(nk, shape, P):
    basis = nk.Basis(shape, P)
    A, J = K.geometry(shape, P, 2, False, take=torch.arange(1))
    geom = nk.Geom(basis, A.cuda(), J.cuda(), False)
    x = torch.zeros((1, basis.num_modes), dtype=torch.float64, device="cuda")
    with simplex_form(nk, 2):
        try:
            nk.mass_apply(basis, geom, x, torch.empty_like(x))
        except nk.NkError as e:
            assert e.code == 2          # NK_ERR_UNSUPPORTED is the only acceptable refusal
            return False
    return True


def test_config5_blocks_small(nk):
    """prisms + tets, deformed, P=5, lambda=10, ONE nk_helmholtz_apply_blocks call."""
    n, P, lam = 4, 5, 10.0
    blocks, refs = [], []
    for shape, zlo, zhi in ((o.TET, 0, 1), (o.PRISM, 1, 4)):
        el = K.element(shape, P)
        A, J = K.geometry(shape, P, n, True, zlo=zlo, zhi=zhi)
        basis = nk.Basis(shape, P)
        geom = nk.Geom(basis, A.cuda(), J.cuda(), True)
        x = wl.coefficients(wl.SEED0 + 5 + shape, J.shape[0], el.Nm)
        y = torch.full_like(x, float("nan")).cuda()
        blocks.append((basis, geom, x.cuda(), y))
        refs.append(o.helmholtz(el, A.numpy(), J.numpy(), lam, x.numpy()))
    nk.helmholtz_apply_blocks(blocks, lam)
    torch.cuda.synchronize()
    for (b, g, x, y), ref in zip(blocks, refs):
        assert K.normwise_err(y.cpu().numpy(), ref) <= TOL


def test_edge_cases(nk):
    basis = nk.Basis(o.HEX, 2)
    el = K.element(o.HEX, 2)
    # nelem = 0: valid, no-op
    A0 = torch.zeros((0, 1, 3, 3), dtype=torch.float64, device="cuda")
    J0 = torch.zeros((0, 1), dtype=torch.float64, device="cuda")
    g0 = nk.Geom(basis, A0, J0, False)
    x0 = torch.zeros((0, el.Nm), dtype=torch.float64, device="cuda")
    nk.helmholtz_apply(basis, g0, 1.0, x0, torch.zeros_like(x0) + 1)
    # nelem = 1 and host-side geometry upload
    A, J = K.geometry(o.HEX, 2, 2, True, take=torch.tensor([5]))
    g1 = nk.Geom(basis, A, J, True)            # host tensors
    x = wl.coefficients(3, 1, el.Nm)
    y = torch.empty_like(x).cuda()
    nk.helmholtz_apply(basis, g1, 2.0, x.cuda(), y)
    ref = o.helmholtz(el, A.numpy(), J.numpy(), 2.0, x.numpy())
    assert K.normwise_err(y.cpu().numpy(), ref) <= TOL
    # NULL components of physderiv / iprod_deriv
    u = wl.point_values(4, 1, el.Nq)
    d1 = torch.empty_like(u).cuda()
    nk.physderiv(basis, g1, u.cuda(), None, d1, None)
    ref = o.physderiv(el, A.numpy(), u.numpy())
    assert K.normwise_err(d1.cpu().numpy(), ref[1]) <= TOL
    c = torch.empty((1, el.Nm), dtype=torch.float64, device="cuda")
    nk.iprod_deriv(basis, g1, None, u.cuda(), None, c)
    gg = np.stack([np.zeros_like(u.numpy()), u.numpy(), np.zeros_like(u.numpy())])
    ref = o.iprod_deriv(el, A.numpy(), J.numpy(), gg)
    assert K.normwise_err(c.cpu().numpy(), ref) <= TOL
    # errors: aliasing, geometry of another basis
    with pytest.raises(nk.NkError) as ei:
        xx = x.cuda()
        nk.helmholtz_apply(basis, g1, 1.0, xx, xx)
    assert ei.value.code == 1
    other = nk.Basis(o.HEX, 3)
    with pytest.raises(nk.NkError) as ei:
        nk.helmholtz_apply(other, g1, 1.0, x.cuda(), y)
    assert ei.value.code == 3


def test_operator_identities_on_gpu(nk):
    """mass = iprod o bwdtrans; laplacian = iprod_deriv o physderiv o bwdtrans;
    helmholtz = laplacian + lambda mass (SURVEY 8(c) 'Operator identities')."""
    for shape in (o.HEX, o.TET, o.PRISM):
        P, lam = 3, 3.5
        el = K.element(shape, P)
        A, J = K.geometry(shape, P, 2, True, zhi=1)
        ne = J.shape[0]
        basis = nk.Basis(shape, P)
        geom = nk.Geom(basis, A.cuda(), J.cuda(), True)
        x = wl.coefficients(11, ne, el.Nm).numpy()
        u = K.gpu_op(nk, "bwdtrans", basis, geom, lam, x)
        m1 = K.gpu_op(nk, "iprod", basis, geom, lam, u)
        m2 = K.gpu_op(nk, "mass", basis, geom, lam, x)
        assert K.normwise_err(m1, m2) <= 1e-13
        gr = K.gpu_op(nk, "physderiv", basis, geom, lam, u)
        l1 = K.gpu_op(nk, "iprod_deriv", basis, geom, lam, gr)
        l2 = K.gpu_op(nk, "laplacian", basis, geom, lam, x)
        assert K.normwise_err(l1, l2) <= 1e-13
        h = K.gpu_op(nk, "helmholtz", basis, geom, lam, x)
        assert K.normwise_err(h, l2 + lam * m2) <= 1e-13


def test_helmholtz_host_entry_affine_tet(nk):
    """host entry on the reference-matrix kernel: the chunks of the pipeline are tiles of 8 elements."""
    P = 4
    el = K.element(o.TET, P)
    full = K.mesh(o.TET, 3)[0].shape[0]
    A, J = K.geometry(o.TET, P, 3, False, take=torch.arange(full - 3))
    basis = nk.Basis(o.TET, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), False)
    x = wl.coefficients(22, J.shape[0], el.Nm).pin_memory()
    ref = o.helmholtz(el, A.numpy(), J.numpy(), 1.5, x.numpy())
    for form in (0, 1):
        y = torch.full_like(x, float("nan")).pin_memory()
        with simplex_form(nk, form):
            nk.helmholtz_apply_host(basis, geom, 1.5, x, y)
        assert K.normwise_err(y.numpy(), ref) <= TOL


@pytest.mark.parametrize("deformed", [True, False])
def test_helmholtz_host_entry(nk, deformed):
    """deformed: quadrature-grid kernel; affine: coefficient-space kernel, whose block size differs from the
    interleave width of the geometry stream (the chunks of the host pipeline follow the kernel's groups)."""
    P = 4
    el = K.element(o.HEX, P)
    full = K.mesh(o.HEX, 3)[0].shape[0]
    A, J = K.geometry(o.HEX, P, 3, deformed, take=torch.arange(full - 2))
    basis = nk.Basis(o.HEX, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    x = wl.coefficients(21, J.shape[0], el.Nm).pin_memory()
    y = torch.empty_like(x).pin_memory()
    n0 = nk.launch_count()
    nk.helmholtz_apply_host(basis, geom, 1.0, x, y)
    assert 1 <= nk.launch_count() - n0 <= 16     # chunked copy / compute / copy pipeline
    ref = o.helmholtz(el, A.numpy(), J.numpy(), 1.0, x.numpy())
    assert K.normwise_err(y.numpy(), ref) <= TOL


@pytest.mark.parametrize("shape,P", [(o.TET, 5), (o.TET, 6), (o.PRISM, 6), (o.TET, 8), (o.PRISM, 8)])
def test_high_order_deformed_simplices_fields_and_repeatability(nk, shape, P):
    """the deformed simplex kernels whose psi^b tables sit in shared memory (tets from P5, with S2 folded into S3; prisms at
    P6, P7) and the wide blocks at P8: single-field and multi-field calls against the oracle, bit-identical to each other
    and over repeated launches (a race on the shared table copy or on T1 in X would show as run-to-run noise)."""
    lam, nf = 1.5, 2
    el = K.element(shape, P)
    A, J = K.geometry(shape, P, 2, True, zhi=1)
    ne = J.shape[0]
    basis = nk.Basis(shape, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), True)
    xs = [wl.coefficients(400 + f, ne, el.Nm) for f in range(nf)]
    dx = [x.cuda() for x in xs]
    dy = [torch.full_like(x, float("nan")) for x in dx]
    nk.helmholtz_apply_fields(basis, geom, lam, dx, dy)
    torch.cuda.synchronize()
    for f in range(nf):
        ref = o.helmholtz(el, A.numpy(), J.numpy(), lam, xs[f].numpy())
        assert K.normwise_err(dy[f].cpu().numpy(), ref) <= TOL
        for _ in range(5):
            y1 = torch.full_like(dx[f], float("nan"))
            nk.helmholtz_apply(basis, geom, lam, dx[f], y1)
            assert torch.equal(y1, dy[f])
    for op in ("mass", "laplacian", "bwdtrans"):          # the operators that share the forward stages
        x = K.make_input(op, 500, ne, el)
        assert K.op_err(op, K.gpu_op(nk, op, basis, geom, lam, x), K.oracle_op(op, el, A, J, lam, x)) <= TOL, op


@pytest.mark.parametrize("shape,deformed", [(o.HEX, True), (o.HEX, False), (o.TET, False), (o.PRISM, True)])
def test_helmholtz_fields(nk, shape, deformed):
    """nk_helmholtz_apply_fields (multi-field block): each field equals the oracle's Helmholtz of that
    field, and is bit-identical to the single-field call."""
    P, lam, nf = 3, 2.5, 3
    el = K.element(shape, P)
    full = K.mesh(shape, 3)[0].shape[0]
    A, J = K.geometry(shape, P, 3, deformed, take=torch.arange(full - 3))
    ne = J.shape[0]
    basis = nk.Basis(shape, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    xs = [wl.coefficients(100 + f, ne, el.Nm) for f in range(nf)]
    dx = [x.cuda() for x in xs]
    dy = [torch.full_like(x, float("nan")) for x in dx]
    n0 = nk.launch_count()
    nk.helmholtz_apply_fields(basis, geom, lam, dx, dy)
    assert nk.launch_count() == n0 + 1          # ONE launch for all fields
    torch.cuda.synchronize()
    for f in range(nf):
        ref = o.helmholtz(el, A.numpy(), J.numpy(), lam, xs[f].numpy())
        assert K.normwise_err(dy[f].cpu().numpy(), ref) <= TOL
        y1 = torch.empty_like(dx[f])
        nk.helmholtz_apply(basis, geom, lam, dx[f], y1)
        assert torch.equal(y1, dy[f])
    with pytest.raises(nk.NkError):
        nk.helmholtz_apply_fields(basis, geom, lam, dx, [dy[0], dy[0], dy[2]])
    with pytest.raises(nk.NkError):
        nk.helmholtz_apply_fields(basis, geom, lam, dx, [dy[0], dx[1], dy[2]])


@pytest.mark.parametrize("shape,P,deformed", [(o.HEX, 4, True), (o.TET, 4, False), (o.PRISM, 5, True), (o.HEX, 7, False)])
def test_repeatable_bitwise(nk, shape, P, deformed):
    """The shared-memory reuse plan has no race: 20 launches on the same input give bit-identical output
    (compute-sanitizer is closed on this pool; a race between stages would show up as run-to-run noise)."""
    full = K.mesh(shape, 3)[0].shape[0]
    A, J = K.geometry(shape, P, 3, deformed, take=torch.arange(full - 1))
    basis = nk.Basis(shape, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    x = wl.coefficients(77, J.shape[0], basis.num_modes).cuda()
    y0 = torch.empty_like(x)
    nk.helmholtz_apply(basis, geom, 1.5, x, y0)
    for _ in range(20):
        y = torch.full_like(x, float("nan"))
        nk.helmholtz_apply(basis, geom, 1.5, x, y)
        assert torch.equal(y, y0)


def test_geometry_streams(nk):
    """nk_geom_upload_streams: a metric-only geometry serves Helmholtz (bit-identical to the full upload) and
    refuses nk_physderiv; a factors-only geometry the other way round."""
    P = 3
    el = K.element(o.TET, P)
    A, J = K.geometry(o.TET, P, 2, True, zhi=1)
    basis = nk.Basis(o.TET, P)
    full = nk.Geom(basis, A.cuda(), J.cuda(), True)
    gm = nk.Geom(basis, A.cuda(), J.cuda(), True, streams=nk.Geom.METRIC)
    gf = nk.Geom(basis, A.cuda(), J.cuda(), True, streams=nk.Geom.FACTORS)
    x = wl.coefficients(5, J.shape[0], el.Nm).cuda()
    y0, y1 = torch.empty_like(x), torch.empty_like(x)
    nk.helmholtz_apply(basis, full, 2.0, x, y0)
    nk.helmholtz_apply(basis, gm, 2.0, x, y1)
    assert torch.equal(y0, y1)
    u = wl.point_values(6, J.shape[0], el.Nq).cuda()
    d = [torch.empty_like(u) for _ in range(3)]
    nk.physderiv(basis, gf, u, d[0], d[1], d[2])
    ref = o.physderiv(el, A.numpy(), u.cpu().numpy())
    assert K.op_err("physderiv", torch.stack(d).cpu().numpy(), ref) <= TOL
    with pytest.raises(nk.NkError) as ei:
        nk.physderiv(basis, gm, u, d[0], d[1], d[2])
    assert ei.value.code == 1
    with pytest.raises(nk.NkError) as ei:
        nk.helmholtz_apply(basis, gf, 2.0, x, y1)
    assert ei.value.code == 1
