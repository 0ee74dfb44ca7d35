"""Pins for the oracle's 3-D tables and operators: closed forms, textbook
element matrices, invariants (north_star / SURVEY 8(c)), brute force."""
import itertools

import numpy as np
import pytest

import golden_io as G
from oracle import nk_oracle as o

SHAPES = (o.HEX, o.TET, o.PRISM)
RNG = np.random.default_rng(7)


def _golden_1d():
    ref = {"M1": np.zeros((5, 5)), "K1": np.zeros((5, 5))}
    for name, r, c, v in G.records("modified_basis_P4.txt"):
        ref[name][int(r), int(c)] = ref[name][int(c), int(r)] = G.number(v)
    return ref["M1"], ref["K1"]


def _random_affine(shape_seed):
    r = np.random.default_rng(shape_seed)
    E = np.eye(3) + 0.15 * r.standard_normal((3, 3))
    if np.linalg.det(E) < 0:
        E[:, 0] *= -1
    v0 = r.standard_normal(3)
    Jm = 0.5 * E                      # dx/dxi
    return v0, Jm, np.linalg.inv(Jm), abs(np.linalg.det(Jm))


def test_standard_element_volumes_and_points():
    for shape, vol in ((o.HEX, 8.0), (o.TET, 4.0 / 3.0), (o.PRISM, 4.0)):
        for P in (1, 4, 7):
            el = o.Element(shape, P, P + 2)
            assert el.wq.sum() == pytest.approx(vol, rel=1e-13)
            xi = el.xi
            assert xi.min() >= -1 - 1e-15
            if shape == o.TET:
                assert (xi.sum(axis=1)).max() <= -1 + 1e-13      # Eq. 11
            if shape == o.PRISM:
                assert (xi[:, 0] + xi[:, 2]).max() <= 1e-13
            # point order n = i + Q(j + Qk): eta_1 fastest
            Q = P + 2
            assert np.all(el.eta[:Q, 0] == el.z[0]) and np.all(el.eta[:Q, 1] == el.z[1][0])
            assert np.all(el.eta[::Q * Q, 2] == el.z[2])
    # first moments of the standard tet / prism (centroids) pin the xi map + weights
    el = o.Element(o.TET, 3, 5)
    np.testing.assert_allclose(el.wq @ el.xi / el.wq.sum(), [-0.5, -0.5, -0.5], atol=1e-14)
    el = o.Element(o.PRISM, 3, 5)
    np.testing.assert_allclose(el.wq @ el.xi / el.wq.sum(), [-1 / 3, 0.0, -1 / 3], atol=1e-14)


def test_hex_affine_kronecker_closed_form():
    M1, K1 = _golden_1d()
    el = o.Element(o.HEX, 4, 6)
    hx, hy, hz = 0.25, 0.4, 0.7
    A = np.diag([2 / hx, 2 / hy, 2 / hz])[None]
    J = np.array([hx * hy * hz / 8])
    M, L = o.element_matrices(el, A, J)
    k3 = lambda a, b, c: np.kron(np.kron(a, b), c)
    Mref = J[0] * k3(M1, M1, M1)
    Lref = J[0] * ((2 / hx) ** 2 * k3(K1, M1, M1) + (2 / hy) ** 2 * k3(M1, K1, M1) + (2 / hz) ** 2 * k3(M1, M1, K1))
    np.testing.assert_allclose(M, Mref, atol=1e-16 + 1e-14 * np.abs(Mref).max())
    np.testing.assert_allclose(L, Lref, atol=1e-14 * np.abs(Lref).max())
    # and through the batched operator entry points
    uh = RNG.uniform(-1, 1, (3, el.Nm))
    Ab, Jb = np.broadcast_to(A, (3, 1, 3, 3)), np.broadcast_to(J, (3, 1))
    np.testing.assert_allclose(o.mass(el, Jb, uh), uh @ Mref.T, atol=1e-15)
    np.testing.assert_allclose(o.laplacian(el, Ab, Jb, uh), uh @ Lref.T, atol=1e-12)
    np.testing.assert_allclose(o.helmholtz(el, Ab, Jb, 10.0, uh), uh @ (Lref + 10.0 * Mref).T, atol=1e-12)


def _p1_reference(verts):
    """Textbook linear simplex: gradients of barycentrics, volume."""
    T = np.hstack([np.ones((4, 1)), verts])
    C = np.linalg.inv(T)                 # column a = coefficients of lambda_a
    grads = C[1:, :].T                   # [a][3]
    vol = abs(np.linalg.det(T)) / 6.0
    return grads, vol


def test_tet_p1_textbook_matrices():
    v0, Jm, A, J = _random_affine(11)
    verts = np.stack([v0, v0 + 2 * Jm[:, 0], v0 + 2 * Jm[:, 1], v0 + 2 * Jm[:, 2]])
    grads, vol = _p1_reference(verts)
    el = o.Element(o.TET, 1, 3)
    M, L = o.element_matrices(el, A[None], np.array([J]))
    order = [0, 3, 2, 1]                 # modes (000),(001),(010),(100) -> vertices v0, v3, v2, v1
    Mref = vol / 20.0 * (np.ones((4, 4)) + np.eye(4))
    Lref = vol * grads[order] @ grads[order].T
    assert vol == pytest.approx(4.0 / 3.0 * J, rel=1e-14)
    np.testing.assert_allclose(M, Mref, atol=1e-15)
    np.testing.assert_allclose(L, Lref, atol=1e-13)
    # reference tet itself: M00 = 2/15, M01 = 1/15
    M, _ = o.element_matrices(el, np.eye(3)[None], np.ones(1))
    assert M[0, 0] == pytest.approx(2 / 15, rel=1e-14) and M[0, 1] == pytest.approx(1 / 15, rel=1e-14)


def test_prism_p1_textbook_matrices():
    # right prism: triangle in the (x,z) plane (sheared/scaled), extruded along y
    Jm = np.array([[0.7, 0.0, 0.2], [0.0, 0.45, 0.0], [0.1, 0.0, 0.6]])     # dx/dxi
    A, J = np.linalg.inv(Jm), abs(np.linalg.det(Jm))
    el = o.Element(o.PRISM, 1, 3)
    M, L = o.element_matrices(el, A[None], np.array([J]))
    # triangle vertices (xi1,xi3) = (-1,-1),(1,-1),(-1,1) -> physical (x,z)
    tri = np.array([[0, 0], 2 * Jm[[0, 2], 0], 2 * Jm[[0, 2], 2]])
    T = np.hstack([np.ones((3, 1)), tri])
    C = np.linalg.inv(T)
    g = C[1:, :].T
    area = abs(np.linalg.det(T)) / 2
    Mt = area / 12 * (np.ones((3, 3)) + np.eye(3))
    Kt = area * g @ g.T
    ly = 2 * Jm[1, 1]
    Ml = ly / 6 * np.array([[2, 1], [1, 2.0]])
    Kl = 1 / ly * np.array([[1, -1], [-1, 1.0]])
    # modes (p,q,r): (000),(001),(010),(011),(100),(110); triangle vertex t(p,r): (0,0)->0,(1,0)->1,(0,1)->2
    modes = o.mode_list(o.PRISM, 1)
    tv = {(0, 0): 0, (1, 0): 1, (0, 1): 2}
    Mref = np.array([[Mt[tv[(a[0], a[2])], tv[(b[0], b[2])]] * Ml[a[1], b[1]] for b in modes] for a in modes])
    Lref = np.array([[Kt[tv[(a[0], a[2])], tv[(b[0], b[2])]] * Ml[a[1], b[1]]
                      + Mt[tv[(a[0], a[2])], tv[(b[0], b[2])]] * Kl[a[1], b[1]] for b in modes] for a in modes])
    np.testing.assert_allclose(M, Mref, atol=1e-15)
    np.testing.assert_allclose(L, Lref, atol=1e-13)


@pytest.mark.parametrize("shape", [o.TET, o.PRISM])
@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_collapsed_basis_is_polynomial_and_complete(shape, P):
    """A8: with the top-vertex/edge corrections every phi is a polynomial in xi,
    the set spans P_P (tet) / P_P(xi1,xi3) x P_P(xi2) (prism) and vertex modes sum to 1."""
    el = o.Element(shape, P, P + 2)
    x, y, z = el.xi.T
    if shape == o.TET:
        mono = [x ** a * y ** b * z ** c for a in range(P + 1) for b in range(P + 1 - a) for c in range(P + 1 - a - b)]
    else:
        mono = [x ** a * z ** c * y ** b for a in range(P + 1) for c in range(P + 1 - a) for b in range(P + 1)]
    V = np.stack(mono, axis=1)
    assert V.shape[1] == el.Nm
    coef, res, rank, _ = np.linalg.lstsq(V, el.Phi, rcond=None)
    assert rank == el.Nm
    assert np.abs(V @ coef - el.Phi).max() < 1e-11           # in the polynomial space
    assert np.linalg.matrix_rank(el.Phi) == el.Nm            # linearly independent
    nm = P + 1
    if shape == o.TET:
        vm = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)]
    else:
        vm = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (1, 1, 0), (0, 0, 1), (0, 1, 1)]
    one = np.zeros(el.Nm)
    for m in vm:
        one[o.mode_index(shape, P, *m)] = 1.0
    np.testing.assert_allclose(el.Phi @ one, 1.0, atol=1e-14)
    # vertex modes are the hat functions: (1 + xi_d)/2 for the three "far" vertices
    np.testing.assert_allclose(el.Phi[:, o.mode_index(shape, P, 1, 0, 0)],
                               (1 + x) / 2 if shape == o.TET else (1 + x) / 2 * (1 - y) / 2, atol=1e-14)
    np.testing.assert_allclose(el.Phi[:, o.mode_index(shape, P, 0, 0, 1)],
                               (1 + z) / 2 if shape == o.TET else (1 + z) / 2 * (1 - y) / 2, atol=1e-14)
    if shape == o.TET:
        np.testing.assert_allclose(el.Phi[:, o.mode_index(shape, P, 0, 1, 0)], (1 + y) / 2, atol=1e-14)


@pytest.mark.parametrize("shape", SHAPES)
def test_invariants_affine(shape):
    P = 3
    el = o.Element(shape, P, P + 2)
    v0, Jm, A, J = _random_affine(5 + shape)
    M, L = o.element_matrices(el, A[None], np.array([J]))
    assert np.abs(M - M.T).max() < 1e-16 + 1e-15 * np.abs(M).max()
    assert np.linalg.eigvalsh(M).min() > 0
    assert np.abs(L - L.T).max() < 1e-14 * np.abs(L).max()
    assert np.linalg.eigvalsh(L).min() > -1e-12 * np.abs(L).max()
    one = np.linalg.lstsq(el.Phi, np.ones(el.Nq), rcond=None)[0]
    assert one @ M @ one == pytest.approx(el.wq.sum() * J, rel=1e-13)      # integrating 1 gives the volume
    assert np.abs(L @ one).max() < 1e-13 * np.abs(L).max()                  # Laplacian annihilates constants
    # quadrature sufficiency: Q=P+2 already gives the exact Galerkin matrices
    el2 = o.Element(shape, P, P + 4)
    M2, L2 = o.element_matrices(el2, A[None], np.array([J]))
    np.testing.assert_allclose(M, M2, atol=1e-14 * np.abs(M).max())
    np.testing.assert_allclose(L, L2, atol=1e-13 * np.abs(L).max())


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("P", [2, 5])
def test_physderiv_exact_for_polynomials(shape, P):
    """North-star invariant (iii): exact for total degree <= P on affine elements."""
    el = o.Element(shape, P, P + 2)
    ne = 3
    A = np.zeros((ne, 1, 3, 3))
    u = np.zeros((ne, el.Nq))
    grad = np.zeros((3, ne, el.Nq))
    r = np.random.default_rng(3)
    for e in range(ne):
        v0, Jm, Ai, J = _random_affine(100 + e)
        A[e, 0] = Ai
        X = v0[None] + (el.xi + 1.0) @ Jm.T
        for (a, b, c) in [(a, b, c) for a in range(P + 1) for b in range(P + 1 - a) for c in range(P + 1 - a - b)]:
            co = r.standard_normal()
            x, y, z = X.T
            u[e] += co * x ** a * y ** b * z ** c
            if a: grad[0, e] += co * a * x ** (a - 1) * y ** b * z ** c
            if b: grad[1, e] += co * b * x ** a * y ** (b - 1) * z ** c
            if c: grad[2, e] += co * c * x ** a * y ** b * z ** (c - 1)
    d = o.physderiv(el, A, u)
    assert np.abs(d - grad).max() < 2e-10 * max(1.0, np.abs(grad).max())


def _quadratic_map(el, seed):
    """x(xi) = Jm (xi+1) + eps * q(xi), q quadratic: a smooth deformed element with
    analytic inverse Jacobian at the points."""
    r = np.random.default_rng(seed)
    _, Jm, _, _ = _random_affine(seed)
    C = 0.02 * r.standard_normal((3, 3, 3))
    xi = el.xi
    X = (xi + 1.0) @ Jm.T + np.einsum("cab,na,nb->nc", C, xi, xi)
    dX = Jm[None] + np.einsum("cab,nb->nca", C, xi) + np.einsum("cab,na->ncb", C, xi)   # dX_c/dxi_a
    A = np.linalg.inv(dX)                    # [n][j][i] = dxi_j/dx_i
    J = np.linalg.det(dX)
    assert J.min() > 0
    return X, A, J


@pytest.mark.parametrize("shape", SHAPES)
def test_deformed_geometry_conventions(shape):
    """On a deformed element grad_x of the coordinate function x_c is e_c exactly
    (pins the [j][i] layout of dxi_dx and the chain factors A17), and
    (L uhat)_m = sum_n W_n (grad_x phi_m)_c for uhat representing x_c."""
    P = 3
    el = o.Element(shape, P, P + 2)
    X, A, J = _quadratic_map(el, 42 + shape)
    Ab, Jb = A[None], J[None]
    for c in range(3):
        d = o.physderiv(el, Ab, X[None, :, c])
        for i in range(3):
            np.testing.assert_allclose(d[i, 0], 1.0 if i == c else 0.0, atol=2e-11)
    if shape == o.HEX:      # x_c(xi) has degree 2 per variable -> in the hex span for P>=2
        for c in range(3):
            uh = np.linalg.lstsq(el.Phi, X[:, c], rcond=None)[0]
            np.testing.assert_allclose(el.Phi @ uh, X[:, c], atol=1e-12)
            Lu = o.laplacian(el, Ab, Jb, uh[None])[0]
            W = el.wq * J
            assert uh @ Lu == pytest.approx(W.sum(), rel=1e-11)          # energy of x_c = volume
            ref = np.array([W @ o.physderiv(el, Ab, el.Phi[None, :, m])[c, 0] for m in range(el.Nm)])
            np.testing.assert_allclose(Lu, ref, atol=1e-11)
    one = np.linalg.lstsq(el.Phi, np.ones(el.Nq), rcond=None)[0]
    assert one @ o.mass(el, Jb, one[None])[0] == pytest.approx((el.wq * J).sum(), rel=1e-13)
    assert np.abs(o.laplacian(el, Ab, Jb, one[None])).max() < 1e-12


@pytest.mark.parametrize("shape", SHAPES)
def test_operator_identities(shape):
    P = 4
    el = o.Element(shape, P, P + 2)
    ne = 4
    geo = [_quadratic_map(el, 60 + e) for e in range(ne)]
    A = np.stack([g[1] for g in geo])
    J = np.stack([g[2] for g in geo])
    uh = RNG.uniform(-1, 1, (ne, el.Nm))
    v = RNG.uniform(-1, 1, (ne, el.Nq))
    u = o.bwdtrans(el, uh)
    # Laplacian via analytic basis gradients == iprod_deriv(physderiv(bwd)) via collocation D
    lap1 = o.laplacian(el, A, J, uh)
    lap2 = o.iprod_deriv(el, A, J, o.physderiv(el, A, u))
    np.testing.assert_allclose(lap1, lap2, atol=1e-11 * np.abs(lap1).max())
    np.testing.assert_allclose(o.helmholtz(el, A, J, 10.0, uh), lap1 + 10.0 * o.iprod(el, J, u), atol=1e-13)
    # adjointness <v, B uh>_W = <iprod(v), uh>
    W = el.wq[None] * J
    np.testing.assert_allclose((W * v * u).sum(1), (o.iprod(el, J, v) * uh).sum(1), rtol=1e-12)
    # iprod_deriv is the adjoint of physderiv o bwd
    g = RNG.uniform(-1, 1, (3, ne, el.Nq))
    lhs = (W[None] * g * o.physderiv(el, A, u)).sum(axis=(0, 2))
    rhs = (o.iprod_deriv(el, A, J, g) * uh).sum(1)
    np.testing.assert_allclose(lhs, rhs, rtol=1e-10)
    # dense matrices agree with the operator entry points (helm = L + lambda*M, Eq. 6 / A6)
    M, L = o.element_matrices(el, A[1], J[1])
    np.testing.assert_allclose(o.helmholtz(el, A[1:2], J[1:2], 10.0, uh[1:2])[0], (L + 10.0 * M) @ uh[1],
                               atol=1e-12 * np.abs(L).max())


@pytest.mark.parametrize("shape", SHAPES)
def test_bwd_then_mass_solve_recovers_coefficients(shape):
    P = 3
    el = o.Element(shape, P, P + 2)
    _, _, A, J = _random_affine(77)
    M, _ = o.element_matrices(el, A[None], np.array([J]))
    uh = RNG.uniform(-1, 1, (2, el.Nm))
    rhs = o.iprod(el, np.full((2, 1), J), o.bwdtrans(el, uh))
    np.testing.assert_allclose(np.linalg.solve(M, rhs.T).T, uh, atol=1e-9)


# ---------------------------------------------------------------------------
# Brute force: Eq. 16 / Eq. 17 written as the paper's nested sums in pure Python
# (plus the A8 correction recipe in sum-factorised form), tiny cases.
# ---------------------------------------------------------------------------
def _sumfact_bwd(shape, P, Q, z, uh):
    nm = P + 1
    out = np.zeros((Q, Q, Q))                      # [i][j][k]
    idx = lambda p, q, r: o.mode_index(shape, P, p, q, r)
    for i, j, k in itertools.product(range(Q), repeat=3):
        acc = 0.0
        for p in range(nm):
            qmax = nm - p if shape == o.TET else nm
            accq = 0.0
            for q in range(qmax):
                rmax = nm if shape == o.HEX else (nm - p - q if shape == o.TET else nm - p)
                accr = 0.0
                for r in range(rmax):
                    if shape == o.HEX:
                        c = o.psi_a(r, z[2][k])
                    elif shape == o.TET:
                        c = o.psi_b(p + q, r, z[2][k])
                    else:
                        c = o.psi_b(p, r, z[2][k])
                    accr += uh[idx(p, q, r)] * c
                # A8 corrections after the r-sum
                if shape == o.TET and (p, q) in ((0, 1), (1, 0)) and P >= 1:
                    accr += uh[idx(0, 0, 1)] * o.psi_b(0, 1, z[2][k])
                if shape == o.PRISM and p == 1:
                    accr += uh[idx(0, q, 1)] * o.psi_b(0, 1, z[2][k])
                b = o.psi_b(p, q, z[1][j]) if shape == o.TET else o.psi_a(q, z[1][j])
                accq += b * accr
                if shape == o.TET and p == 1 and q == 0:
                    # A8: add the (0,1) column times psi^b_01(eta2_j) to row p=1
                    acc01 = sum(uh[idx(0, 1, r)] * o.psi_b(1, r, z[2][k]) for r in range(nm - 1))
                    acc01 += uh[idx(0, 0, 1)] * o.psi_b(0, 1, z[2][k])
                    accq += o.psi_b(0, 1, z[1][j]) * acc01
            acc += o.psi_a(p, z[0][i]) * accq
        out[i, j, k] = acc
    return out.transpose(2, 1, 0).reshape(-1)      # n = i + Q(j + Qk)


@pytest.mark.parametrize("shape,P", [(o.HEX, 2), (o.TET, 1), (o.TET, 3), (o.PRISM, 1), (o.PRISM, 3)])
def test_brute_force_sum_factorised_bwd(shape, P):
    Q = P + 2
    el = o.Element(shape, P, Q)
    uh = np.random.default_rng(shape * 10 + P).uniform(-1, 1, el.Nm)
    ref = _sumfact_bwd(shape, P, Q, el.z, uh)
    np.testing.assert_allclose(o.bwdtrans(el, uh[None])[0], ref, atol=1e-14)


class _ExtendedElement:
    """the oracle's element tables cast to np.longdouble (80-bit extended on x86): the SAME tables, so that running the
    oracle's operator functions on it repeats their dense sums with 11 more bits in every product and accumulation"""

    def __init__(self, el):
        self.__dict__.update(el.__dict__)
        for k, v in el.__dict__.items():
            if isinstance(v, np.ndarray) and v.dtype == np.float64:
                setattr(self, k, v.astype(np.longdouble))
            elif isinstance(v, (list, tuple)) and v and all(isinstance(a, np.ndarray) for a in v):
                setattr(self, k, [a.astype(np.longdouble) if a.dtype == np.float64 else a for a in v])
        self._el = el

    def chain(self, dEta):
        return type(self._el).chain(self, dEta)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_oracle_rounding_against_extended_precision(cfg):
    """the oracle's own fp64 rounding.  On a sample of each configuration (<= 256 elements) the
    oracle's Helmholtz in fp64 agrees with the same sums carried in extended precision to <= 1e-13 normwise, i.e.
    the 1e-12 parity gate of the GPU tests is not consumed by the oracle's accumulation order."""
    if np.finfo(np.longdouble).eps >= np.finfo(np.float64).eps:
        pytest.skip("np.longdouble is not wider than float64 on this platform")
    from workloads import configs as cfgs
    from workloads import synthetic as wl
    title, op, blocks = cfgs.config_blocks(cfg, device="cpu", scale=0.2)
    for b in blocks:
        el = o.Element(b["shape"], b["P"], b["P"] + 2)
        ne = min(b["v0"].shape[0], 256 if el.Nq <= 216 else 48)
        idx = np.linspace(0, b["v0"].shape[0] - 1, ne).astype(np.int64)
        v0, E = b["v0"][idx], b["E"][idx]
        A, J = (wl.sinusoidal_factors(v0, E, el.xi) if b["deformed"] else wl.affine_factors(v0, E))
        x = wl.coefficients(b["seed"], ne, el.Nm).numpy()
        lam = b["lam"] if b["lam"] else 1.0
        y64 = o.helmholtz(el, A.numpy(), J.numpy(), lam, x)
        ld = np.longdouble
        yld = o.helmholtz(_ExtendedElement(el), A.numpy().astype(ld), J.numpy().astype(ld), ld(lam), x.astype(ld))
        assert yld.dtype == np.longdouble
        err = (np.abs(y64 - yld).max(axis=1) / np.abs(yld).max(axis=1)).max()
        assert float(err) <= 1e-13, "%s: fp64 vs extended %.2e" % (title, float(err))


def test_assembled_matrix_pins():
    """oracle.assembled_matrix: one element reproduces L + lambda M; on a 2^3 mesh of deformed
    hexes the matrix is symmetric positive definite, 1^T A 1 = lambda * volume (vertex modes of the connected
    mesh sum to 1 and L 1 = 0), and a global trilinear function has the energy of its exact integrals."""
    from workloads import assembly as asm
    from workloads import synthetic as wl
    P, lam, n = 2, 2.5, 2
    el = o.Element(o.HEX, P, P + 2)
    v0, E = wl.hex_mesh(n)
    A, J = wl.affine_factors(v0, E)
    A, J = A.numpy(), J.numpy()
    l2g, ng = asm.hex_l2g(n, P)
    l2g = l2g.numpy()
    # one element on its own: the map is a permutation-free identity when numbered locally
    M0, L0 = o.element_matrices(el, A[0], J[0])
    A1 = o.assembled_matrix(el, A[:1], J[:1], lam, np.arange(el.Nm)[None, :], el.Nm)
    assert np.abs(A1 - (L0 + lam * M0)).max() <= 1e-15 * np.abs(A1).max()
    G = o.assembled_matrix(el, A, J, lam, l2g, ng)
    assert np.abs(G - G.T).max() <= 1e-14 * np.abs(G).max()
    assert np.linalg.eigvalsh(G).min() > 0
    # the constant 1 on the connected mesh: coefficient 1 on every VERTEX dof, 0 elsewhere
    one = np.zeros(ng)
    N1 = n * P + 1
    vid = [(gx * N1 + gy) * N1 + gz for gx in range(0, N1, P) for gy in range(0, N1, P) for gz in range(0, N1, P)]
    one[vid] = 1.0
    assert abs(one @ G @ one - lam * 1.0) <= 1e-13           # 1^T (L + lam M) 1 = lam * volume of the unit cube
    assert np.abs(G @ one - lam * o.assembled_matrix(el, A, J, 1.0, l2g, ng) @ one + lam * o.assembled_matrix(el, A, J, 0.0, l2g, ng) @ one).max() <= 1e-13
    assert np.abs(o.assembled_matrix(el, A, J, 0.0, l2g, ng) @ one).max() <= 1e-13     # L 1 = 0 on the assembled mesh
    # u = x y z (trilinear, in the span of the vertex modes): energy = int |grad u|^2 + lam u^2 over the unit cube
    h = 1.0 / n
    u = np.zeros(ng)
    for gx in range(0, N1, P):
        for gy in range(0, N1, P):
            for gz in range(0, N1, P):
                u[(gx * N1 + gy) * N1 + gz] = (gx // P * h) * (gy // P * h) * (gz // P * h)
    exact = 3.0 * (1.0 / 9.0) + lam * (1.0 / 27.0)            # int (yz)^2 + (xz)^2 + (xy)^2 = 3/9 ; int (xyz)^2 = 1/27
    assert abs(u @ G @ u - exact) <= 1e-13
    # signs: flipping the sign of one shared dof in every element that holds it flips the matching rows and columns
    sign = np.ones_like(l2g, dtype=np.int8)
    g0 = int(l2g[0, el.Nm - 1])
    sign[l2g == g0] = -1
    Gs = o.assembled_matrix(el, A, J, lam, l2g, ng, sign)
    D = np.ones(ng)
    D[g0] = -1.0
    assert np.abs(Gs - D[:, None] * G * D[None, :]).max() <= 1e-15 * np.abs(G).max()


def test_constrained_matrix_pins():
    from workloads import assembly as asm
    from workloads import synthetic as wl
    P, n = 2, 2
    el = o.Element(o.HEX, P, P + 2)
    v0, E = wl.hex_mesh(n)
    A, J = wl.affine_factors(v0, E)
    l2g, ng = asm.hex_l2g(n, P)
    bd = asm.hex_boundary_dofs(n, P).numpy()
    N1 = n * P + 1
    assert len(bd) == N1 ** 3 - (N1 - 2) ** 3 and len(set(bd.tolist())) == len(bd)
    L = o.assembled_matrix(el, A.numpy(), J.numpy(), 0.0, l2g.numpy(), ng)
    assert np.linalg.eigvalsh(L).min() < 1e-12                     # pure Neumann Laplacian: singular (constants)
    Lc = o.constrained_matrix(L, bd)
    free = np.setdiff1d(np.arange(ng), bd)
    assert np.array_equal(Lc[np.ix_(free, free)], L[np.ix_(free, free)])
    assert np.array_equal(Lc[np.ix_(bd, bd)], np.eye(len(bd)))
    assert not Lc[np.ix_(bd, free)].any() and not Lc[np.ix_(free, bd)].any()
    assert np.linalg.eigvalsh(Lc).min() > 1e-6                     # boundary held: positive definite (8e-5 here)
