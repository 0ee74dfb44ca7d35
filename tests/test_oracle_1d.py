"""Pins for the oracle's 1-D ingredients (SURVEY 8(c) 'What pins each part').
None of these retypes the oracle's own formula: closed forms, textbook
tables (tests/golden/), scipy's independent routines, exactness properties."""
import math

import numpy as np
import pytest
import scipy.special as sps

import golden_io as G
from oracle import nk_oracle as o


def test_jacobi_value_at_one_is_binomial():
    for n in range(0, 9):
        for a in (0, 1, 2, 3, 5):
            for b in (0, 1):
                assert o.jacobi(n, a, b, 1.0) == pytest.approx(math.comb(n + a, n), rel=1e-14)
    assert o.jacobi(3, 2, 1, 1.0) == pytest.approx(10.0, rel=1e-15)


def test_jacobi_explicit_polynomials():
    z = np.linspace(-1, 1, 11)
    np.testing.assert_allclose(o.jacobi(2, 1, 1, z), (15 * z * z - 3) / 4, atol=1e-15)
    np.testing.assert_allclose(o.jacobi(1, 3, 1, z), 3 * z + 1, atol=1e-15)
    np.testing.assert_allclose(o.jacobi(2, 0, 0, z), (3 * z * z - 1) / 2, atol=1e-15)
    np.testing.assert_allclose(o.jacobi(3, 0, 0, z), (5 * z ** 3 - 3 * z) / 2, atol=1e-15)


def test_jacobi_against_scipy_and_derivative():
    z = np.linspace(-0.97, 0.93, 13)
    for n in range(0, 11):
        for a, b in ((0, 0), (1, 1), (1, 0), (2, 0), (3, 1), (7, 1), (2, 1)):
            ref = sps.eval_jacobi(n, a, b, z)
            np.testing.assert_allclose(o.jacobi(n, a, b, z), ref, rtol=1e-12, atol=1e-13)
            h = 1e-6  # central difference of scipy's values pins the derivative rule
            fd = (sps.eval_jacobi(n, a, b, z + h) - sps.eval_jacobi(n, a, b, z - h)) / (2 * h)
            np.testing.assert_allclose(o.jacobi_deriv(n, a, b, z), fd, rtol=1e-6, atol=1e-6)


def _rule(tag, Q):
    if tag == "gll":
        return "gll", 0
    return ("grj", int(tag[3])), int(tag[3])


def test_quadrature_textbook_values():
    for tag, Q, zs, ws in G.records("quadrature_textbook.txt"):
        Q = int(Q)
        if tag == "grj00":
            z = np.concatenate(([-1.0], o.jacobi_roots(Q - 1, 0.0, 1.0)))
            alpha = 0
        else:
            rule, alpha = _rule(tag, Q)
            z = o.nodes(rule, Q)
        np.testing.assert_allclose(z, G.numbers(zs), atol=2e-15, err_msg=f"{tag} {Q}")
        w = o.weights(z, alpha) * 2.0 ** alpha      # undo the collapse factor (A16)
        np.testing.assert_allclose(w, G.numbers(ws), atol=5e-15, err_msg=f"{tag} {Q}")


@pytest.mark.parametrize("Q", range(3, 13))
def test_quadrature_sums_and_exactness(Q):
    # GLL: exact to degree 2Q-3, fails at 2Q-2.  GRJ(alpha,0): exact to 2Q-2
    # against ((1-z)/2)^alpha, fails at 2Q-1.
    for rule, alpha, deg in (("gll", 0, 2 * Q - 3), (("grj", 1), 1, 2 * Q - 2), (("grj", 2), 2, 2 * Q - 2)):
        z = o.nodes(rule, Q)
        w = o.weights(z, alpha)
        assert np.all(w > 0) and np.all(np.diff(z) > 0)
        assert z[0] == -1.0 and (z[-1] == 1.0 if rule == "gll" else z[-1] < 1.0)
        assert w.sum() == pytest.approx(2.0 / (alpha + 1.0), rel=1e-14)

        def exact(k):  # int ((1-z)/2)^alpha z^k dz by a 64-point Gauss-Legendre rule
            xg, wg = np.polynomial.legendre.leggauss(64)
            return np.sum(wg * (0.5 * (1 - xg)) ** alpha * xg ** k)
        for k in range(deg + 1):
            assert np.sum(w * z ** k) == pytest.approx(exact(k), abs=2e-14)
        assert abs(np.sum(w * z ** (deg + 1)) - exact(deg + 1)) > 1e-9   # one degree higher must fail


def test_gll_nodes_are_extrema_of_legendre():
    # independent characterisation: interior GLL nodes are roots of L'_{Q-1}
    for Q in range(3, 13):
        z = o.nodes("gll", Q)[1:-1]
        c = np.zeros(Q)
        c[-1] = 1
        d = np.polynomial.legendre.legval(z, np.polynomial.legendre.legder(c))
        assert np.abs(d).max() < 1e-10
        # closed-form weights 2/(Q(Q-1) L_{Q-1}(z)^2)
        zz = o.nodes("gll", Q)
        L = np.polynomial.legendre.legval(zz, c)
        np.testing.assert_allclose(o.weights(zz, 0), 2.0 / (Q * (Q - 1) * L * L), rtol=1e-12)


@pytest.mark.parametrize("Q", [3, 5, 8, 12])
def test_lagrange_derivative_matrix(Q):
    for rule in ("gll", ("grj", 1), ("grj", 2)):
        z = o.nodes(rule, Q)
        D = o.lagrange_deriv_matrix(z)
        # exact on every polynomial of degree <= Q-1, in particular constants
        assert np.abs(D.sum(axis=1)).max() < 1e-11
        for k in range(1, Q):
            np.testing.assert_allclose(D @ z ** k, k * z ** (k - 1), atol=2e-11)
        # numpy's polynomial fit/derivative as an independent interpolant
        f = np.cos(1.3 * z) + z ** 2
        co = np.polynomial.polynomial.polyfit(z, f, Q - 1)
        ref = np.polynomial.polynomial.polyval(z, np.polynomial.polynomial.polyder(co))
        np.testing.assert_allclose(D @ f, ref, atol=1e-9)


def test_modified_basis_exact_1d_matrices():
    P = 4
    xg, wg = np.polynomial.legendre.leggauss(12)
    B = np.stack([o.psi_a(p, xg) for p in range(P + 1)])
    dB = np.stack([o.dpsi_a(p, xg) for p in range(P + 1)])
    M1 = (B * wg) @ B.T
    K1 = (dB * wg) @ dB.T
    ref = {"M1": np.zeros((5, 5)), "K1": np.zeros((5, 5))}
    for name, r, c, v in G.records("modified_basis_P4.txt"):
        ref[name][int(r), int(c)] = ref[name][int(c), int(r)] = G.number(v)
    np.testing.assert_allclose(M1, ref["M1"], atol=1e-15)
    np.testing.assert_allclose(K1, ref["K1"], atol=1e-15)
    # interior derivative modes orthogonal: K1 diag = (p-1)^2 / (2(2p-1))
    for p in range(2, 5):
        assert K1[p, p] == pytest.approx((p - 1) ** 2 / (2.0 * (2 * p - 1)), rel=1e-14)


def test_psi_derivatives_by_collocation():
    # D . psi = psi' for every 1-D function used (degree <= P < Q): pins dpsi_a / dpsi_b
    P, Q = 6, 8
    for rule in ("gll", ("grj", 1), ("grj", 2)):
        z = o.nodes(rule, Q)
        D = o.lagrange_deriv_matrix(z)
        for p in range(P + 1):
            np.testing.assert_allclose(D @ o.psi_a(p, z), o.dpsi_a(p, z), atol=5e-13)
        for i in range(P + 1):
            for j in range(P + 1 - i):
                np.testing.assert_allclose(D @ o.psi_b(i, j, z), o.dpsi_b(i, j, z), atol=5e-13)


def test_psi_b_special_values():
    z = np.linspace(-1, 1, 9)
    np.testing.assert_allclose(o.psi_b(0, 3, z), o.psi_a(3, z))
    np.testing.assert_allclose(o.psi_b(2, 0, z), ((1 - z) / 2) ** 2)
    np.testing.assert_allclose(o.psi_b(1, 1, z), (1 - z) / 2 * (1 + z) / 2)          # P^{1,1}_0 = 1
    np.testing.assert_allclose(o.psi_b(2, 2, z), ((1 - z) / 2) ** 2 * (1 + z) / 2 * (3 * z + 1))   # P^{3,1}_1


def test_mode_map():
    for nm, p, q, r, m in G.records("tet_mode_map.txt"):
        assert o.mode_index(o.TET, int(nm) - 1, int(p), int(q), int(r)) == int(m)
    for shape in (o.HEX, o.TET, o.PRISM):
        for P in range(1, 11):
            ml = o.mode_list(shape, P)
            nm = P + 1
            want = {o.HEX: nm ** 3, o.TET: nm * (nm + 1) * (nm + 2) // 6, o.PRISM: nm * nm * (nm + 1) // 2}[shape]
            assert len(ml) == want and len(set(ml)) == want
            assert ml == sorted(ml)                      # lexicographic, p outermost
            assert [o.mode_index(shape, P, *t) for t in ml] == list(range(want))
            if shape != o.HEX:
                assert want < nm ** 3                    # P:211 storage count
