"""nk_oracle -- plain CPU fp64 oracle for the spectral/hp elemental operators.

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2606_20917_b200/)
imports, links or executes this file; only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may.  It shares no code, table
or constant with the CUDA library: every number here is built from the
definitions below (numpy + numpy.polynomial.legendre.leggauss as library steps).

What it computes (citations: P:<line> = /root/reference/PAPER.md line;
A<n> = the reading of that number in DESIGN.md section 3):

  * 1-D ingredients: Jacobi polynomials by the three-term recurrence, GLL /
    Gauss-Radau-Jacobi nodes by Newton iteration, weights by the interpolatory
    definition w_i = int ((1-z)/2)^alpha h_i(z) dz (A9, A16), Lagrange
    derivative matrices by the product formula (Eq. 22).
  * the basis phi_m(xi_n) (Eq. 8) and its reference gradient, explicitly,
    for every mode m and every quadrature point n (A7, A8, A17);
  * per element, the *plain definition* of each operator as a dense
    O(Nq*Nm) sum (Eqs. 14-15, 19, 9, 7, 6): no sum-factorisation, no fusion.
    Sum-factorisation is a reassociation of these same sums, so the
    plain definition is the oracle.

Parity pins (tests/test_oracle_*.py, all CPU): Jacobi closed forms and scipy,
textbook quadrature values, exact 1-D mass/stiffness matrices, Kronecker closed
forms for affine hexes, textbook P1 tet/prism matrices, polynomial-span and
partition-of-unity checks of the collapsed bases, exact differentiation of
polynomials, operator identities.  The paper prints no numerical example, so
every pin comes from the mathematics; no function is unpinned.
"""
import numpy as np
from numpy.polynomial.legendre import leggauss

HEX, TET, PRISM = 0, 1, 2


# --------------------------------------------------------------------------
# O1. Jacobi polynomials (A7: standard three-term recurrence)
# --------------------------------------------------------------------------
def jacobi(n, alpha, beta, z):
    """P_n^{alpha,beta}(z).  P_0 = 1, P_1 = ((alpha-beta) + (alpha+beta+2) z)/2."""
    z = np.asarray(z, dtype=np.float64)
    if n < 0:
        return np.zeros_like(z)
    pm1 = np.ones_like(z)
    if n == 0:
        return pm1
    p = 0.5 * ((alpha - beta) + (alpha + beta + 2.0) * z)
    for k in range(1, n):
        s = 2.0 * k + alpha + beta
        a1 = 2.0 * (k + 1.0) * (k + alpha + beta + 1.0) * s
        a2 = (s + 1.0) * (alpha * alpha - beta * beta)
        a3 = s * (s + 1.0) * (s + 2.0)
        a4 = 2.0 * (k + alpha) * (k + beta) * (s + 2.0)
        pm1, p = p, ((a2 + a3 * z) * p - a4 * pm1) / a1
    return p


def jacobi_deriv(n, alpha, beta, z):
    """d/dz P_n^{alpha,beta} = (n+alpha+beta+1)/2 * P_{n-1}^{alpha+1,beta+1}."""
    z = np.asarray(z, dtype=np.float64)
    if n == 0:
        return np.zeros_like(z)
    return 0.5 * (n + alpha + beta + 1.0) * jacobi(n - 1, alpha + 1.0, beta + 1.0, z)


def jacobi_roots(n, alpha, beta):
    """The n roots of P_n^{alpha,beta}, ascending: Newton iteration with
    deflation from Chebyshev starting points."""
    r = np.zeros(n)
    for k in range(n):
        x = -np.cos((2.0 * k + 1.0) * np.pi / (2.0 * n))
        if k > 0:
            x = 0.5 * (x + r[k - 1])
        for _ in range(200):
            s = np.sum(1.0 / (x - r[:k]))
            f = float(jacobi(n, alpha, beta, x))
            df = float(jacobi_deriv(n, alpha, beta, x))
            dx = -f / (df - s * f)
            x += dx
            if abs(dx) < 1e-16:
                break
        r[k] = x
    return np.sort(r)


# --------------------------------------------------------------------------
# O1. Quadrature rules (A9) and Lagrange derivative matrices (Eq. 22)
# --------------------------------------------------------------------------
def nodes(rule, Q):
    """rule 'gll': +-1 and the roots of P^{1,1}_{Q-2};
    rule ('grj', alpha): -1 and the roots of P^{alpha,1}_{Q-1} (Radau node at -1,
    +1 excluded so that the collapsed-coordinate factors stay finite)."""
    if rule == "gll":
        return np.concatenate(([-1.0], jacobi_roots(Q - 2, 1.0, 1.0), [1.0]))
    kind, alpha = rule
    assert kind == "grj"
    return np.concatenate(([-1.0], jacobi_roots(Q - 1, float(alpha), 1.0)))


def lagrange_basis(z, r, x):
    """h_r(x): the Lagrange polynomial through nodes z that is 1 at z_r."""
    x = np.asarray(x, dtype=np.float64)
    h = np.ones_like(x)
    for l in range(len(z)):
        if l != r:
            h = h * (x - z[l]) / (z[r] - z[l])
    return h


def weights(z, alpha):
    """Interpolatory definition, collapse Jacobian folded in (A16):
    w_i = int_{-1}^{1} ((1-x)/2)^alpha h_i(x) dx, by a 40-point Gauss-Legendre
    rule (exact: the integrand has degree len(z)-1+alpha <= 13)."""
    xg, wg = leggauss(40)
    return np.array([np.sum(wg * (0.5 * (1.0 - xg)) ** alpha * lagrange_basis(z, i, xg))
                     for i in range(len(z))])


def lagrange_deriv_matrix(z):
    """D[i][r] = h_r'(z_i) by the product formula
    h_r'(x) = sum_{m!=r} 1/(z_r-z_m) prod_{l!=r,m} (x-z_l)/(z_r-z_l)  (Eq. 22)."""
    Q = len(z)
    D = np.zeros((Q, Q))
    for i in range(Q):
        for r in range(Q):
            acc = 0.0
            for m in range(Q):
                if m == r:
                    continue
                term = 1.0 / (z[r] - z[m])
                for l in range(Q):
                    if l != r and l != m:
                        term *= (z[i] - z[l]) / (z[r] - z[l])
                acc += term
            D[i, r] = acc
    return D


# --------------------------------------------------------------------------
# O2. 1-D modified principal functions (A7) and their derivatives
# --------------------------------------------------------------------------
def psi_a(p, z):
    z = np.asarray(z, dtype=np.float64)
    if p == 0:
        return 0.5 * (1.0 - z)
    if p == 1:
        return 0.5 * (1.0 + z)
    return 0.25 * (1.0 - z) * (1.0 + z) * jacobi(p - 2, 1.0, 1.0, z)


def dpsi_a(p, z):
    z = np.asarray(z, dtype=np.float64)
    if p == 0:
        return -0.5 * np.ones_like(z)
    if p == 1:
        return 0.5 * np.ones_like(z)
    return (-0.5 * z) * jacobi(p - 2, 1.0, 1.0, z) \
        + 0.25 * (1.0 - z) * (1.0 + z) * jacobi_deriv(p - 2, 1.0, 1.0, z)


def psi_b(i, j, z):
    z = np.asarray(z, dtype=np.float64)
    if i == 0:
        return psi_a(j, z)
    if j == 0:
        return (0.5 * (1.0 - z)) ** i
    return (0.5 * (1.0 - z)) ** i * 0.5 * (1.0 + z) * jacobi(j - 1, 2.0 * i - 1.0, 1.0, z)


def dpsi_b(i, j, z):
    z = np.asarray(z, dtype=np.float64)
    if i == 0:
        return dpsi_a(j, z)
    g = (0.5 * (1.0 - z)) ** i
    dg = -0.5 * i * (0.5 * (1.0 - z)) ** (i - 1)
    if j == 0:
        return dg
    h = 0.5 * (1.0 + z)
    J = jacobi(j - 1, 2.0 * i - 1.0, 1.0, z)
    dJ = jacobi_deriv(j - 1, 2.0 * i - 1.0, 1.0, z)
    return dg * h * J + g * 0.5 * J + g * h * dJ


# --------------------------------------------------------------------------
# Mode ordering (A3: the nest order of Eq. 17 -- p outermost, r innermost)
# --------------------------------------------------------------------------
def mode_list(shape, P):
    """All (p,q,r) of an order-P expansion in storage order."""
    out = []
    for p in range(P + 1):
        if shape == HEX:
            qs = range(P + 1)
        elif shape == TET:
            qs = range(P + 1 - p)
        else:
            qs = range(P + 1)
        for q in qs:
            if shape == HEX:
                rs = range(P + 1)
            elif shape == TET:
                rs = range(P + 1 - p - q)
            else:
                rs = range(P + 1 - p)
            for r in rs:
                out.append((p, q, r))
    return out


def mode_index(shape, P, p, q, r):
    """Closed form of the rank of (p,q,r) in mode_list (A3 reading of Eq. 18)."""
    nm = P + 1
    if shape == HEX:
        return (p * nm + q) * nm + r
    if shape == TET:
        return p * (3 * nm * nm - 3 * nm * p + 6 * nm + p * p - 3 * p + 2) // 6 \
            + q * (2 * nm - 2 * p - q + 1) // 2 + r
    # prism: sum_{a<p} nm*(nm-a) + q*(nm-p) + r
    return nm * (p * nm - p * (p - 1) // 2) + q * (nm - p) + r


# --------------------------------------------------------------------------
# O2. The standard element: points, weights, explicit basis and gradient
# --------------------------------------------------------------------------
class Element:
    """Standard element of `shape`, order P, Q points per direction.

    Point index n = i + Q*(j + Q*k) (A11).  Attributes:
      z[d], w[d]   1-D nodes / weights (collapse Jacobian folded in, A16)
      D[d]         Lagrange derivative matrix of direction d (Eq. 22)
      eta [Nq,3]   collapsed coordinates of the points; xi [Nq,3] standard ones
      wq  [Nq]     w1_i w2_j w3_k
      Phi [Nq,Nm]  phi_m(xi_n)            (Eq. 8)
      dPhi[3][Nq,Nm]  d phi_m / d xi_d    (analytic, then Eq. 23 chain, A17)
    """

    def __init__(self, shape, P, Q):
        self.shape, self.P, self.Q = shape, P, Q
        if shape == HEX:
            rules = ["gll", "gll", "gll"]
            alphas = [0, 0, 0]
        elif shape == TET:
            rules = ["gll", ("grj", 1), ("grj", 2)]
            alphas = [0, 1, 2]
        else:
            rules = ["gll", "gll", ("grj", 1)]
            alphas = [0, 0, 1]
        self.z = [nodes(rules[d], Q) for d in range(3)]
        self.w = [weights(self.z[d], alphas[d]) for d in range(3)]
        self.D = [lagrange_deriv_matrix(self.z[d]) for d in range(3)]
        self.modes = mode_list(shape, P)
        self.Nm, self.Nq = len(self.modes), Q ** 3

        def grid(f3, f2, f1):  # [k][j][i] flattened: n = i + Q j + Q^2 k
            return np.einsum("k,j,i->kji", f3, f2, f1).reshape(-1)

        one = np.ones(Q)
        z1, z2, z3 = self.z
        e1, e2, e3 = grid(one, one, z1), grid(one, z2, one), grid(z3, one, one)
        self.eta = np.stack([e1, e2, e3], axis=1)
        self.wq = grid(self.w[2], self.w[1], self.w[0])
        if shape == HEX:
            self.xi = self.eta.copy()
        elif shape == TET:      # inverse of Eq. 13 (A2)
            self.xi = np.stack([(1 + e1) * (1 - e2) * (1 - e3) / 4 - 1,
                                (1 + e2) * (1 - e3) / 2 - 1, e3], axis=1)
        else:
            self.xi = np.stack([(1 + e1) * (1 - e3) / 2 - 1, e2, e3], axis=1)

        Phi = np.zeros((self.Nq, self.Nm))
        dEta = np.zeros((3, self.Nq, self.Nm))
        zero = np.zeros(Q)
        for m, (p, q, r) in enumerate(self.modes):
            if shape == HEX:
                f = [psi_a(p, z1), psi_a(q, z2), psi_a(r, z3)]
                df = [dpsi_a(p, z1), dpsi_a(q, z2), dpsi_a(r, z3)]
            elif shape == TET:
                f = [psi_a(p, z1), psi_b(p, q, z2), psi_b(p + q, r, z3)]
                df = [dpsi_a(p, z1), dpsi_b(p, q, z2), dpsi_b(p + q, r, z3)]
                if (p, q) == (0, 1):            # A8: top-edge modes
                    f[0], df[0] = one, zero
                if (p, q, r) == (0, 0, 1):      # A8: top vertex
                    f[0], df[0] = one, zero
                    f[1], df[1] = one, zero
            else:
                f = [psi_a(p, z1), psi_a(q, z2), psi_b(p, r, z3)]
                df = [dpsi_a(p, z1), dpsi_a(q, z2), dpsi_b(p, r, z3)]
                if (p, r) == (0, 1):            # A8: collapsed-edge modes
                    f[0], df[0] = one, zero
            Phi[:, m] = grid(f[2], f[1], f[0])
            dEta[0, :, m] = grid(f[2], f[1], df[0])
            dEta[1, :, m] = grid(f[2], df[1], f[0])
            dEta[2, :, m] = grid(df[2], f[1], f[0])
        self.Phi = Phi
        self.dPhi = self.chain(dEta)

    def chain(self, dEta):
        """Eq. 23 with the factors of A17: d/d xi from d/d eta, pointwise.
        dEta: [3][Nq, ...] -> [3][Nq, ...]."""
        if self.shape == HEX:
            return np.array(dEta, copy=True)
        e1, e2, e3 = (self.eta[:, d].reshape((-1,) + (1,) * (dEta[0].ndim - 1)) for d in range(3))
        out = np.empty_like(np.asarray(dEta))
        if self.shape == TET:
            c1 = 4.0 / ((1 - e2) * (1 - e3))
            c2 = 2.0 * (1 + e1) / ((1 - e2) * (1 - e3))
            c3 = 2.0 / (1 - e3)
            c4 = (1 + e2) / (1 - e3)
            out[0] = c1 * dEta[0]
            out[1] = c2 * dEta[0] + c3 * dEta[1]
            out[2] = c2 * dEta[0] + c4 * dEta[1] + dEta[2]
        else:
            out[0] = 2.0 / (1 - e3) * dEta[0]
            out[1] = dEta[1]
            out[2] = (1 + e1) / (1 - e3) * dEta[0] + dEta[2]
        return out


# --------------------------------------------------------------------------
# O3. Operators, per element, as plain dense sums.
# Geometry: dxi_dx [ne][npt][3][3], entry [j][i] = d xi_j / d x_i (A14);
# detJ [ne][npt] > 0; npt = 1 (affine) or Nq (deformed).
# Fields are element-major: coefficients [ne][Nm], point values [ne][Nq].
# --------------------------------------------------------------------------
def _W(el, detJ):
    """Diagonal of W^e: quadrature weights times |J|."""
    return el.wq[None, :] * np.broadcast_to(detJ, (detJ.shape[0], el.Nq))


def _A(el, dxi_dx):
    return np.broadcast_to(dxi_dx, (dxi_dx.shape[0], el.Nq, 3, 3))


def bwdtrans(el, uhat):
    """u_n = sum_m uhat_m phi_m(xi_n)  (Eq. 15)."""
    return np.einsum("nm,em->en", el.Phi, uhat)


def iprod(el, detJ, u):
    """uhat_m = sum_n W_n phi_m(xi_n) u_n  (Eq. 19)."""
    return np.einsum("nm,en->em", el.Phi, _W(el, detJ) * u)


def standard_deriv(el, u):
    """Eq. 22 (A5) along each direction of the point grid, then Eq. 23.
    Returns [3][ne][Nq]: d u / d xi_d."""
    Q = el.Q
    g = u.reshape(-1, Q, Q, Q)                       # [e][k][j][i]
    d1 = np.einsum("ir,ekjr->ekji", el.D[0], g).reshape(u.shape)
    d2 = np.einsum("js,eksi->ekji", el.D[1], g).reshape(u.shape)
    d3 = np.einsum("kt,etji->ekji", el.D[2], g).reshape(u.shape)
    dEta = np.stack([d1.T, d2.T, d3.T])              # [3][Nq][ne]
    dXi = el.chain(dEta)
    return np.stack([dXi[d].T for d in range(3)])


def physderiv(el, dxi_dx, u):
    """(du/dx_i)_n = sum_j (d xi_j/d x_i)_n (du/d xi_j)_n  (Eq. 9).
    Returns [3][ne][Nq]."""
    dXi = standard_deriv(el, u)
    return np.einsum("enji,jen->ien", _A(el, dxi_dx), dXi)


def iprod_deriv(el, dxi_dx, detJ, g):
    """uhat_m = sum_n W_n sum_i (grad_x phi_m)_i(xi_n) g_i,n,
    grad_x phi_m = A^T grad_xi phi_m  (Eq. 7).  g: [3][ne][Nq]."""
    W = _W(el, detJ)
    t = np.einsum("enji,ien->jen", _A(el, dxi_dx), g) * W[None]     # [j][e][n]
    return np.einsum("jnm,jen->em", el.dPhi, t)


def mass(el, detJ, uhat):
    """(M uhat)_m = sum_n W_n phi_m(xi_n) u_n,  u = B uhat  (Eq. 7)."""
    return iprod(el, detJ, bwdtrans(el, uhat))


def laplacian(el, dxi_dx, detJ, uhat):
    """(L uhat)_m = sum_n W_n grad_x phi_m . grad_x u  (Eq. 7), with
    grad_x u = sum_m' uhat_m' grad_x phi_m' from the ANALYTIC basis gradient."""
    dXi = np.einsum("jnm,em->jen", el.dPhi, uhat)
    gx = np.einsum("enji,jen->ien", _A(el, dxi_dx), dXi)
    return iprod_deriv(el, dxi_dx, detJ, gx)


def helmholtz(el, dxi_dx, detJ, lam, uhat):
    """H uhat = (L + lambda M) uhat  (Eq. 6; A6)."""
    return laplacian(el, dxi_dx, detJ, uhat) + lam * mass(el, detJ, uhat)


def element_matrices(el, dxi_dx, detJ):
    """Dense M^e and L^e of ONE element (Eq. 7) -- for the pins.
    dxi_dx [npt][3][3], detJ [npt]."""
    W = el.wq * np.broadcast_to(detJ, (el.Nq,))
    A = np.broadcast_to(dxi_dx, (el.Nq, 3, 3))
    M = el.Phi.T @ (W[:, None] * el.Phi)
    gx = np.einsum("nji,jnm->inm", A, el.dPhi)       # grad_x phi_m at n
    L = np.einsum("inm,n,inl->ml", gx, W, gx)
    return M, L



# --------------------------------------------------------------------------
# O4. Assembled operator (the paper leaves assembly out).
# By definition the global matrix is the sum of the elemental matrices placed by
# the local-to-global map: A = sum_e Q_e^T (L^e + lambda M^e) Q_e with
# (Q_e)[m][g] = sign[e][m] if g == l2g[e][m] else 0.  Dense, tiny meshes only.
# Pins (tests/test_oracle_operators.py): one element reproduces L^e + lambda M^e;
# A is symmetric positive definite for lambda > 0; 1^T A 1 = lambda * volume and
# L 1 = 0 (the vertex modes sum to 1); a global polynomial of degree <= P,
# interpolated on the C0 modes, has the energy u^T A u of its exact integrals.
# --------------------------------------------------------------------------
def assembled_matrix(el, dxi_dx, detJ, lam, l2g, nglobal, sign=None):
    """dense [nglobal][nglobal]; dxi_dx [ne][npt][3][3], detJ [ne][npt], l2g [ne][Nm] ints, sign [ne][Nm] of +-1."""
    A = np.zeros((nglobal, nglobal))
    for e in range(l2g.shape[0]):
        M, L = element_matrices(el, dxi_dx[e], detJ[e])
        H = L + lam * M
        s = np.ones(el.Nm) if sign is None else sign[e].astype(np.float64)
        H = s[:, None] * H * s[None, :]
        for m in range(el.Nm):
            for n in range(el.Nm):
                A[l2g[e, m], l2g[e, n]] += H[m, n]
    return A


def constrained_matrix(A, dofs):
    """A_c = P A P + (I - P), P = projector on the dofs NOT in `dofs`: rows and columns of the constrained dofs replaced
    by those of the identity (homogeneous Dirichlet conditions).  Pins: equals A on the free-free block, identity on the
    constrained block, zero between them; the Poisson matrix (lambda = 0) with the whole boundary held is positive definite."""
    Ac = A.copy()
    Ac[dofs, :] = 0.0
    Ac[:, dofs] = 0.0
    Ac[dofs, dofs] = 1.0
    return Ac
