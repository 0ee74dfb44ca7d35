// nk_host_tables.cpp -- host precompute (layer B2): nodes, weights, derivative
// matrices, modified-basis tables and the row-major psi^b tables of the simplex
// contractions.  The formulas are deliberately NOT the ones oracle/ uses:
//   nodes     GLL: Newton on L_N' with Legendre recurrences from Chebyshev-Lobatto
//             guesses; GRJ: Newton with deflation on P^{alpha,1}_{Q-1}
//   weights   closed forms (A9), not the interpolatory integral
//   D         barycentric formula, not the Lagrange product formula
// so that the table-level parity test (tests/test_library_cpu.py) is a real check.
#include "nk_host_tables.h"

#include <cmath>

namespace nk {

double jacobi(int n, double a, double b, double x)
{
    if (n < 0) return 0.0;
    if (n == 0) return 1.0;
    double pm = 1.0, p = 0.5 * (a - b + (a + b + 2.0) * x);
    for (int k = 1; k < n; ++k) {
        const double c = 2.0 * k + a + b;
        const double num = (c + 1.0) * ((c + 2.0) * c * x + a * a - b * b) * p - 2.0 * (k + a) * (k + b) * (c + 2.0) * pm;
        const double den = 2.0 * (k + 1.0) * (k + a + b + 1.0) * c;
        pm = p;
        p = num / den;
    }
    return p;
}

static double jacobi_d(int n, double a, double b, double x)
{
    return n == 0 ? 0.0 : 0.5 * (n + a + b + 1.0) * jacobi(n - 1, a + 1.0, b + 1.0, x);
}

double psi_a(int p, double z)
{
    if (p == 0) return 0.5 * (1.0 - z);
    if (p == 1) return 0.5 * (1.0 + z);
    return 0.5 * (1.0 - z) * 0.5 * (1.0 + z) * jacobi(p - 2, 1.0, 1.0, z);
}

double psi_b(int i, int j, double z)
{
    if (i == 0) return psi_a(j, z);
    const double g = std::pow(0.5 * (1.0 - z), i);
    if (j == 0) return g;
    return g * 0.5 * (1.0 + z) * jacobi(j - 1, 2.0 * i - 1.0, 1.0, z);
}

int pair_index(int nm, int a, int b)
{
    int s = 0;
    for (int c = 0; c < a; ++c) s += nm - c;
    return s + b;
}

int num_modes(int shape, int nm)
{
    if (shape == HEX) return nm * nm * nm;
    if (shape == TET) return nm * (nm + 1) * (nm + 2) / 6;
    return nm * nm * (nm + 1) / 2;
}

static int q_count(int shape, int nm, int p) { return shape == TET ? nm - p : nm; }
static int r_count(int shape, int nm, int p, int q)
{
    if (shape == HEX) return nm;
    if (shape == TET) return nm - p - q;
    return nm - p;
}

int mode_index(int shape, int nm, int p, int q, int r)
{
    if (p < 0 || q < 0 || r < 0 || p >= nm) return -1;
    if (q >= q_count(shape, nm, p) || r >= r_count(shape, nm, p, q)) return -1;
    int m = 0;
    for (int a = 0; a < p; ++a)
        for (int b = 0; b < q_count(shape, nm, a); ++b) m += r_count(shape, nm, a, b);
    for (int b = 0; b < q; ++b) m += r_count(shape, nm, p, b);
    return m + r;
}

// ---- quadrature --------------------------------------------------------------------------
static void gll(int Q, std::vector<double>& z, std::vector<double>& w)
{
    const int N = Q - 1;
    z.assign(Q, 0.0);
    w.assign(Q, 0.0);
    auto legendre = [N](double x, double& LN, double& LNm1) {
        double pm = 1.0, p = x;
        for (int k = 1; k < N; ++k) {
            const double pn = ((2.0 * k + 1.0) * x * p - k * pm) / (k + 1.0);
            pm = p;
            p = pn;
        }
        LN = (N == 0) ? 1.0 : p;
        LNm1 = pm;
    };
    z[0] = -1.0;
    z[N] = 1.0;
    for (int i = 1; i < N; ++i) {
        double x = -std::cos(M_PI * i / N);
        for (int it = 0; it < 100; ++it) {
            double LN, LNm1;
            legendre(x, LN, LNm1);
            const double om = 1.0 - x * x;
            const double d1 = N * (LNm1 - x * LN) / om;           // L_N'
            const double d2 = (2.0 * x * d1 - N * (N + 1.0) * LN) / om; // L_N''
            const double dx = d1 / d2;
            x -= dx;
            if (std::fabs(dx) < 1e-16) break;
        }
        z[i] = x;
    }
    if (Q % 2 == 1) z[N / 2] = 0.0;
    for (int i = 0; i < Q; ++i) {
        double LN, LNm1;
        legendre(z[i], LN, LNm1);
        w[i] = 2.0 / (N * (N + 1.0) * LN * LN);
    }
}

// Gauss-Radau-Jacobi, weight (1-z)^alpha, node at -1 (A9).  Weights returned against (1-z)^alpha.
static void grj(int Q, double alpha, std::vector<double>& z, std::vector<double>& w)
{
    const int n = Q - 1;
    z.assign(Q, 0.0);
    w.assign(Q, 0.0);
    z[0] = -1.0;
    std::vector<double> r(n);
    for (int k = 0; k < n; ++k) {
        double x = -std::cos((2.0 * k + 1.0) * M_PI / (2.0 * n));
        if (k > 0) x = 0.5 * (x + r[k - 1]);
        for (int it = 0; it < 200; ++it) {
            double s = 0.0;
            for (int m = 0; m < k; ++m) s += 1.0 / (x - r[m]);
            const double f = jacobi(n, alpha, 1.0, x);
            const double df = jacobi_d(n, alpha, 1.0, x);
            const double dx = f / (df - s * f);
            x -= dx;
            if (std::fabs(dx) < 1e-16) break;
        }
        r[k] = x;
    }
    for (int k = 0; k < n; ++k) z[k + 1] = r[k];
    // insertion sort (roots come out ascending already; keep it robust)
    for (int i = 1; i < Q; ++i)
        for (int j = i; j > 0 && z[j] < z[j - 1]; --j) std::swap(z[j], z[j - 1]);
    const double c = std::pow(2.0, alpha) / (Q * (alpha + Q)); // beta = 0
    for (int i = 0; i < Q; ++i) {
        const double pv = jacobi(Q - 1, alpha, 0.0, z[i]);
        w[i] = c * (1.0 - z[i]) / (pv * pv);
    }
}

static void bary_deriv(const std::vector<double>& z, std::vector<double>& D)
{
    const int Q = (int)z.size();
    std::vector<double> lam(Q, 1.0);
    for (int j = 0; j < Q; ++j) {
        double p = 1.0;
        for (int m = 0; m < Q; ++m)
            if (m != j) p *= (z[j] - z[m]);
        lam[j] = 1.0 / p;
    }
    D.assign((size_t)Q * Q, 0.0);
    for (int i = 0; i < Q; ++i) {
        double diag = 0.0;
        for (int j = 0; j < Q; ++j) {
            if (j == i) continue;
            const double v = (lam[j] / lam[i]) / (z[i] - z[j]);
            D[(size_t)i * Q + j] = v;
            diag -= v;
        }
        D[(size_t)i * Q + i] = diag;
    }
}

bool build_host_tables(int shape, int P, int Q, HostTables& t)
{
    if (shape < HEX || shape > PRISM || P < 1 || Q < 3) return false;
    const int nm = P + 1;
    t.shape = shape;
    t.P = P;
    t.Q = Q;
    t.nm = nm;
    t.Nm = num_modes(shape, nm);
    t.Nq = Q * Q * Q;
    t.npair = nm * (nm + 1) / 2;

    // rules per direction (A9) and the collapse Jacobian folded into the weights (A16)
    double alpha[3] = {0, 0, 0};
    if (shape == TET) {
        alpha[1] = 1;
        alpha[2] = 2;
    } else if (shape == PRISM) {
        alpha[2] = 1;
    }
    for (int d = 0; d < 3; ++d) {
        if (alpha[d] == 0) {
            gll(Q, t.z[d], t.w[d]);
        } else {
            grj(Q, alpha[d], t.z[d], t.w[d]);
            const double fold = std::pow(0.5, alpha[d]);
            for (double& v : t.w[d]) v *= fold;
        }
        bary_deriv(t.z[d], t.D[d]);
    }

    // basis tables, point-major
    auto fill_a = [&](int d) {
        t.ncol[d] = nm;
        t.psi[d].assign((size_t)Q * nm, 0.0);
        for (int i = 0; i < Q; ++i)
            for (int p = 0; p < nm; ++p) t.psi[d][(size_t)i * nm + p] = psi_a(p, t.z[d][i]);
    };
    auto fill_b = [&](int d) {
        t.ncol[d] = t.npair;
        t.psi[d].assign((size_t)Q * t.npair, 0.0);
        for (int i = 0; i < Q; ++i)
            for (int a = 0; a < nm; ++a)
                for (int b = 0; b < nm - a; ++b)
                    t.psi[d][(size_t)i * t.npair + pair_index(nm, a, b)] = psi_b(a, b, t.z[d][i]);
    };
    fill_a(0);
    if (shape == TET) fill_b(1); else fill_a(1);
    if (shape == HEX) fill_a(2); else fill_b(2);

    t.n1 = 0;
    if (shape == HEX) return true;

    // ---- row-major psi^b tables of the triangular stages (Eq. 17 / Eq. 21) -------------------
    t.tab3.assign((size_t)t.npair * Q, 0.0);
    for (int row = 0; row < t.npair; ++row)
        for (int k = 0; k < Q; ++k) t.tab3[(size_t)row * Q + k] = t.psi[2][(size_t)k * t.npair + row];
    if (shape == TET) {
        t.n1 = t.npair;
        t.tab2.assign((size_t)t.npair * Q, 0.0);
        for (int row = 0; row < t.npair; ++row)
            for (int j = 0; j < Q; ++j) t.tab2[(size_t)row * Q + j] = t.psi[1][(size_t)j * t.npair + row];
    } else {
        t.n1 = nm * nm;
    }
    return true;
}

// ---- reference-element matrices of the coefficient-space form (affine elements) ------------
// Every basis function is evaluated at every quadrature point as the product of its three 1-D factors
// (A7) with the top-vertex / top-edge corrections of A8 written out as their definition (factor 1 instead
// of psi^a_0, or of psi^a_0 psi^b_00); its eta-derivatives are taken with the collocation matrices of
// Eq. 22, exactly as the kernels differentiate point values, and mapped to xi-derivatives by Eq. 23 (A17).
void build_reference_matrices(const HostTables& t, std::vector<double>& K7)
{
    const int Q = t.Q, nm = t.nm, Nm = t.Nm, Nq = t.Nq;
    std::vector<double> phi((size_t)Nq * Nm, 0.0);
    auto pt = [Q](int i, int j, int k) { return (size_t)i + (size_t)Q * (j + (size_t)Q * k); };
    for (int p = 0; p < nm; ++p) {
        const int nq2 = t.shape == TET ? nm - p : nm;
        for (int q = 0; q < nq2; ++q) {
            const int nr = t.shape == HEX ? nm : t.shape == TET ? nm - p - q : nm - p;
            for (int r = 0; r < nr; ++r) {
                const int m = mode_index(t.shape, nm, p, q, r);
                for (int k = 0; k < Q; ++k)
                    for (int j = 0; j < Q; ++j)
                        for (int i = 0; i < Q; ++i) {
                            double fa = t.psi[0][(size_t)i * nm + p], fb, fc;
                            if (t.shape == HEX) {
                                fb = t.psi[1][(size_t)j * nm + q];
                                fc = t.psi[2][(size_t)k * nm + r];
                            } else if (t.shape == TET) {
                                fb = t.psi[1][(size_t)j * t.npair + pair_index(nm, p, q)];
                                fc = t.psi[2][(size_t)k * t.npair + pair_index(nm, p + q, r)];
                                if (p == 0 && q == 1) fa = 1.0;                       // A8: top edge
                                if (p == 0 && q == 0 && r == 1) { fa = 1.0; fb = 1.0; } // A8: top vertex
                            } else {
                                fb = t.psi[1][(size_t)j * nm + q];
                                fc = t.psi[2][(size_t)k * t.npair + pair_index(nm, p, r)];
                                if (p == 0 && r == 1) fa = 1.0;                       // A8: top edge of the prism
                            }
                            phi[pt(i, j, k) * Nm + m] = fa * fb * fc;
                        }
            }
        }
    }
    // xi-derivatives, one direction at a time: g[d][n][m]
    std::vector<double> g[3];
    for (int d = 0; d < 3; ++d) g[d].assign((size_t)Nq * Nm, 0.0);
    std::vector<double> e1((size_t)Nm), e2((size_t)Nm), e3((size_t)Nm);
    for (int k = 0; k < Q; ++k)
        for (int j = 0; j < Q; ++j)
            for (int i = 0; i < Q; ++i) {
                for (int m = 0; m < Nm; ++m) e1[m] = e2[m] = e3[m] = 0.0;
                for (int r = 0; r < Q; ++r) {
                    const double a = t.D[0][(size_t)i * Q + r], b = t.D[1][(size_t)j * Q + r], c = t.D[2][(size_t)k * Q + r];
                    const double *f1 = &phi[pt(r, j, k) * Nm], *f2 = &phi[pt(i, r, k) * Nm], *f3 = &phi[pt(i, j, r) * Nm];
                    for (int m = 0; m < Nm; ++m) {
                        e1[m] += a * f1[m];
                        e2[m] += b * f2[m];
                        e3[m] += c * f3[m];
                    }
                }
                const double z1 = t.z[0][i], z2 = t.z[1][j], z3 = t.z[2][k];
                double *x1 = &g[0][pt(i, j, k) * Nm], *x2 = &g[1][pt(i, j, k) * Nm], *x3 = &g[2][pt(i, j, k) * Nm];
                for (int m = 0; m < Nm; ++m) {
                    if (t.shape == TET) {
                        const double c1 = 4.0 / ((1.0 - z2) * (1.0 - z3)), c2 = 2.0 * (1.0 + z1) / ((1.0 - z2) * (1.0 - z3));
                        const double c3 = 2.0 / (1.0 - z3), c4 = (1.0 + z2) / (1.0 - z3);
                        x1[m] = c1 * e1[m];
                        x2[m] = c2 * e1[m] + c3 * e2[m];
                        x3[m] = c2 * e1[m] + c4 * e2[m] + e3[m];
                    } else if (t.shape == PRISM) {
                        x1[m] = 2.0 / (1.0 - z3) * e1[m];
                        x2[m] = e2[m];
                        x3[m] = (1.0 + z1) / (1.0 - z3) * e1[m] + e3[m];
                    } else {
                        x1[m] = e1[m];
                        x2[m] = e2[m];
                        x3[m] = e3[m];
                    }
                }
            }
    K7.assign((size_t)7 * Nm * Nm, 0.0);
    const size_t MM = (size_t)Nm * Nm;
    for (int k = 0; k < Q; ++k)
        for (int j = 0; j < Q; ++j)
            for (int i = 0; i < Q; ++i) {
                const double w = t.w[0][i] * t.w[1][j] * t.w[2][k];
                const size_t n = pt(i, j, k) * Nm;
                const double *f = &phi[n], *x1 = &g[0][n], *x2 = &g[1][n], *x3 = &g[2][n];
                for (int m = 0; m < Nm; ++m) {
                    const double wf = w * f[m], w1 = w * x1[m], w2 = w * x2[m], w3 = w * x3[m];
                    double* row = &K7[(size_t)m * Nm];
                    for (int c = 0; c <= m; ++c) { // lower triangle; mirrored below
                        row[0 * MM + c] += w1 * x1[c];
                        row[1 * MM + c] += w1 * x2[c] + w2 * x1[c];
                        row[2 * MM + c] += w1 * x3[c] + w3 * x1[c];
                        row[3 * MM + c] += w2 * x2[c];
                        row[4 * MM + c] += w2 * x3[c] + w3 * x2[c];
                        row[5 * MM + c] += w3 * x3[c];
                        row[6 * MM + c] += wf * f[c];
                    }
                }
            }
    for (int c = 0; c < 7; ++c)
        for (int m = 0; m < Nm; ++m)
            for (int n = m + 1; n < Nm; ++n) K7[c * MM + (size_t)m * Nm + n] = K7[c * MM + (size_t)n * Nm + m];
}

} // namespace nk
