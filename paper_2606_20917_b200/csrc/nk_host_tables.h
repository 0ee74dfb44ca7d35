// nk_host_tables.h -- host precompute of the 1-D ingredients of the modified
// C0 basis and its quadrature (layer B2).  Plain C++; no CUDA; shares nothing
// with oracle/.  Citations: P:<n> = paper line, A<n> = DESIGN.md section 3.
#pragma once
#include <vector>

namespace nk {

enum { HEX = 0, TET = 1, PRISM = 2 };

struct HostTables {
    int shape = 0, P = 0, Q = 0, nm = 0, Nm = 0, Nq = 0, npair = 0;
    std::vector<double> z[3], w[3]; // nodes; weights with the collapse Jacobian folded in (A16)
    std::vector<double> D[3];       // D[d][i*Q + r] = h_r'(z_i)   (Eq. 22)
    int ncol[3] = {0, 0, 0};
    std::vector<double> psi[3];     // psi[d][i*ncol[d] + col]   (point-major, see nk.h NK_TAB_PSI)
    // simplices only: row-major copies of psi[2] / psi[1] (constant-bank operands of the triangular stages,
    // Eq. 17 / Eq. 21; the A8 corrections are compile-time special cases in csrc/nk_stage_sx.inc)
    int n1 = 0;                     // number of (p,q) lines after the r-sum
    std::vector<double> tab3;       // [row][k]  psi^b_{s,r}(z3_k), row = pair(s,r)
    std::vector<double> tab2;       // [row][j]  psi^b_{p,q}(z2_j), row = pair(p,q)   (tet)
};

// Jacobi polynomial P_n^{a,b}(x) (A7)
double jacobi(int n, double a, double b, double x);
// modified principal functions (A7)
double psi_a(int p, double z);
double psi_b(int i, int j, double z);

int pair_index(int nm, int a, int b);                   // sum_{c<a}(nm-c) + b
int mode_index(int shape, int nm, int p, int q, int r); // Eq. 18 (A3); -1 if not a mode
int num_modes(int shape, int nm);

// returns false if (shape,P,Q) is malformed (P<1, Q<2)
bool build_host_tables(int shape, int P, int Q, HostTables& t);

// Reference-element matrices of the coefficient-space form of the AFFINE operators (csrc/nk_dense.cuh):
// K7[c][m][n], c = 0..6, each Nm x Nm row-major and symmetric, with xi = standard-element coordinates,
//   c = 0: (1,1)  1: (1,2)+(2,1)  2: (1,3)+(3,1)  3: (2,2)  4: (2,3)+(3,2)  5: (3,3):
//          sum_q w_q d_a phi_m(xi_q) d_b phi_n(xi_q)   (Eq. 7, with the chain of Eq. 23, applied to the basis)
//   c = 6: sum_q w_q phi_m(xi_q) phi_n(xi_q)            (M = B^T w B, Eq. 7)
// the same discrete quadrature sums as the sum-factorised chain (w includes the collapse Jacobian, A16), so that
// (L + lambda M)_e = sum_{c<6} G^e_c K_c + lambda |J_e| K_6 for an element with constant metric G^e = |J| A A^T.
void build_reference_matrices(const HostTables& t, std::vector<double>& K7);

} // namespace nk
