// nk_kernels.cuh -- sm_100a kernels of libnk (layer B0).
//
// One kernel template, nk_kernel<SHAPE,P,DEF,OP>, covers every operator of nk.h.
// Design:
//   * a thread block works on a GROUP of E elements at a time; all on-chip arrays are
//     element-interleaved, index = idx*E + e, thread = (e = tid % E, slot = tid / E).
//     A half-warp therefore touches E consecutive doubles of 16/E lines whose strides are odd
//     multiples of E: conflict-free when 16/E divides Q (a few two-way conflicts otherwise); the
//     geometry stream (stored in the same interleaved order) is read as full 32-byte sectors.
//     One block = one group (grid = number of groups): a persistent loop makes ptxas hoist and
//     spill the constant-bank matrices.
//   * every tensor contraction is "one thread per quadrature LINE": the thread pulls one
//     line of one element into registers and contracts it with a 1-D matrix whose entries
//     are compile-time-indexed kernel parameters, i.e. constant-bank operands of DFMA --
//     no shared-memory traffic for the basis / derivative matrices (Eq. 16, 20, 22).
//   * the simplex contractions with triangular bounds (Eq. 17, 21) give each warp one class
//     of lines, so that bounds and psi^b rows are warp-uniform compile-time constants
//     (nk_stage_sx.inc); the C0 corrections of A8 are compile-time special cases.
//   * the Helmholtz chain (a1..a9 of SURVEY 8(a)) is fused: three shared arrays X, Y, Z of
//     Q^3*E doubles are reused by a static plan (cf. the buffer-reuse pass);
//     quadrature-point data never goes to HBM.
#pragma once
#ifndef __CUDACC_RTC__
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>
#else
// NVRTC (run-time specialisation, csrc/nk_jit.cu) has no host headers: the one std type this file uses
namespace std {
template <class T, T v>
struct integral_constant {
    static constexpr T value = v;
    using value_type = T;
};
} // namespace std
#endif

namespace nk {

enum { K_HEX = 0, K_TET = 1, K_PRISM = 2 };
// OP_HELMF = OP_HELM on a multi-field block (its own instantiation: the field bookkeeping costs the
// single-field affine kernels 6 % at their 64-register budget)
enum { OP_BWD = 0, OP_IPROD, OP_PHYSDERIV, OP_IPDERIV, OP_MASS, OP_LAP, OP_HELM, OP_HELMF, OP_COUNT };

__host__ __device__ constexpr int k_num_modes(int shape, int nm)
{
    return shape == K_HEX ? nm * nm * nm : shape == K_TET ? nm * (nm + 1) * (nm + 2) / 6 : nm * nm * (nm + 1) / 2;
}

// ---- launch configuration per (shape, P, deformed, Q) ------------------------------------
// QQ = points per direction.  The prebuilt table (nk_inst.cu) holds QQ = P+2, the default; any other NM <= QQ <= 12 is
// specialised at run time (csrc/nk_jit.cu) with the rules below, which depend on Q rather than on P.
// E  = elements per group (interleave width), LS = line slots, threads = E*LS,
// LQ = padded length of an i-line in the point arrays (odd when E < 16 so that the
//      (j,k)-line pass stays bank-conflict-free), MINB = blocks per SM asked of ptxas.
// Values from the round-1 sweeps on B200 (profiles/r1_notes.md): deformed (HBM-bound) kernels want small
// blocks (about 150-200 threads) at up to 96 registers, many of them per SM; affine (issue / shared-memory
// bound) kernels want 72 registers and as many resident threads as that allows.
template <int SHAPE, int P, int DEF, int QQ = P + 2>
struct Tune {
    static constexpr int Q = QQ;
    static_assert(QQ >= P + 1, "a quadrature line must hold at least P+1 points (the on-chip arrays are sized by Q)");
#if defined(NK_TUNE_E)
    static constexpr int E = NK_TUNE_E;
#else
    // (deformed prisms at Q = 8: 4 since their psi^b tables sit in shared memory -- 256 threads, three blocks per SM: 0.71 -> 0.76 of HBM;
    //  tets keep 8 there: 0.67 against 0.66; simplices at Q = 10: 8 without the geometry ring -- one block of 864 threads per SM --
    //  against 4 with it: tet P8 launch 0.37 -> 0.49, prism P8 0.46 -> 0.55)
    static constexpr int E = DEF ? (Q <= 4 ? 8 : Q <= 7 ? 4 : SHAPE == K_HEX ? 2 : Q <= 8 ? (SHAPE == K_PRISM ? 4 : 8) : Q == 10 ? 8 : Q <= 11 ? 4 : 2)   // simplices at Q = 12: shared memory
                                 : (Q <= 3 ? 32 : Q <= 4 ? (SHAPE == K_HEX ? 16 : 8) : Q <= 5 ? 8 : Q <= 7 ? 4 : Q <= 8 ? 8
                                    : Q <= 10 ? 4 : 2);
#endif
    static constexpr int LQ = (E >= 16) ? Q : (Q | 1);
    static constexpr int NQP = LQ * Q * Q;
    // On simplices the triangular stages give every WARP one (s) or (p) value, so that the psi^b entries are
    // warp-uniform constant-bank operands; LS is rounded up to what those stages need.
    static constexpr int NM = P + 1, SPW = 32 / E;          // SPW = line slots per warp
    __host__ __device__ static constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }
    __host__ __device__ static constexpr int warps_s1_tet()
    {
        int w = 0;
        for (int s = 0; s < NM; ++s) w += cdiv(s + 1, SPW);
        return w;
    }
    static constexpr int WARPS_SX = SHAPE == K_HEX ? 0
                                    : SHAPE == K_TET ? (warps_s1_tet() > NM * cdiv(Q, SPW) ? warps_s1_tet() : NM * cdiv(Q, SPW))
                                                     : NM * cdiv(NM, SPW);
    static constexpr int LS_min = SHAPE == K_HEX ? 0 : WARPS_SX * SPW;
#if defined(NK_TUNE_LS)
    static constexpr int LS = NK_TUNE_LS > LS_min ? NK_TUNE_LS : LS_min;
#else
    // one line per thread per pass: single-trip stages are straight-line code whose matrix operands are
    // used once (nothing for the compiler to hoist and spill)
    static constexpr int LS = SHAPE == K_HEX ? Q * Q : cdiv((Q * Q > LS_min ? Q * Q : LS_min), SPW) * SPW;
#endif
    static constexpr int NT = E * LS;
    // RING: depth (in k-planes) of the per-thread geometry ring of the deformed Laplacian / Helmholtz kernels
    // (nk_stage_mid.inc, pass C): the 7 metric entries of the thread's next RING points are copied global -> shared
    // by cp.async while the thread works, the first RING planes from kernel entry on.  0 = plain __ldg in pass C.
#if defined(NK_TUNE_RING)
    static constexpr int RING = DEF ? (NK_TUNE_RING < Q ? NK_TUNE_RING : Q) : 0;
#else
    // B200 sweep (profiles/r2_notes.md): the ring costs 7 LDGSTS + 7 LDS per point instead of 7 LDG and loses wherever the
    // L2 prefetch alone keeps pass C fed (hexes at every order: cfg2 49.0 -> 42.8; simplices up to Q = 9: cfg5 19.5 -> 16.3);
    // it won on the simplices at Q = 10 with four elements per block (cfg5:8 10.2 -> 11.6 GDoF/s), where few warps were resident
    // to hide the L2 latency; eight elements per block without it do better still (12.6 -> 15.8, see E above), so the ring is
    // left to Q >= 11 (run-time specialised orders 9 and 10), where eight elements do not fit the shared memory
    static constexpr int RING = (DEF && SHAPE != K_HEX && Q >= 11) ? 2 : 0;
#endif
    static constexpr size_t smem_ring = (size_t)NT * RING * 7 * sizeof(double);
    // EARLY: number of k-planes of the thread's pass-C line whose 7 metric entries are requested BEFORE the barrier in
    // front of pass C (registers held across it), so that their L2 latency overlaps the wait at the barrier
    // (nk_stage_mid.inc; B200 sweep in profiles/r2_notes.md section 7)
#if defined(NK_TUNE_EARLY)
    static constexpr int EARLY = (DEF && RING == 0) ? (NK_TUNE_EARLY < Q ? NK_TUNE_EARLY : Q) : 0;
#else
    // (simplices at Q = 8, re-swept with the shared-memory tables: two planes -- prism P6 launch 0.76 -> 0.83 of HBM, tet P6 0.67 -> 0.70)
    static constexpr int EARLY = (DEF && RING == 0) ? (SHAPE != K_HEX ? (Q == 8 ? 2 : 1) : Q == 9 ? 2 : 0) : 0;
#endif
    // COLS: form of the 1-D contractions (contract below): input-outermost over the transposed tables
#if defined(NK_TUNE_COLS)
    static constexpr bool COLS = NK_TUNE_COLS != 0;
#else
    // B200 sweep over every order (profiles/r2_notes.md section 10): wins where ptxas' uniform-register shuffle is heavy --
    // hexes from Q = 10 (deformed P8 / P9 / P10 +5 / +11 / +14 %; affine Laplacian P8 / P10 +8 / +14 %, P9 -2 %) and
    // simplices from Q = 9 (config 5 P7 / P8 +3 / +9 %); below, the two forms are within 1-3 % and the row form stays
    static constexpr bool COLS = SHAPE == K_HEX ? (Q >= 10 && (DEF || Q != 11)) : Q >= 9;
#endif
    // SXS: the psi^b tables of the triangular stages (nk_stage_sx.inc) read from a shared-memory copy that every block makes
    // at entry ([2][npair * Q] doubles behind the point arrays and the ring) instead of as constant-bank operands.  In those
    // stages every warp works on its own class with its own table rows, once per block: the constant loads (LDCU) find nothing
    // in the constant cache that another warp has just used, and an ablation on B200 showed the four triangular stages of the
    // deformed tet P5 kernel cost 35 % of its time for 8 % of its DFMA (profiles/r2_notes.md section 14).  From shared
    // memory the same operands cost a fixed LDS latency.  B200 sweep (fraction of HBM, constant bank -> shared): tets P5 0.62 ->
    // 0.69, P6 0.64 -> 0.66, P7 0.36 -> 0.38, P8 0.36 -> 0.37; prisms P6 0.70 -> 0.71, P7 0.57 -> 0.63; it LOSES 2-9 % at P1..P4
    // (short blocks: the copy costs more than the few operands save) and on prisms at P5 and P8.
#if defined(NK_TUNE_SXS)
    static constexpr bool SXS = SHAPE != K_HEX && NK_TUNE_SXS != 0;
#else
    static constexpr bool SXS = DEF && ((SHAPE == K_TET && Q >= 7 && Q <= 10) || (SHAPE == K_PRISM && (Q == 8 || Q == 9)));
#endif
    // FUSE23 (tets with SXS): the q-sum S2 is done by the S3 thread for its own (j,k) line -- 21 more FMA per thread with
    // psi^b_{pq}(eta2_j) read per lane from the shared-memory table -- instead of in a triangular stage of its own: one stage
    // and one block barrier less, every thread busy (the S2 stage keeps one warp per p with 6..1 q-terms)
#if defined(NK_TUNE_FUSE23)
    static constexpr bool FUSE23 = SXS && SHAPE == K_TET && NK_TUNE_FUSE23 != 0;
#else
    static constexpr bool FUSE23 = SXS && SHAPE == K_TET;
#endif
    static constexpr size_t smem_sx = SXS ? (size_t)2 * (NM * (NM + 1) / 2) * Q * sizeof(double) : 0;
    static constexpr size_t smem_grid = (size_t)3 * NQP * E * sizeof(double) + smem_sx;
#if defined(NK_TUNE_MINB)
    static constexpr int MINB = NK_TUNE_MINB;
#else
    // registers per thread asked of ptxas (through the blocks-per-SM bound); round-2 sweep of the bound on every
    // deformed workload (profiles/r2_notes.md section 7): hexes 96 except Q = 4 (64: cfg2:2 +4 %), Q = 7 and Q = 10
    // (80: cfg2:5 +5 %, cfg2:8 +7 %); simplices 72 except Q = 6 and Q = 8 (64: cfg5:4 +6 %, cfg5:6 +12 %, where 64
    // registers let a second 512-thread block fit); tets at Q = 7: 56 since their psi^b tables sit in shared memory (SXS below:
    // five blocks of 224 threads per SM instead of four, 16 B of spills; config 5's tet launch 0.721 -> 0.741 of HBM), and at
    // Q = 9: 64 (a second 512-thread block per SM: tet P7 launch 0.38 -> 0.49)
#if defined(NK_TUNE_REGS)
    static constexpr int REGS = NK_TUNE_REGS;
#else
    static constexpr int REGS = DEF ? (SHAPE == K_HEX ? (Q == 4 ? 64 : (Q == 7 || Q == 10) ? 80 : 96) : (Q == 6 || Q == 8 || (SHAPE == K_TET && Q == 9)) ? 64 : (SHAPE == K_TET && Q == 7) ? 56 : 72)
                                    : Q <= 6 ? 56 : 64;
#endif
    static constexpr int MINB_smem = (int)((227 * 1024) / (smem_grid + smem_ring + 1024));
    static constexpr int MINB_reg = 65536 / (NT * REGS);
    static constexpr int MINB = MINB_smem < 1 ? 1 : (MINB_smem < MINB_reg ? MINB_smem : (MINB_reg < 1 ? 1 : MINB_reg));
#endif
};

// Per-operator launch configuration.  Only the affine-hex mass operator in coefficient space
// (nk_stage_masskron.inc) departs from Tune: it has nm^2 lines of nm entries, no quadrature-point arrays, and
// is bandwidth-bound, so it takes more elements per block (its own E; the geometry stream keeps Tune's E).
template <int SHAPE, int P, int DEF, int OPX, int QQ = P + 2>
struct TuneOp : Tune<SHAPE, P, DEF, QQ> {
    using B = Tune<SHAPE, P, DEF, QQ>;
    static constexpr bool AFF_HEX = (SHAPE == K_HEX && !DEF);
    static constexpr bool MASS_KRON = AFF_HEX && OPX == OP_MASS;                                   // nk_stage_masskron.inc
#if defined(NK_NO_LAPKRON)
    static constexpr bool LAP_KRON = false;
#else
    // nk_stage_lapkron.inc; up to P = 7: beyond, its stage 2 (4 nm inputs + 9 accumulators in registers) spills and the
    // quadrature-grid path is faster (B200: P8 49 vs 59 GDoF/s)
#ifndef NK_LAPKRON_MAXNM
#define NK_LAPKRON_MAXNM 8
#endif
    static constexpr bool LAP_KRON = AFF_HEX && (P + 1) <= NK_LAPKRON_MAXNM && (OPX == OP_LAP || OPX == OP_HELM || OPX == OP_HELMF);
#endif
    static constexpr bool KRON = MASS_KRON || LAP_KRON;
#if defined(NK_TUNE_KCOLS)
    static constexpr bool KCOLS = NK_TUNE_KCOLS != 0;
#else
    // coefficient-space kernels (same sweep): mass from nm = 9 on (P8..P10 +4..6 %), Laplacian / Helmholtz up to nm = 6
    // (P3 / P4 / P5 +6 / +2 / +15 %); at nm = 7, 8 the column form of stage 1 adds local-memory spills to stage 2's
    static constexpr bool KCOLS = MASS_KRON ? (P + 1) >= 9 : (P + 1) <= 6;
#endif
    static constexpr int NM = P + 1;
#if defined(NK_TUNE_EMASS)
    static constexpr int EK = NK_TUNE_EMASS;
#else
    static constexpr int EK = NM <= 2 ? 16 : NM <= 3 ? 8 : NM <= 5 ? 4 : NM <= 9 ? 2 : 1;   // 64..162 threads per block (B200 sweep)
#endif
#if defined(NK_TUNE_ELAP)
    static constexpr int EL = NK_TUNE_ELAP;
#else
    static constexpr int EL = NM <= 2 ? 16 : NM <= 3 ? 8 : NM <= 4 ? 4 : NM <= 5 ? 5 : NM <= 6 ? 2 : 1;   // B200 sweep (r1_notes.md);
                                                // 5 x 25 lines = 125 threads fill four warps, 4 x 25 = 100 waste a fifth
#endif
    static constexpr int E = MASS_KRON ? EK : LAP_KRON ? EL : B::E;
    static constexpr int LQ = KRON ? B::Q : B::LQ;        // unused by the coefficient-space kernels
    static constexpr int NMP = (NM % 4 == 0) ? NM + 1 : NM;   // padded stride of the coefficient cube
    static constexpr int NQP = KRON ? NMP * NMP * NMP : B::NQP;
    static constexpr int NARR = MASS_KRON ? 2 : LAP_KRON ? 4 : 3;
    static constexpr int LS = KRON ? NM * NM : B::LS;
    static constexpr int NT = KRON ? E * LS : B::NT;
    static constexpr bool USE_RING = B::RING > 0 && DEF && (OPX == OP_LAP || OPX == OP_HELM || OPX == OP_HELMF);
    static constexpr int RING = USE_RING ? B::RING : 0;
    static constexpr size_t smem_grid = KRON ? (size_t)NARR * NQP * E * sizeof(double) : B::smem_grid + (USE_RING ? B::smem_ring : 0);
#if defined(NK_TUNE_REGSK)
    static constexpr int REGSK = NK_TUNE_REGSK;
#else
    static constexpr int REGSK = MASS_KRON ? 40 : NM <= 2 ? 64 : NM <= 5 ? 96 : 128;
#endif
    static constexpr int MINB_k = 65536 / (NT * REGSK) > 16 ? 16 : 65536 / (NT * REGSK);
    // affine tet P4 Laplacian / Helmholtz: 48 registers = 8 blocks of 160 threads per SM (24 B of spills) instead of 7 at
    // 56: 20.67 against 20.43 GDoF/s (r1_notes.md 16); the other operators of that block spill more and keep 56
#if defined(NK_TUNE_MINB)
    static constexpr bool TET48 = false;
#else
    static constexpr bool TET48 = SHAPE == K_TET && !DEF && P == 4 && QQ == 6 && B::E == 4 && (OPX == OP_LAP || OPX == OP_HELM || OPX == OP_HELMF);
#endif
    static constexpr int MINB = KRON ? (MINB_k < 1 ? 1 : MINB_k) : TET48 ? 8 : B::MINB;
};

// ---- kernel parameters (constant bank) -------------------------------------------------
template <int NM, int Q, bool HEXK = true>
struct DenseTabs {
    double Ba[3][Q * NM];  // [d][i][p]  psi^a_p at the GLL points, one copy per direction that uses it
    double BaT[3][NM * Q]; // [d][p][i]  transposes: operands of the adjoint passes (Eq. 20).
                           // One copy per use site on purpose: loads of one address would be merged by the
                           // compiler, kept in registers from a forward pass to its adjoint, and spilled.
    // 1-D matrices of the coefficient-space (Kronecker) form of the affine hex operators, [stage][which][p'][p]:
    // which = 0: M = Ba^T w Ba, 1: K = (D Ba)^T w (D Ba), 2: C = Ba^T w (D Ba), 3: C^T; stage 0 acts on index r,
    // 1 on q, 2 on p (one copy per stage: see Ba).  nk_stage_masskron.inc, nk_stage_lapkron.inc
    double KM[3][4][HEXK ? NM * NM : 1];   // hexes only (one dummy entry each on simplices: parameter space)
    double D[3][Q * Q];  // [d][i][r]  D^(d)[i][r] = h_r'(z_i)   (Eq. 22)
    double DT[3][Q * Q]; // [d][r][i]  transposes
    double w[3][Q];      // 1-D weights (collapse Jacobian folded in, A16)
    double aux[7][Q];    // chain helpers (A17): 1+z1, 1+z2, 1/(1-z2), s = 1/(1-z3), 1/s, w3 s^2 (tet) or w3 s (prism), w3 s
};

// pair index of the psi^b tables: row (a,b), a+b <= P  ->  sum_{c<a}(nm-c) + b
__host__ __device__ constexpr int k_pair(int nm, int a, int b) { return a * nm - a * (a - 1) / 2 + b; }
// storage rank of mode (p,q,0) (Eq. 18, A3)
__host__ __device__ constexpr int k_tet_mode0(int nm, int p, int q)
{
    return p * (3 * nm * nm - 3 * nm * p + 6 * nm + p * p - 3 * p + 2) / 6 + q * (nm - p) - q * (q - 1) / 2;
}
__host__ __device__ constexpr int k_prism_mode0(int nm, int p, int q)
{
    return nm * (p * nm - p * (p - 1) / 2) + q * (nm - p);
}

// psi^b tables of the collapsed directions (A7), constant-bank operands of the simplex stages.
// Row = k_pair(a,b), Q entries per row (contiguous in the point index).  Forward and adjoint stages have
// their own copies (same reason as DenseTabs).  NRQ = npair*Q on simplices, 1 on hexes (unused).
// DUP = false: ONE copy serves both (the adjoint accessors return the forward arrays).  Only where two copies do not fit
// the 32 KB kernel-parameter space next to DenseTabs: tets and prisms at P = 10, Q = 12 (run-time specialised only).
template <int NRQ, bool DUPL = true>
struct SimplexTabs {
    static constexpr bool DUP = DUPL;
    double b3f[NRQ], b3a[DUPL ? NRQ : 1]; // psi^b_{s,r}(eta3_k): tet s = p+q, prism s = p
    double b2f[NRQ], b2a[DUPL ? NRQ : 1]; // psi^b_{p,q}(eta2_j): tet only
    __device__ __forceinline__ const double* a3() const { if constexpr (DUPL) return b3a; else return b3f; }
    __device__ __forceinline__ const double* a2() const { if constexpr (DUPL) return b2a; else return b2f; }
};
// doubles of DenseTabs<NM, Q, HEXK> (declaration order: Ba, BaT, KM, D, DT, w, aux)
__host__ __device__ constexpr int k_dense_doubles(int nm, int Q, bool hexk) { return 6 * Q * nm + 12 * (hexk ? nm * nm : 1) + 6 * Q * Q + 10 * Q; }
// do two copies of the psi^b tables fit the kernel-parameter space (32000 B with 512 B left for KArgs)?
__host__ __device__ constexpr bool k_sx_dup(int shape, int nm, int Q)
{
    return shape == K_HEX || (k_dense_doubles(nm, Q, false) + 4 * (nm * (nm + 1) / 2) * Q) * 8 + 512 <= 32000;
}
template <int SHAPE, int NM, int Q>
struct SimplexTabsFor {
    using type = SimplexTabs<(SHAPE == K_HEX) ? 1 : (NM * (NM + 1) / 2) * Q, k_sx_dup(SHAPE, NM, Q)>;
};

enum { K_MAX_FIELDS = 8 };
struct KArgs {
    const double* in[3];
    double* out[3];
    // multi-field blocks: nfields coefficient fields share one geometry.  Block b works on group
    // b / nfields of field b % nfields: the blocks of one group are neighbours in launch order, run at the
    // same time, and the geometry is read from DRAM once and from L2 by the others.
    const double* fin[K_MAX_FIELDS];
    double* fout[K_MAX_FIELDS];
    int nfields;             // 1 for the single-field calls (then fin[0] == in[0], fout[0] == out[0])
    const double* geom;      // metric stream (7 comps) or factor stream (10 comps), see nk_api.cu
    double lambda;
    long long nelem;
    int ngroups;             // groups of the whole block of elements
    int g0, grid_groups;     // this launch works on groups [g0, g0 + grid_groups) (chunked host pipeline)
    int pf_dist;             // L2 prefetch distance in groups = number of co-resident blocks
};

// runtime value -> compile-time constant: f(std::integral_constant<int, v>) for v in [0, N)
template <int N, class F>
__device__ __forceinline__ void static_switch(int v, F&& f)
{
    if constexpr (N > 0) {
        if (v == N - 1)
            f(std::integral_constant<int, N - 1>{});
        else
            static_switch<N - 1>(v, static_cast<F&&>(f));
    }
}

#define NK_UNROLL _Pragma("unroll")
// acc[o] += sum_r M[o][r] * in[r]: a register line times a constant-bank 1-D matrix, given both as M ([o][r], row-major)
// and as its transpose MT ([r][o], contiguous in the OUTPUT index).
//   COLS = false: output-outermost over M (one dot product after the other in the source).
//   COLS = true:  input-outermost over MT.
// ptxas runs the NOUT accumulators side by side whatever the source order.  From the row-major table it then fetches
// pairs along the INPUT index (LDCU.128), parks their second halves in uniform registers and shuffles them with UMOV:
// 0.6 UMOV per DFMA at Q = 12 and uniform-register spills from Q = 9 on, a quarter of all instructions of the deformed
// hex P10 kernel (profiles/r2_notes.md section 10).  With MT every LDCU.128 pair feeds the next two DFMA and dies.
// The order of every single sum (r ascending) is the same in both forms: results are bit-identical.
template <bool COLS, int NOUT, int NIN>
__device__ __forceinline__ void contract(const double* __restrict__ M, const double* __restrict__ MT, const double (&in)[NIN],
                                         double (&acc)[NOUT])
{
    if constexpr (COLS) {
        NK_UNROLL for (int r = 0; r < NIN; ++r)
            NK_UNROLL for (int o = 0; o < NOUT; ++o) acc[o] = fma(MT[r * NOUT + o], in[r], acc[o]);
    } else {
        NK_UNROLL for (int o = 0; o < NOUT; ++o) {
            double a = acc[o];
            NK_UNROLL for (int r = 0; r < NIN; ++r) a = fma(M[o * NIN + r], in[r], a);
            acc[o] = a;
        }
    }
}
template <int N>
__device__ __forceinline__ void zero(double (&v)[N])
{
    NK_UNROLL for (int i = 0; i < N; ++i) v[i] = 0.0;
}
// line loop of a stage: thread `slot` takes lines slot, slot+LS, ...  The trip count is a compile-time
// constant so that single-trip stages are straight-line code.
// NK_FORU: the same, fully unrolled (global loads/stores: all trips in flight at once)
#define NK_FORU(l, N) \
    _Pragma("unroll") for (int l = slot, l##_t = 0; l##_t < ((N) + LS - 1) / LS; ++l##_t, l += LS) if (active && l < (N))
#define NK_FOR(l, N) \
    _Pragma("unroll 1") for (int l = slot, l##_t = 0; l##_t < ((N) + LS - 1) / LS; ++l##_t, l += LS) if (active && l < (N))

} // namespace nk
