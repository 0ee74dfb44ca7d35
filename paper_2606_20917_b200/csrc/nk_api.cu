// nk_api.cu -- the C-ABI of include/nk.h (layer B3), the dispatcher (B1), the geometry repack
// kernels and the fp64 probe.  No torch types, no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/nk.h"
#include "nk_dense_launch.h"
#include "nk_host_tables.h"
#include "nk_launch.h"

#define NK_DECL(s, p) extern "C" const nk::InstInfo* NK_INST_NAME(s, p)();
#define NK_LIST10(s) NK_DECL(s, 1) NK_DECL(s, 2) NK_DECL(s, 3) NK_DECL(s, 4) NK_DECL(s, 5) NK_DECL(s, 6) NK_DECL(s, 7) NK_DECL(s, 8)
NK_LIST10(0) NK_DECL(0, 9) NK_DECL(0, 10)
NK_LIST10(1)
NK_LIST10(2)

namespace {

thread_local std::string g_err;
long long g_launches = 0;
std::mutex g_mutex;

nk_status fail(nk_status s, const std::string& msg)
{
    g_err = msg;
    return s;
}
nk_status cuda_fail(cudaError_t e, const char* what)
{
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return NK_ERR_CUDA;
}

typedef const nk::InstInfo* (*InstGetter)();
const int kMaxP[3] = {10, 8, 8};
InstGetter inst_getter(int shape, int P)
{
#define NK_G(s, p) NK_INST_NAME(s, p)
    static const InstGetter tab[3][10] = {
        {NK_G(0, 1), NK_G(0, 2), NK_G(0, 3), NK_G(0, 4), NK_G(0, 5), NK_G(0, 6), NK_G(0, 7), NK_G(0, 8), NK_G(0, 9), NK_G(0, 10)},
        {NK_G(1, 1), NK_G(1, 2), NK_G(1, 3), NK_G(1, 4), NK_G(1, 5), NK_G(1, 6), NK_G(1, 7), NK_G(1, 8), nullptr, nullptr},
        {NK_G(2, 1), NK_G(2, 2), NK_G(2, 3), NK_G(2, 4), NK_G(2, 5), NK_G(2, 6), NK_G(2, 7), NK_G(2, 8), nullptr, nullptr}};
    if (shape < 0 || shape > 2 || P < 1 || P > kMaxP[shape]) return nullptr;
    return tab[shape][P - 1];
}

// form of the affine mass / Laplacian / Helmholtz operators (nk.h, nk_set_affine_simplex_form): 0 = automatic (the
// reference-matrix DMMA kernel where it is the faster one, see use_dense below), 1 = never the reference-matrix kernel,
// 2 = always (specialised at run time where no kernel is prebuilt).  Initial value from the environment variable
// NK_SIMPLEX_FORM.
int g_simplex_form = -1;
int simplex_form()
{
    std::lock_guard<std::mutex> lk(g_mutex);
    if (g_simplex_form < 0) {
        const char* ev = std::getenv("NK_SIMPLEX_FORM");
        const int v = ev ? std::atoi(ev) : 0;
        g_simplex_form = (v >= 0 && v <= 2) ? v : 0;
    }
    return g_simplex_form;
}

// SM count of the CURRENT device (cached per device ordinal)
thread_local int g_num_sms = 0;
nk_status ensure_device()
{
    enum { kMaxDevices = 64 };
    static int sms[kMaxDevices] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice (no CUDA device: libnk has no CPU fallback)");
    if (dev < 0 || dev >= kMaxDevices) return fail(NK_ERR_UNSUPPORTED, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lk(g_mutex);
    if (sms[dev] == 0) {
        int n = 0;
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
        sms[dev] = n;
    }
    g_num_sms = sms[dev];
    return NK_OK;
}

} // namespace

struct nk_basis {
    nk::HostTables t;
    const nk::InstInfo* inst = nullptr;
    // (shape, P, Q) outside the prebuilt table: the kernels are specialised at run time (csrc/nk_jit.cu); `inst` then
    // points at own_inst, which carries the interleave widths but no launch functions
    bool jit = false;
    nk::JitInfo jinfo;
    nk::InstInfo own_inst;
    std::vector<double> tabs_flat; // DenseTabs<nm,Q> in declaration order
    std::vector<double> sx_flat;   // SimplexTabs in declaration order (simplices only)
    std::vector<double> kron[3];   // hex: the 1-D matrices M, K, C of the coefficient-space forms (NK_TAB_KRON)
    // reference-matrix form of the affine operators (nk_dense.cuh): built on first use, under `mu`
    mutable std::mutex mu;
    mutable std::vector<double> refmat;                              // K7[7][Nm][Nm]
    mutable double* d_frag[nk::DENSE_KINDS] = {nullptr, nullptr, nullptr}; // fragment-ordered device copies per operator kind
    mutable int frag_dev = -1;                                       // device ordinal the copies live on
};

namespace {
const std::vector<double>& reference_matrices(const nk_basis* b)
{
    std::lock_guard<std::mutex> lk(b->mu);
    if (b->refmat.empty()) nk::build_reference_matrices(b->t, b->refmat);
    return b->refmat;
}
// device copy of the fragment-ordered matrices of one operator kind (lazily, once per basis)
nk_status dense_fragments(const nk_basis* b, int kind, const double** out)
{
    const std::vector<double>& K7 = reference_matrices(b);
    std::lock_guard<std::mutex> lk(b->mu);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (b->frag_dev >= 0 && b->frag_dev != dev)
        return fail(NK_ERR_UNSUPPORTED, "this basis already holds device tables on another GPU: create one nk_basis per device");
    if (!b->d_frag[kind]) {
        const int c0 = nk::dense_c0(kind), nc = nk::dense_nc(kind);
        std::vector<double> frag(nk::dense_pack_size(b->t.Nm, nc));
        nk::dense_pack(K7.data(), b->t.Nm, c0, nc, frag.data());
        double* d = nullptr;
        e = cudaMalloc(&d, frag.size() * sizeof(double));
        if (e != cudaSuccess) { g_err = "reference matrices: cudaMalloc failed"; return NK_ERR_ALLOC; }
        e = cudaMemcpy(d, frag.data(), frag.size() * sizeof(double), cudaMemcpyHostToDevice);   // synchronous, once per basis
        if (e != cudaSuccess) { cudaFree(d); return cuda_fail(e, "reference matrices: upload"); }
        b->d_frag[kind] = d;
        b->frag_dev = dev;
    }
    *out = b->d_frag[kind];
    return NK_OK;
}
// does this (basis, geometry, operator) take the reference-matrix kernel?
//   form 1: never.  form 2: every affine block (mode counts outside the prebuilt table are specialised at run time by
//   NVRTC, csrc/nk_jit.cu; a failure there surfaces at launch).  form 0: where it is the faster kernel -- tets of every
//   order, prisms up to P = 3 (92 / 84 / 54 against 34 / 43 / 41 GDoF/s for the chain; at P = 4 the chain wins) and
//   trilinear hexes (14 DMMA per 8 elements against the Kronecker form's 272 FMA in 64-thread blocks with three
//   barriers); hexes of order >= 2 keep the Kronecker forms (nm^4 against nm^6 work).  profiles/r2_notes.md
bool use_dense(const nk_basis* b, int deformed, int op, nk_status* st)
{
    *st = NK_OK;
    if (deformed) return false;
    if (op != nk::OP_MASS && op != nk::OP_LAP && op != nk::OP_HELM && op != nk::OP_HELMF) return false;
    const int form = simplex_form();
    if (form == 1) return false;
    if (form == 2) return true;
    const int shape = b->t.shape, P = b->t.P;
    const bool faster = shape == nk::TET || (shape == nk::PRISM && P <= 3) || (shape == nk::HEX && P == 1);
    // tets outside the prebuilt table (P = 9, run-time specialised basis): the reference-matrix kernel is specialised too
    return faster && (nk::dense_supported(b->t.Nm) || (b->jit && shape == nk::TET));
}
} // namespace

struct nk_geom {
    const nk_basis* b = nullptr;
    int64_t nelem = 0, ngroups = 0;
    int deformed = 0, E = 1;
    double* d_metric = nullptr; // [group][7][npt][E]
    double* d_factor = nullptr; // [group][10][npt][E]
    // nk_helmholtz_apply_host: device staging buffers and the copy-in / copy-out pipeline
    double* d_stage_in = nullptr;
    double* d_stage_out = nullptr;
    enum { kChunks = 16 };
    std::mutex host_mu;          // nk_helmholtz_apply_host is serialised per geometry (one set of staging buffers)
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_done = nullptr, ev_in[kChunks] = {}, ev_k[kChunks] = {};
};

// =========================== basis ===========================
extern "C" nk_status nk_basis_create(nk_shape shape, int P, int Q, nk_basis** out)
{
    if (!out) return fail(NK_ERR_INVALID_ARG, "nk_basis_create: out is NULL");
    *out = nullptr;
    if ((int)shape < 0 || (int)shape > 2 || P < 1 || Q < 2) return fail(NK_ERR_INVALID_ARG, "nk_basis_create: bad shape/P/Q");
    InstGetter get = (Q == P + 2) ? inst_getter((int)shape, P) : nullptr;
    nk::JitInfo jinfo;
    if (!get) {
        // outside the prebuilt table (Q = P+2; hex P <= 10, tet / prism P <= 8): specialised at run time on first use
        std::string why;
        if (!nk::sumfac_jit_info((int)shape, P, Q, &jinfo, &why)) {
            char buf[128];
            snprintf(buf, sizeof buf, "nk_basis_create: (shape=%d,P=%d,Q=%d) is neither prebuilt nor specialisable: ", (int)shape, P, Q);
            return fail(NK_ERR_UNSUPPORTED, buf + why);
        }
    }
    nk_basis* b = new (std::nothrow) nk_basis;
    if (!b) return fail(NK_ERR_ALLOC, "nk_basis_create: out of memory");
    if (!nk::build_host_tables((int)shape, P, Q, b->t)) {
        delete b;
        return fail(NK_ERR_INVALID_ARG, "nk_basis_create: table construction failed");
    }
    if (get) {
        b->inst = get();
    } else {
        b->jit = true;
        b->jinfo = jinfo;
        nk::InstInfo& oi = b->own_inst;
        std::memset(&oi, 0, sizeof oi);
        oi.shape = (int)shape; oi.P = P; oi.Q = Q;
        for (int d = 0; d < 2; ++d) {
            oi.E[d] = jinfo.E[d];
            oi.threads[d] = jinfo.op[d][nk::OP_HELM].threads;
            oi.blocks_per_sm_hint[d] = jinfo.op[d][nk::OP_HELM].minb;
            oi.smem_grid[d] = jinfo.op[d][nk::OP_HELM].smem;
        }
        for (int k = 0; k < nk::OP_COUNT; ++k) oi.E_op_affine[k] = jinfo.op[0][k].E;
        b->inst = &oi;
    }
    const nk::HostTables& t = b->t;
    const int nm = t.nm;
    // DenseTabs: Ba[3][Q*nm], BaT[3][nm*Q], KM[3][4][nm*nm], D[3][Q*Q], DT[3][Q*Q], w[3][Q], aux[7][Q]
    std::vector<double>& f = b->tabs_flat;
    for (int d = 0; d < 3; ++d) f.insert(f.end(), t.psi[0].begin(), t.psi[0].end()); // psi^a at GLL, [i][p]
    for (int d = 0; d < 3; ++d)
        for (int p = 0; p < nm; ++p)
            for (int i = 0; i < Q; ++i) f.push_back(t.psi[0][i * nm + p]); // BaT
    {   // KM[stage][which]: stage 0 acts on index r (direction 3), 1 on q (direction 2), 2 on p (direction 1);
        // which = M, K, C, C^T built from psi^a, D and w of that direction (used on hexes only: all alike there)
        std::vector<double> DB((size_t)Q * nm);
        for (int st = 0; st < 3; ++st) {
            const int dir = 2 - st;
            for (int i = 0; i < Q; ++i)
                for (int p = 0; p < nm; ++p) {
                    double s = 0.0;
                    for (int r = 0; r < Q; ++r) s += t.D[dir][i * Q + r] * t.psi[0][r * nm + p];
                    DB[(size_t)i * nm + p] = s;
                }
            for (int which = 0; which < 4; ++which) {
                if (shape != NK_HEX) { f.push_back(0.0); continue; }   // DenseTabs<.,.,false>: one dummy entry
                for (int pp = 0; pp < nm; ++pp)
                    for (int p = 0; p < nm; ++p) {
                        double m = 0.0;
                        for (int i = 0; i < Q; ++i) {
                            const double w = t.w[dir][i], b1 = t.psi[0][i * nm + pp], b0 = t.psi[0][i * nm + p];
                            const double d1 = DB[(size_t)i * nm + pp], d0 = DB[(size_t)i * nm + p];
                            m += w * (which == 0 ? b1 * b0 : which == 1 ? d1 * d0 : which == 2 ? b1 * d0 : d1 * b0);
                        }
                        f.push_back(m);
                        if (st == 2 && which < 3) b->kron[which].push_back(m);
                    }
            }
        }
    }
    for (int d = 0; d < 3; ++d) f.insert(f.end(), t.D[d].begin(), t.D[d].end());
    for (int d = 0; d < 3; ++d)
        for (int r = 0; r < Q; ++r)
            for (int i = 0; i < Q; ++i) f.push_back(t.D[d][i * Q + r]); // DT
    for (int d = 0; d < 3; ++d) f.insert(f.end(), t.w[d].begin(), t.w[d].end());
    for (int i = 0; i < Q; ++i) f.push_back(1.0 + t.z[0][i]);
    for (int i = 0; i < Q; ++i) f.push_back(1.0 + t.z[1][i]);
    for (int i = 0; i < Q; ++i) f.push_back(shape == NK_TET ? 1.0 / (1.0 - t.z[1][i]) : 0.0);
    for (int i = 0; i < Q; ++i) f.push_back(shape != NK_HEX ? 1.0 / (1.0 - t.z[2][i]) : 0.0);
    for (int i = 0; i < Q; ++i) f.push_back(shape != NK_HEX ? (1.0 - t.z[2][i]) : 0.0);
    for (int i = 0; i < Q; ++i) {
        const double s = shape != NK_HEX ? 1.0 / (1.0 - t.z[2][i]) : 0.0;
        f.push_back(shape == NK_TET ? t.w[2][i] * s * s : t.w[2][i] * s);
    }
    for (int i = 0; i < Q; ++i) f.push_back(shape != NK_HEX ? t.w[2][i] / (1.0 - t.z[2][i]) : 0.0);
    // SimplexTabs: b3f, b3a (psi^b at the direction-3 points), b2f, b2a (direction 2; tet only); where two copies do not
    // fit the kernel-parameter space (k_sx_dup: tets / prisms at P = 10) the adjoint copies shrink to one unused entry
    if (shape != NK_HEX) {
        std::vector<double>& x = b->sx_flat;
        const size_t n = (size_t)t.npair * Q;
        const bool dup = nk::k_sx_dup((int)shape, nm, Q);
        x.insert(x.end(), t.tab3.begin(), t.tab3.end());
        if (dup) x.insert(x.end(), t.tab3.begin(), t.tab3.end()); else x.push_back(0.0);
        for (int c = 0; c < 2; ++c) {
            if (c == 1 && !dup) { x.push_back(0.0); break; }
            if (shape == NK_TET) x.insert(x.end(), t.tab2.begin(), t.tab2.end());
            else x.insert(x.end(), n, 0.0);
        }
    }
    *out = b;
    return NK_OK;
}

extern "C" nk_status nk_basis_destroy(nk_basis* b)
{
    if (!b) return NK_OK;
    for (int k = 0; k < nk::DENSE_KINDS; ++k)
        if (b->d_frag[k]) cudaFree(b->d_frag[k]);
    delete b;
    return NK_OK;
}

extern "C" int nk_basis_num_modes(const nk_basis* b) { return b ? b->t.Nm : -1; }
extern "C" int nk_basis_num_points(const nk_basis* b) { return b ? b->t.Nq : -1; }
extern "C" int nk_basis_interleave(const nk_basis* b, int deformed) { return b ? b->inst->E[deformed ? 1 : 0] : -1; }

extern "C" nk_status nk_basis_get_table(const nk_basis* b, int which, int dir, double* host_out, size_t cap, size_t* count)
{
    if (!b || dir < 0 || dir > 2) return fail(NK_ERR_INVALID_ARG, "nk_basis_get_table: bad basis/dir");
    const std::vector<double>* v = nullptr;
    switch (which) {
    case NK_TAB_NODES: v = &b->t.z[dir]; break;
    case NK_TAB_WEIGHTS: v = &b->t.w[dir]; break;
    case NK_TAB_DERIV: v = &b->t.D[dir]; break;
    case NK_TAB_PSI: v = &b->t.psi[dir]; break;
    case NK_TAB_KRON:
        if (b->t.shape != nk::HEX) return fail(NK_ERR_INVALID_ARG, "nk_basis_get_table: NK_TAB_KRON exists on hexes only");
        v = &b->kron[dir];
        break;
    default: return fail(NK_ERR_INVALID_ARG, "nk_basis_get_table: unknown table");
    }
    if (count) *count = v->size();
    if (!host_out) return NK_OK;
    if (cap < v->size()) return fail(NK_ERR_INVALID_ARG, "nk_basis_get_table: capacity too small");
    std::memcpy(host_out, v->data(), v->size() * sizeof(double));
    return NK_OK;
}

extern "C" nk_status nk_basis_get_points(const nk_basis* b, double* xi_out, size_t cap)
{
    if (!b || !xi_out) return fail(NK_ERR_INVALID_ARG, "nk_basis_get_points: NULL argument");
    const nk::HostTables& t = b->t;
    const int Q = t.Q;
    if (cap < (size_t)3 * t.Nq) return fail(NK_ERR_INVALID_ARG, "nk_basis_get_points: capacity too small");
    for (int k = 0; k < Q; ++k)
        for (int j = 0; j < Q; ++j)
            for (int i = 0; i < Q; ++i) {
                const double e1 = t.z[0][i], e2 = t.z[1][j], e3 = t.z[2][k];
                double* x = xi_out + 3 * ((size_t)i + Q * (j + (size_t)Q * k));
                x[0] = e1; x[1] = e2; x[2] = e3;
                if (t.shape == nk::TET) {
                    x[0] = 0.25 * (1.0 + e1) * (1.0 - e2) * (1.0 - e3) - 1.0;
                    x[1] = 0.5 * (1.0 + e2) * (1.0 - e3) - 1.0;
                } else if (t.shape == nk::PRISM) {
                    x[0] = 0.5 * (1.0 + e1) * (1.0 - e3) - 1.0;
                }
            }
    return NK_OK;
}

extern "C" int nk_basis_mode_index(const nk_basis* b, int p, int q, int r)
{
    return b ? nk::mode_index(b->t.shape, b->t.nm, p, q, r) : -1;
}

// =========================== geometry ===========================
namespace {

struct RepackTabs {
    double z[3][12], w[3][12];
    int shape, Q;
};

// chain matrix of Eq. 23 (A17) folded into the user's dxi/dx:  A'[l][i] = sum_j C[j][l] A[j][i]
__device__ inline void fold_chain(int shape, const RepackTabs& rt, int i, int j, int k, double (&A)[9])
{
    if (shape == nk::K_TET) {
        const double r2 = 1.0 / (1.0 - rt.z[1][j]), r3 = 1.0 / (1.0 - rt.z[2][k]);
        const double c1 = 4.0 * r2 * r3, c2 = 2.0 * (1.0 + rt.z[0][i]) * r2 * r3, c3 = 2.0 * r3, c4 = (1.0 + rt.z[1][j]) * r3;
        for (int x = 0; x < 3; ++x) {
            const double a0 = A[0 + x], a1 = A[3 + x], a2 = A[6 + x];
            A[0 + x] = c1 * a0 + c2 * (a1 + a2);
            A[3 + x] = c3 * a1 + c4 * a2;
        }
    } else if (shape == nk::K_PRISM) {
        const double r3 = 1.0 / (1.0 - rt.z[2][k]);
        const double ca = 2.0 * r3, cb = (1.0 + rt.z[0][i]) * r3;
        for (int x = 0; x < 3; ++x) A[0 + x] = ca * A[0 + x] + cb * A[6 + x];
    }
}

// one thread per (group, point, e).  Deformed: quadrature weight and chain folded in.
// Affine: npt = 1, plain factors (weights and chain are applied inside the kernels).
__global__ void repack_kernel(const __grid_constant__ RepackTabs rt, const double* __restrict__ dxi_dx,
                              const double* __restrict__ detJ, long long nelem, long long ngroups, int E, int deformed,
                              double* __restrict__ metric, double* __restrict__ factor)
{
    const int Q = rt.Q;
    const long long npt = deformed ? (long long)Q * Q * Q : 1;
    const long long total = ngroups * npt * E;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int e = (int)(t % E);
        const long long n = (t / E) % npt, g = t / ((long long)E * npt);
        const long long elem = g * E + e;
        double A[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, wJ = 0.0;
        if (elem < nelem) {
            const double* ap = dxi_dx + (elem * npt + n) * 9;
            for (int c = 0; c < 9; ++c) A[c] = ap[c];
            wJ = detJ[elem * npt + n];
            if (deformed) {
                const int k = (int)(n / (Q * Q)), j = (int)((n / Q) % Q), i = (int)(n % Q);
                fold_chain(rt.shape, rt, i, j, k, A);
                wJ *= rt.w[0][i] * rt.w[1][j] * rt.w[2][k];
            }
        }
        double G[6];
        G[0] = wJ * (A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
        G[1] = wJ * (A[0] * A[3] + A[1] * A[4] + A[2] * A[5]);
        G[2] = wJ * (A[0] * A[6] + A[1] * A[7] + A[2] * A[8]);
        G[3] = wJ * (A[3] * A[3] + A[4] * A[4] + A[5] * A[5]);
        G[4] = wJ * (A[3] * A[6] + A[4] * A[7] + A[5] * A[8]);
        G[5] = wJ * (A[6] * A[6] + A[7] * A[7] + A[8] * A[8]);
        if (metric) {
            for (int c = 0; c < 6; ++c) metric[((g * 7 + c) * npt + n) * E + e] = G[c];
            metric[((g * 7 + 6) * npt + n) * E + e] = wJ;
        }
        if (factor) {
            for (int c = 0; c < 9; ++c) factor[((g * 10 + c) * npt + n) * E + e] = A[c];
            factor[((g * 10 + 9) * npt + n) * E + e] = wJ;
        }
    }
}

} // namespace

extern "C" nk_status nk_geom_upload(const nk_basis* b, int64_t nelem, int deformed, const double* dxi_dx,
                                    const double* detJ, int on_device, void* stream, nk_geom** out)
{
    return nk_geom_upload_streams(b, nelem, deformed, dxi_dx, detJ, on_device, NK_GEOM_METRIC | NK_GEOM_FACTORS, stream, out);
}

extern "C" nk_status nk_geom_upload_streams(const nk_basis* b, int64_t nelem, int deformed, const double* dxi_dx,
                                            const double* detJ, int on_device, unsigned streams, void* stream, nk_geom** out)
{
    if ((streams & (NK_GEOM_METRIC | NK_GEOM_FACTORS)) == 0 || (streams & ~(unsigned)(NK_GEOM_METRIC | NK_GEOM_FACTORS)))
        return fail(NK_ERR_INVALID_ARG, "nk_geom_upload_streams: streams must be a combination of NK_GEOM_METRIC and NK_GEOM_FACTORS");
    if (!out) return fail(NK_ERR_INVALID_ARG, "nk_geom_upload: out is NULL");
    *out = nullptr;
    if (!b || nelem < 0 || (nelem > 0 && (!dxi_dx || !detJ))) return fail(NK_ERR_INVALID_ARG, "nk_geom_upload: bad arguments");
    nk_status st = ensure_device();
    if (st != NK_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    nk_geom* g = new (std::nothrow) nk_geom;
    if (!g) return fail(NK_ERR_ALLOC, "nk_geom_upload: out of memory");
    g->b = b;
    g->nelem = nelem;
    g->deformed = deformed ? 1 : 0;
    g->E = b->inst->E[g->deformed];
    g->ngroups = (nelem + g->E - 1) / g->E;
    *out = g;
    if (nelem == 0) return NK_OK;
    const long long npt = g->deformed ? b->t.Nq : 1;
    const size_t slots = (size_t)g->ngroups * npt * g->E;
    cudaError_t e = cudaSuccess;
    if (streams & NK_GEOM_METRIC) e = cudaMalloc(&g->d_metric, slots * 7 * sizeof(double));
    if (e == cudaSuccess && (streams & NK_GEOM_FACTORS)) e = cudaMalloc(&g->d_factor, slots * 10 * sizeof(double));
    if (e != cudaSuccess) {
        nk_geom_destroy(g);
        *out = nullptr;
        g_err = std::string("nk_geom_upload: cudaMalloc: ") + cudaGetErrorString(e);
        return NK_ERR_ALLOC;
    }
    const double *dA = dxi_dx, *dJ = detJ;
    double *tA = nullptr, *tJ = nullptr;
    if (!on_device) {
        const size_t nA = (size_t)nelem * npt * 9, nJ = (size_t)nelem * npt;
        e = cudaMalloc(&tA, nA * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc(&tJ, nJ * sizeof(double));
        if (e == cudaSuccess) e = cudaMemcpyAsync(tA, dxi_dx, nA * sizeof(double), cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(tJ, detJ, nJ * sizeof(double), cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) {
            cudaFree(tA); cudaFree(tJ);
            nk_geom_destroy(g);
            *out = nullptr;
            return cuda_fail(e, "nk_geom_upload: staging copy");
        }
        dA = tA;
        dJ = tJ;
    }
    RepackTabs rt;
    std::memset(&rt, 0, sizeof rt);
    rt.shape = b->t.shape;
    rt.Q = b->t.Q;
    for (int d = 0; d < 3; ++d)
        for (int i = 0; i < b->t.Q; ++i) {
            rt.z[d][i] = b->t.z[d][i];
            rt.w[d][i] = b->t.w[d][i];
        }
    const int threads = 256;
    long long blocks = ((long long)slots + threads - 1) / threads;
    if (blocks > 148LL * 32) blocks = 148LL * 32;
    repack_kernel<<<(int)blocks, threads, 0, s>>>(rt, dA, dJ, nelem, g->ngroups, g->E, g->deformed, g->d_metric, g->d_factor);
    e = cudaGetLastError();
    { std::lock_guard<std::mutex> lk(g_mutex); ++g_launches; }
    if (!on_device) {
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        cudaFree(tA);
        cudaFree(tJ);
    }
    if (e != cudaSuccess) {
        nk_geom_destroy(g);
        *out = nullptr;
        return cuda_fail(e, "nk_geom_upload: repack");
    }
    return NK_OK;
}

extern "C" nk_status nk_geom_destroy(nk_geom* g)
{
    if (!g) return NK_OK;
    if (g->d_metric) cudaFree(g->d_metric);
    if (g->d_factor) cudaFree(g->d_factor);
    if (g->d_stage_in) cudaFree(g->d_stage_in);
    if (g->d_stage_out) cudaFree(g->d_stage_out);
    if (g->s_in) cudaStreamDestroy(g->s_in);
    if (g->s_out) cudaStreamDestroy(g->s_out);
    if (g->ev_start) cudaEventDestroy(g->ev_start);
    if (g->ev_done) cudaEventDestroy(g->ev_done);
    for (int c = 0; c < nk_geom::kChunks; ++c) {
        if (g->ev_in[c]) cudaEventDestroy(g->ev_in[c]);
        if (g->ev_k[c]) cudaEventDestroy(g->ev_k[c]);
    }
    delete g;
    return NK_OK;
}

extern "C" int64_t nk_geom_num_elements(const nk_geom* g) { return g ? g->nelem : -1; }

// =========================== operators ===========================
namespace {

nk_status run_op(int op, const char* name, const nk_basis* b, const nk_geom* g, int64_t nelem, const double* in0,
                 const double* in1, const double* in2, double* out0, double* out1, double* out2, double lambda,
                 void* stream, int nfields = 1, const double* const* fin = nullptr, double* const* fout = nullptr,
                 int64_t group0 = 0, int64_t group_count = -1)
{
    if (!b) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": basis is NULL");
    if (op != nk::OP_BWD) {
        if (!g) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": geom is NULL");
        if (g->b != b && (g->b->t.shape != b->t.shape || g->b->t.P != b->t.P || g->b->t.Q != b->t.Q))
            return fail(NK_ERR_SHAPE_MISMATCH, std::string(name) + ": geom was uploaded for another basis");
        nelem = g->nelem;
    }
    if (nelem < 0) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": nelem < 0");
    if (nelem == 0) return NK_OK;
    const bool need_in0 = (op != nk::OP_IPDERIV);
    if ((need_in0 && !in0) || (op != nk::OP_PHYSDERIV && !out0))
        return fail(NK_ERR_INVALID_ARG, std::string(name) + ": NULL field pointer");
    if (in0 && (in0 == out0)) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": in and out alias");
    if (fin) {
        for (int f = 0; f < nfields; ++f) {
            if (!fin[f] || !fout[f]) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": NULL field pointer");
            for (int h = 0; h < nfields; ++h)
                if (fin[f] == fout[h]) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": in and out alias");
            for (int h = 0; h < f; ++h)
                if (fout[f] == fout[h]) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": two fields share an output");
        }
    }
    nk_status st = ensure_device();
    if (st != NK_OK) return st;
    if (g && use_dense(b, g->deformed, op, &st)) {
        // affine simplex mass / Laplacian / Helmholtz in coefficient space on the FP64 tensor cores (nk_dense.cuh);
        // group0 / group_count are in tiles of 8 elements here (dense_tile_elems)
        if (!g->d_metric) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": this geometry was uploaded without NK_GEOM_METRIC");
        const int kind = op == nk::OP_MASS ? nk::DENSE_MASS : op == nk::OP_LAP ? nk::DENSE_LAP : nk::DENSE_HELM;
        nk::DenseArgs d;
        st = dense_fragments(b, kind, &d.bfrag);
        if (st != NK_OK) return st;
        d.geom = g->d_metric;
        d.EG = g->E;
        d.EGshift = 0;
        while ((1 << d.EGshift) < g->E) ++d.EGshift;
        if ((1 << d.EGshift) != g->E) return fail(NK_ERR_UNSUPPORTED, std::string(name) + ": interleave width is not a power of two");
        d.nfields = fin ? nfields : 1;
        for (int f = 0; f < nk::DENSE_MAX_FIELDS; ++f) {
            d.in[f] = (fin && f < nfields) ? fin[f] : in0;
            d.out[f] = (fout && f < nfields) ? fout[f] : out0;
        }
        d.e0 = group0 * 8;
        d.e1 = group_count < 0 ? nelem : std::min<int64_t>(nelem, (group0 + group_count) * 8);
        if (d.e0 < 0 || d.e0 > nelem) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": bad tile range");
        d.scale6 = (kind == nk::DENSE_MASS) ? 1.0 : lambda;
        int launched = 0;
        if (nk::dense_supported(b->t.Nm)) {
            cudaError_t e = nk::dense_launch(b->t.Nm, kind, d, (cudaStream_t)stream, &launched);
            if (e != cudaSuccess) return cuda_fail(e, name);
        } else {
            // mode count outside the prebuilt table: NVRTC specialisation of the same kernel source, cached
            std::string why;
            if (!nk::dense_jit_launch(b->t.Nm, kind, d, (cudaStream_t)stream, &launched, &why))
                return fail(NK_ERR_UNSUPPORTED, std::string(name) + ": no reference-matrix kernel for this (shape, P) and run-time "
                                                                    "specialisation failed: " + why);
        }
        if (launched) { std::lock_guard<std::mutex> lk(g_mutex); ++g_launches; }
        return NK_OK;
    }
    if (st != NK_OK) return st;
    const int E = (g && g->deformed) ? b->inst->E[1] : b->inst->E_op_affine[op];
    nk::KArgs a;
    a.in[0] = in0; a.in[1] = in1; a.in[2] = in2;
    a.out[0] = out0; a.out[1] = out1; a.out[2] = out2;
    for (int f = 0; f < nk::K_MAX_FIELDS; ++f) {
        a.fin[f] = (fin && f < nfields) ? fin[f] : in0;
        a.fout[f] = (fout && f < nfields) ? fout[f] : out0;
    }
    a.nfields = fin ? nfields : 1;
    a.geom = nullptr;
    int def = 0;
    if (g) {
        def = g->deformed;
        a.geom = (op == nk::OP_PHYSDERIV || op == nk::OP_IPDERIV) ? g->d_factor : g->d_metric;
        if (!a.geom && g->nelem > 0)
            return fail(NK_ERR_INVALID_ARG, std::string(name) + ": this geometry was uploaded without the stream the operator reads "
                                                                "(NK_GEOM_METRIC / NK_GEOM_FACTORS)");
    }
    a.lambda = lambda;
    a.nelem = nelem;
    const int64_t ngroups = (nelem + E - 1) / E;
    if (ngroups > 0x7fffffffLL) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": too many elements");
    a.ngroups = (int)ngroups;
    a.g0 = (int)group0;
    a.grid_groups = (int)(group_count < 0 ? ngroups : group_count);
    if (a.g0 < 0 || a.g0 + (int64_t)a.grid_groups > ngroups) return fail(NK_ERR_INVALID_ARG, std::string(name) + ": bad group range");
    if (b->jit) {
        std::string why;
        if (!nk::sumfac_jit_launch(b->jinfo, def, op, b->tabs_flat.data(), b->sx_flat.data(), a, g_num_sms, (cudaStream_t)stream, &why))
            return fail(NK_ERR_UNSUPPORTED, std::string(name) + ": run-time specialisation failed: " + why);
        { std::lock_guard<std::mutex> lk(g_mutex); ++g_launches; }
        return NK_OK;
    }
    cudaError_t e = b->inst->fn[def][op](b->tabs_flat.data(), b->sx_flat.data(), a, g_num_sms, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, name);
    { std::lock_guard<std::mutex> lk(g_mutex); ++g_launches; }
    return NK_OK;
}

} // namespace

extern "C" nk_status nk_bwdtrans(const nk_basis* b, int64_t nelem, const double* coeffs, double* phys, void* stream)
{
    return run_op(nk::OP_BWD, "nk_bwdtrans", b, nullptr, nelem, coeffs, nullptr, nullptr, phys, nullptr, nullptr, 0.0, stream);
}
extern "C" nk_status nk_iprod(const nk_basis* b, const nk_geom* g, const double* phys, double* coeffs, void* stream)
{
    return run_op(nk::OP_IPROD, "nk_iprod", b, g, 0, phys, nullptr, nullptr, coeffs, nullptr, nullptr, 0.0, stream);
}
extern "C" nk_status nk_physderiv(const nk_basis* b, const nk_geom* g, const double* phys, double* d0, double* d1,
                                  double* d2, void* stream)
{
    return run_op(nk::OP_PHYSDERIV, "nk_physderiv", b, g, 0, phys, nullptr, nullptr, d0, d1, d2, 0.0, stream);
}
extern "C" nk_status nk_iprod_deriv(const nk_basis* b, const nk_geom* g, const double* g0, const double* g1,
                                    const double* g2, double* coeffs, void* stream)
{
    return run_op(nk::OP_IPDERIV, "nk_iprod_deriv", b, g, 0, g0, g1, g2, coeffs, nullptr, nullptr, 0.0, stream);
}
extern "C" nk_status nk_mass_apply(const nk_basis* b, const nk_geom* g, const double* in, double* out, void* stream)
{
    return run_op(nk::OP_MASS, "nk_mass_apply", b, g, 0, in, nullptr, nullptr, out, nullptr, nullptr, 0.0, stream);
}
extern "C" nk_status nk_laplacian_apply(const nk_basis* b, const nk_geom* g, const double* in, double* out, void* stream)
{
    return run_op(nk::OP_LAP, "nk_laplacian_apply", b, g, 0, in, nullptr, nullptr, out, nullptr, nullptr, 0.0, stream);
}
extern "C" nk_status nk_helmholtz_apply(const nk_basis* b, const nk_geom* g, double lambda, const double* in,
                                        double* out, void* stream)
{
    return run_op(nk::OP_HELM, "nk_helmholtz_apply", b, g, 0, in, nullptr, nullptr, out, nullptr, nullptr, lambda, stream);
}

extern "C" nk_status nk_helmholtz_apply_fields(const nk_basis* b, const nk_geom* g, double lambda, int nfields,
                                               const double* const* in, double* const* out, void* stream)
{
    if (nfields < 1 || nfields > nk::K_MAX_FIELDS || !in || !out)
        return fail(NK_ERR_INVALID_ARG, "nk_helmholtz_apply_fields: nfields must be 1..8 and the pointer arrays non-NULL");
    return run_op(nfields > 1 ? nk::OP_HELMF : nk::OP_HELM, "nk_helmholtz_apply_fields", b, g, 0, in[0], nullptr, nullptr, out[0], nullptr, nullptr, lambda,
                  stream, nfields, in, out);
}

namespace {
// side streams of nk_helmholtz_apply_blocks: block i > 0 runs on side stream (i-1) % kSide, forked from and joined to the
// caller's stream by events, so that the tail of one block's kernel overlaps the head of the next one's
enum { kSide = 3, kMaxDev = 64 };
struct SidePool {
    cudaStream_t s[kSide] = {};
    cudaEvent_t fork = nullptr, join[kSide] = {};
    bool ok = false;
};
SidePool g_side[kMaxDev];
std::mutex g_side_mutex;     // one nk_helmholtz_apply_blocks at a time per process (the pool is shared)
} // namespace

extern "C" nk_status nk_helmholtz_apply_blocks(int nblocks, const nk_block* blocks, double lambda, void* stream)
{
    if (nblocks < 0 || (nblocks > 0 && !blocks)) return fail(NK_ERR_INVALID_ARG, "nk_helmholtz_apply_blocks: bad arguments");
    if (nblocks <= 1) return nblocks == 0 ? NK_OK : nk_helmholtz_apply(blocks[0].basis, blocks[0].geom, lambda, blocks[0].in, blocks[0].out, stream);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice (no CUDA device: libnk has no CPU fallback)");
    if (dev < 0 || dev >= kMaxDev) return fail(NK_ERR_UNSUPPORTED, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lk(g_side_mutex);
    SidePool& sp = g_side[dev];
    if (!sp.ok) {
        for (int i = 0; i < kSide && e == cudaSuccess; ++i) {
            e = cudaStreamCreateWithFlags(&sp.s[i], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&sp.join[i], cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&sp.fork, cudaEventDisableTiming);
        if (e != cudaSuccess) return cuda_fail(e, "nk_helmholtz_apply_blocks: stream / event creation");
        sp.ok = true;
    }
    cudaStream_t s = (cudaStream_t)stream;
    e = cudaEventRecord(sp.fork, s);
    if (e != cudaSuccess) return cuda_fail(e, "nk_helmholtz_apply_blocks: fork");
    nk_status st = NK_OK;
    bool used[kSide] = {};
    for (int i = 0; i < nblocks && st == NK_OK; ++i) {
        cudaStream_t si = s;
        if (i > 0) {
            const int k = (i - 1) % kSide;
            si = sp.s[k];
            if (!used[k]) {
                e = cudaStreamWaitEvent(si, sp.fork, 0);
                if (e != cudaSuccess) { st = cuda_fail(e, "nk_helmholtz_apply_blocks: fork"); break; }
                used[k] = true;
            }
        }
        st = nk_helmholtz_apply(blocks[i].basis, blocks[i].geom, lambda, blocks[i].in, blocks[i].out, (void*)si);
    }
    // join whatever was forked, also on error (the caller's stream must not run ahead of work already enqueued)
    for (int k = 0; k < kSide; ++k) {
        if (!used[k]) continue;
        e = cudaEventRecord(sp.join[k], sp.s[k]);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, sp.join[k], 0);
        if (e != cudaSuccess && st == NK_OK) st = cuda_fail(e, "nk_helmholtz_apply_blocks: join");
    }
    return st;
}

extern "C" nk_status nk_helmholtz_apply_host(const nk_basis* b, const nk_geom* gc, double lambda, const double* host_in,
                                             double* host_out, void* stream)
{
    if (!b || !gc || !host_in || !host_out) return fail(NK_ERR_INVALID_ARG, "nk_helmholtz_apply_host: NULL argument");
    nk_geom* g = const_cast<nk_geom*>(gc);   // the staging buffers and pipeline objects live in the geometry handle
    // validate BEFORE anything is allocated: the buffers are sized from the geometry's own basis
    if (g->b != b && (g->b->t.shape != b->t.shape || g->b->t.P != b->t.P || g->b->t.Q != b->t.Q))
        return fail(NK_ERR_SHAPE_MISMATCH, "nk_helmholtz_apply_host: geom was uploaded for another basis");
    if (g->nelem == 0) return NK_OK;
    if (!g->d_metric) return fail(NK_ERR_INVALID_ARG, "nk_helmholtz_apply_host: this geometry was uploaded without NK_GEOM_METRIC");
    nk_status dst = ensure_device();
    if (dst != NK_OK) return dst;
    const bool dense = use_dense(b, g->deformed, nk::OP_HELM, &dst);
    if (dst != NK_OK) return dst;
    std::lock_guard<std::mutex> host_lock(g->host_mu);   // one caller at a time per geometry (documented in nk.h)
    const int Nm = g->b->t.Nm;
    const size_t bytes = (size_t)g->nelem * Nm * sizeof(double);
    cudaError_t e = cudaSuccess;
    if (!g->d_stage_in || !g->d_stage_out) {
        // both buffers or neither
        double *bi = nullptr, *bo = nullptr;
        e = cudaMalloc(&bi, bytes);
        if (e == cudaSuccess) e = cudaMalloc(&bo, bytes);
        if (e != cudaSuccess) {
            if (bi) cudaFree(bi);
            if (bo) cudaFree(bo);
            cudaGetLastError();
            g_err = "nk_helmholtz_apply_host: cudaMalloc of the staging buffers failed";
            return NK_ERR_ALLOC;
        }
        g->d_stage_in = bi;
        g->d_stage_out = bo;
    }
    cudaStream_t s = (cudaStream_t)stream;
    // Pipeline over chunks: H2D on s_in, the fused kernel on the caller's stream, D2H on s_out, chained by events, so
    // that the copy-in of chunk c+1 and the copy-out of chunk c-1 (PCIe is full duplex) overlap the kernel of chunk c.
    if (!g->s_in) {
        e = cudaStreamCreateWithFlags(&g->s_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&g->s_out, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g->ev_start, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g->ev_done, cudaEventDisableTiming);
        for (int c = 0; c < nk_geom::kChunks && e == cudaSuccess; ++c) {
            e = cudaEventCreateWithFlags(&g->ev_in[c], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g->ev_k[c], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) {
            // leave the handle in the "nothing created" state: the next call starts over
            if (g->s_in) { cudaStreamDestroy(g->s_in); g->s_in = nullptr; }
            if (g->s_out) { cudaStreamDestroy(g->s_out); g->s_out = nullptr; }
            if (g->ev_start) { cudaEventDestroy(g->ev_start); g->ev_start = nullptr; }
            if (g->ev_done) { cudaEventDestroy(g->ev_done); g->ev_done = nullptr; }
            for (int c = 0; c < nk_geom::kChunks; ++c) {
                if (g->ev_in[c]) { cudaEventDestroy(g->ev_in[c]); g->ev_in[c] = nullptr; }
                if (g->ev_k[c]) { cudaEventDestroy(g->ev_k[c]); g->ev_k[c] = nullptr; }
            }
            return cuda_fail(e, "nk_helmholtz_apply_host: stream / event creation");
        }
    }
    // chunk unit: groups of the kernel (not of the stream), or tiles of 8 elements of the reference-matrix kernel
    const int Eop = dense ? 8 : g->deformed ? b->inst->E[1] : b->inst->E_op_affine[nk::OP_HELM];
    const int64_t ngroups_op = (g->nelem + Eop - 1) / Eop;
    // chunk size: NK_HOST_CHUNK_MB (default 8 MB; B200 sweep in profiles/r2_notes.md): smaller chunks pay the per-copy
    // latency more often than the extra overlap gains
    static const long long chunk_mb = [] {
        const char* ev = std::getenv("NK_HOST_CHUNK_MB");
        const long long v = ev ? std::atoll(ev) : 8;
        return v < 1 ? 1LL : v;
    }();
    int nchunks = (int)std::min<int64_t>(nk_geom::kChunks, std::max<int64_t>(1, (int64_t)(bytes / ((size_t)chunk_mb << 20))));
    const int64_t per = (ngroups_op + nchunks - 1) / nchunks;
    const size_t elem_bytes = (size_t)Nm * sizeof(double);
    nk_status st = NK_OK;
    const char* what = nullptr;
    e = cudaEventRecord(g->ev_start, s);                  // order after the caller's earlier work on `stream`
    if (e == cudaSuccess) e = cudaStreamWaitEvent(g->s_in, g->ev_start, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(g->s_out, g->ev_start, 0);
    if (e != cudaSuccess) what = "nk_helmholtz_apply_host: pipeline start";
    for (int c = 0; c < nchunks && e == cudaSuccess && st == NK_OK; ++c) {
        const int64_t g0 = c * per, g1 = std::min<int64_t>(ngroups_op, g0 + per);
        if (g0 >= g1) break;
        const int64_t e0 = g0 * Eop, e1 = std::min<int64_t>(g->nelem, g1 * Eop);
        const size_t off = (size_t)e0 * Nm, nb = (size_t)(e1 - e0) * elem_bytes;
        e = cudaMemcpyAsync(g->d_stage_in + off, host_in + off, nb, cudaMemcpyHostToDevice, g->s_in);
        if (e == cudaSuccess) e = cudaEventRecord(g->ev_in[c], g->s_in);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, g->ev_in[c], 0);
        if (e != cudaSuccess) { what = "nk_helmholtz_apply_host: H2D"; break; }
        st = run_op(nk::OP_HELM, "nk_helmholtz_apply_host", b, g, 0, g->d_stage_in, nullptr, nullptr, g->d_stage_out,
                    nullptr, nullptr, lambda, stream, 1, nullptr, nullptr, g0, g1 - g0);
        if (st != NK_OK) break;
        e = cudaEventRecord(g->ev_k[c], s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(g->s_out, g->ev_k[c], 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync(host_out + off, g->d_stage_out + off, nb, cudaMemcpyDeviceToHost, g->s_out);
        if (e != cudaSuccess) { what = "nk_helmholtz_apply_host: D2H"; break; }
    }
    if (e != cudaSuccess || st != NK_OK) {
        // drain everything that was enqueued: no copy into host_out may still be in flight when we return
        const std::string keep = g_err;
        cudaStreamSynchronize(g->s_in);
        cudaStreamSynchronize(s);
        cudaStreamSynchronize(g->s_out);
        if (st != NK_OK) { g_err = keep; return st; }
        return cuda_fail(e, what ? what : "nk_helmholtz_apply_host");
    }
    e = cudaEventRecord(g->ev_done, g->s_out);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s, g->ev_done, 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) {
        cudaStreamSynchronize(g->s_in);
        cudaStreamSynchronize(g->s_out);
        return cuda_fail(e, "nk_helmholtz_apply_host: synchronise");
    }
    return NK_OK;
}

// =========================== options ===========================
extern "C" nk_status nk_set_affine_simplex_form(int form)
{
    if (form < 0 || form > 2) return fail(NK_ERR_INVALID_ARG, "nk_set_affine_simplex_form: form must be 0 (auto), 1 (sum-factorised) or 2 (reference-matrix)");
    simplex_form();      // reads the environment default first
    std::lock_guard<std::mutex> lk(g_mutex);
    g_simplex_form = form;
    return NK_OK;
}
extern "C" int nk_get_affine_simplex_form(void) { return simplex_form(); }

extern "C" nk_status nk_basis_get_reference_matrix(const nk_basis* b, int c, double* host_out, size_t cap)
{
    if (!b || c < 0 || c > 6 || !host_out) return fail(NK_ERR_INVALID_ARG, "nk_basis_get_reference_matrix: bad arguments");
    const size_t n = (size_t)b->t.Nm * b->t.Nm;
    if (cap < n) return fail(NK_ERR_INVALID_ARG, "nk_basis_get_reference_matrix: capacity too small");
    const std::vector<double>& K7 = reference_matrices(b);
    std::memcpy(host_out, K7.data() + (size_t)c * n, n * sizeof(double));
    return NK_OK;
}

extern "C" nk_status nk_jit_compile_check(int nmodes, double* compile_ms, size_t* cubin_bytes)
{
    if (nmodes < 1 || nmodes > 1024) return fail(NK_ERR_INVALID_ARG, "nk_jit_compile_check: 1 <= nmodes <= 1024");
    std::string why;
    if (!nk::dense_jit_compile_check(nmodes, nk::DENSE_HELM, compile_ms, cubin_bytes, &why)) return fail(NK_ERR_UNSUPPORTED, why);
    return NK_OK;
}
extern "C" nk_status nk_jit_compile_check_kernel(nk_shape shape, int P, int Q, int deformed, int op, double* compile_ms, size_t* cubin_bytes)
{
    std::string why;
    if (!nk::sumfac_jit_compile_check((int)shape, P, Q, deformed, op, compile_ms, cubin_bytes, &why)) return fail(NK_ERR_UNSUPPORTED, why);
    return NK_OK;
}
extern "C" nk_status nk_jit_stats(int64_t* kernels, double* compile_ms)
{
    long long k = 0;
    double ms = 0.0;
    nk::dense_jit_stats(&k, &ms);
    if (kernels) *kernels = k;
    if (compile_ms) *compile_ms = ms;
    return NK_OK;
}

// =========================== diagnostics ===========================
namespace {
__global__ void __launch_bounds__(256) dfma_probe(int iters, double x, double y, double* sink)
{
    double acc[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) acc[c] = threadIdx.x * 1e-9 + c;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 128; ++u) { // 1024 DFMA per trip: the loop body stays inside the instruction cache
                                        // (a 4096-DFMA body measured 33 instead of 37 TFLOP/s)
#pragma unroll
            for (int c = 0; c < 8; ++c) acc[c] = fma(acc[c], x, y);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 8; ++c) s += acc[c];
    if (s == 123.456) sink[0] = s;
}
} // namespace

extern "C" nk_status nk_probe_fp64_peak(int iters, double* tflops, double* ms_out)
{
    if (iters < 1 || !tflops) return fail(NK_ERR_INVALID_ARG, "nk_probe_fp64_peak: bad arguments");
    nk_status st = ensure_device();
    if (st != NK_OK) return st;
    double* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return cuda_fail(e, "nk_probe_fp64_peak: cudaMalloc");
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = g_num_sms * 8, threads = 256;
    dfma_probe<<<blocks, threads>>>(1, 0.999999, 1e-9, sink); // warm-up
    cudaEventRecord(t0);
    dfma_probe<<<blocks, threads>>>(iters, 0.999999, 1e-9, sink);
    cudaEventRecord(t1);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, t0, t1);
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    { std::lock_guard<std::mutex> lk(g_mutex); g_launches += 2; }
    if (e != cudaSuccess) return cuda_fail(e, "nk_probe_fp64_peak");
    const double flops = 2.0 * 1024.0 * iters * (double)blocks * threads;
    *tflops = flops / (ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = ms;
    return NK_OK;
}

namespace {
// the same for the FP64 tensor-core path: 8 independent DMMA.8x8x4 accumulator chains per warp, 128 DMMA per trip
__global__ void __launch_bounds__(256) dmma_probe(int iters, double x, double y, double* sink)
{
    double acc[8][2];
#pragma unroll
    for (int c = 0; c < 8; ++c) { acc[c][0] = threadIdx.x * 1e-9 + c; acc[c][1] = c; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u)
#pragma unroll
            for (int c = 0; c < 8; ++c) nk::dmma884(acc[c][0], acc[c][1], x, y);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 8; ++c) s += acc[c][0] + acc[c][1];
    if (s == 123.456) sink[0] = s;
}
} // namespace

extern "C" nk_status nk_probe_fp64_dmma_peak(int iters, double* tflops, double* ms_out)
{
    if (iters < 1 || !tflops) return fail(NK_ERR_INVALID_ARG, "nk_probe_fp64_dmma_peak: bad arguments");
    nk_status st = ensure_device();
    if (st != NK_OK) return st;
    double* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return cuda_fail(e, "nk_probe_fp64_dmma_peak: cudaMalloc");
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = g_num_sms * 8, threads = 256;
    dmma_probe<<<blocks, threads>>>(1, 0.999999, 1e-9, sink); // warm-up
    cudaEventRecord(t0);
    dmma_probe<<<blocks, threads>>>(iters, 0.999999, 1e-9, sink);
    cudaEventRecord(t1);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, t0, t1);
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    { std::lock_guard<std::mutex> lk(g_mutex); g_launches += 2; }
    if (e != cudaSuccess) return cuda_fail(e, "nk_probe_fp64_dmma_peak");
    // one m8n8k4 DMMA = 8 x 8 x 4 FMA per warp
    const double flops = 2.0 * 256.0 * 128.0 * iters * (double)blocks * (threads / 32);
    *tflops = flops / (ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = ms;
    return NK_OK;
}

extern "C" int64_t nk_launch_count(void)
{
    std::lock_guard<std::mutex> lk(g_mutex);
    return g_launches;
}
extern "C" const char* nk_last_error(void) { return g_err.c_str(); }
// for the other translation units of the library (nk_solver.cu): not declared in nk.h
extern "C" void nk_set_error_(const char* msg) { g_err = msg ? msg : ""; }
extern "C" void nk_count_launches_(int n)
{
    std::lock_guard<std::mutex> lk(g_mutex);
    g_launches += n;
}
// Would nk_helmholtz_apply(b, g, ...) allocate device memory or load a module if called NOW on the current device?
// 0 = no: the sum-factorised / Kronecker kernels take their tables as kernel parameters, and a prebuilt reference-matrix
// kernel whose fragment-ordered matrices are already resident on this device allocates nothing; 1 = yes: the matrices
// are still to be uploaded (first apply on this basis) or the kernel would be specialised at run time (nk_jit.cu).
// For nk_assembled_helmholtz_apply_static (nk_solver.cu), which must not allocate.  Not declared in nk.h.
extern "C" int nk_helmholtz_apply_allocates_(const nk_basis* b, const nk_geom* g)
{
    if (!b || !g) return 1;
    if (b->jit) return 1;      // a basis outside the prebuilt table: its kernels are compiled and loaded on first use
    nk_status st = NK_OK;
    if (!use_dense(b, g->deformed, nk::OP_HELM, &st)) return st == NK_OK ? 0 : 1;
    if (!nk::dense_supported(b->t.Nm)) return 1;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return 1;
    std::lock_guard<std::mutex> lk(b->mu);
    return (b->d_frag[nk::DENSE_HELM] && b->frag_dev == dev) ? 0 : 1;
}
extern "C" const char* nk_version(void) { return "libnk 0.2 (sm_100a)"; }
