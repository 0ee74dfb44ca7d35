// nk_solver.cu -- SURVEY 8(f) item 3: global gather-scatter for C0 continuity and a matrix-free conjugate-gradient
// solve of the assembled Helmholtz system.  The paper leaves assembly out ("the local contributions ... must be
// assembled into a global system ... not discussed as a part of this work") and names the consumer of the elemental
// operators ("operator evaluations are required within the solver as part of a conjugate gradient or GMRES
// iteration"); this file is that consumer:
//     A = Q^T diag(H^e) Q,   H^e = L^e + lambda M^e (Eq. 6),   (Q u)[e][m] = s[e][m] u[l2g[e][m]]
// with the caller's local-to-global map l2g and orientation signs s (+-1).  Every vector operation is deterministic:
// the scatter Q^T runs over the TRANSPOSED map (one thread per global dof sums its local copies in a fixed order, no
// atomics), dot products are two-stage reductions with a fixed grid, and the CG scalars never leave the device
// except for the convergence test (one 8-byte read per iteration).
#include <cmath>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/nk.h"

namespace {


enum { kRedBlocks = 592, kRedThreads = 256 };   // 4 blocks per SM of a B200; the grid is FIXED so that sums are reproducible

// free: optional [nglobal] flags, 1 = free dof, 0 = constrained (reads as 0: the operator acts on the free dofs only)
__global__ void gather_kernel(const int* __restrict__ l2g, const signed char* __restrict__ sgn, const unsigned char* __restrict__ free,
                              const double* __restrict__ glob, double* __restrict__ loc, long long n)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int g = l2g[i];
        const double v = (!free || free[g]) ? __ldg(glob + g) : 0.0;
        loc[i] = sgn ? (sgn[i] < 0 ? -v : v) : v;
    }
}

// global[g] = sum over the local copies of g, in the order of the transposed map (CSR: rowptr, col = local index)
// free / ident: a constrained dof takes ident[g] (identity row of the constrained operator) or 1 if ident is NULL
__global__ void scatter_kernel(const long long* __restrict__ rowptr, const int* __restrict__ col, const signed char* __restrict__ sgn,
                               const double* __restrict__ loc, double* __restrict__ glob, long long nglobal,
                               const unsigned char* __restrict__ free = nullptr, const double* __restrict__ ident = nullptr)
{
    for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < nglobal; g += (long long)gridDim.x * blockDim.x) {
        if (free && !free[g]) {
            glob[g] = ident ? ident[g] : 1.0;
            continue;
        }
        double s = 0.0;
        for (long long k = rowptr[g]; k < rowptr[g + 1]; ++k) {
            const int c = col[k];
            const double v = __ldg(loc + c);
            s += sgn ? (sgn[c] < 0 ? -v : v) : v;
        }
        glob[g] = s;
    }
}

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double part[kRedThreads / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x < 32) {
        s = threadIdx.x < kRedThreads / 32 ? part[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    }
    return s;   // valid in thread 0
}

// stage 1 of a dot product: partial[b] = sum over this block's strided share of a[i] b[i]
__global__ void __launch_bounds__(kRedThreads) dot_partial(const double* __restrict__ a, const double* __restrict__ b, long long n,
                                                            double* __restrict__ partial)
{
    double v = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) v = fma(a[i], b[i], v);
    const double s = block_sum(v);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// CG scalars on the device: sc[0] = rr, sc[1] = pAp, sc[2] = alpha, sc[3] = beta, sc[4] = rr_new
// (S_RR holds r.z, the preconditioned product; S_NORM2 the plain r.r of the convergence test)
enum { S_RR = 0, S_PAP = 1, S_ALPHA = 2, S_BETA = 3, S_RRNEW = 4, S_NORM2 = 5, S_COUNT = 8 };
// stage 2: out = sum of the partials (one block), then the scalar update that follows this dot product
__global__ void __launch_bounds__(kRedThreads) dot_final(const double* __restrict__ partial, int nb, double* __restrict__ sc, int which)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < nb; i += blockDim.x) v += partial[i];
    const double s = block_sum(v);
    if (threadIdx.x == 0) {
        if (which == S_RR) {
            sc[S_RR] = s;
        } else if (which == S_NORM2) {
            sc[S_NORM2] = s;
        } else if (which == S_PAP) {
            sc[S_PAP] = s;
            sc[S_ALPHA] = s != 0.0 ? sc[S_RR] / s : 0.0;
        } else {
            sc[S_RRNEW] = s;
            sc[S_BETA] = sc[S_RR] != 0.0 ? s / sc[S_RR] : 0.0;
            sc[S_RR] = s;
        }
    }
}

// x += alpha p ; r -= alpha Ap
__global__ void update_xr(double* __restrict__ x, double* __restrict__ r, const double* __restrict__ p, const double* __restrict__ Ap,
                          const double* __restrict__ sc, long long n)
{
    const double alpha = sc[S_ALPHA];
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        x[i] = fma(alpha, p[i], x[i]);
        r[i] = fma(-alpha, Ap[i], r[i]);
    }
}
// p = r + beta p
__global__ void update_p(double* __restrict__ p, const double* __restrict__ r, const double* __restrict__ sc, long long n)
{
    const double beta = sc[S_BETA];
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) p[i] = fma(beta, p[i], r[i]);
}
// z = r / d (Jacobi)
__global__ void jacobi_apply(double* __restrict__ z, const double* __restrict__ r, const double* __restrict__ d, long long n)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) z[i] = r[i] / d[i];
}
// x[e][m] = (m == mode) ? 1 : 0   and   diag[e][mode] = y[e][mode]
__global__ void unit_mode(double* __restrict__ x, long long nelem, int nm, int mode)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < nelem * nm; i += (long long)gridDim.x * blockDim.x)
        x[i] = (int)(i % nm) == mode ? 1.0 : 0.0;
}
__global__ void take_mode(double* __restrict__ diag, const double* __restrict__ y, long long nelem, int nm, int mode)
{
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < nelem; e += (long long)gridDim.x * blockDim.x)
        diag[e * nm + mode] = y[e * nm + mode];
}
// r = b - Ax ; p = r
__global__ void init_rp(double* __restrict__ r, double* __restrict__ p, const double* __restrict__ b, const double* __restrict__ Ax, long long n)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double v = b[i] - Ax[i];
        r[i] = v;
        p[i] = v;
    }
}

} // namespace

// nk_api.cu owns the thread-local message of nk_last_error() and the launch counter of nk_launch_count()
extern "C" void nk_set_error_(const char* msg);
extern "C" void nk_count_launches_(int n);

namespace {
nk_status sfail(nk_status s, const std::string& m)
{
    nk_set_error_(m.c_str());
    return s;
}
} // namespace

struct nk_gs {
    int64_t nelem = 0, nglobal = 0, nlocal = 0;
    int nm = 0;
    int* d_l2g = nullptr;            // [nlocal]
    signed char* d_sgn = nullptr;    // [nlocal] or NULL (all +1)
    long long* d_rowptr = nullptr;   // [nglobal + 1]
    int* d_col = nullptr;            // [nlocal]
    unsigned char* d_free = nullptr; // [nglobal] 1 = free, 0 = constrained; NULL = no constraints (nk_gs_set_constrained)
    // work space of nk_assembled_apply / nk_cg_solve (allocated on first use, under mu)
    std::mutex mu;
    double *d_lin = nullptr, *d_lout = nullptr, *d_r = nullptr, *d_p = nullptr, *d_Ap = nullptr, *d_partial = nullptr, *d_sc = nullptr;
    double *d_z = nullptr, *d_diag = nullptr, *d_ldiag = nullptr;     // Jacobi: z, diag(A) (global), elemental diagonals (local)
    const void* diag_geom = nullptr;                                   // the (geometry, lambda) the cached diagonal belongs to
    double diag_lambda = 0.0;
};

extern "C" nk_status nk_gs_create(int64_t nelem, int nm_local, int64_t nglobal, const int64_t* l2g, const signed char* sign, nk_gs** out)
{
    if (!out) return sfail(NK_ERR_INVALID_ARG, "nk_gs_create: out is NULL");
    *out = nullptr;
    if (nelem < 0 || nm_local < 1 || nglobal < 0 || (nelem > 0 && !l2g)) return sfail(NK_ERR_INVALID_ARG, "nk_gs_create: bad arguments");
    const int64_t nlocal = nelem * nm_local;
    if (nlocal >= 0x7fffffffLL || nglobal >= 0x7fffffffLL) return sfail(NK_ERR_UNSUPPORTED, "nk_gs_create: more than 2^31 - 1 local or global dofs");
    // transposed map (counting sort): the local copies of each global dof, in increasing local index
    std::vector<long long> rowptr((size_t)nglobal + 1, 0);
    for (int64_t i = 0; i < nlocal; ++i) {
        if (l2g[i] < 0 || l2g[i] >= nglobal) return sfail(NK_ERR_INVALID_ARG, "nk_gs_create: l2g entry out of range");
        if (sign && sign[i] != 1 && sign[i] != -1) return sfail(NK_ERR_INVALID_ARG, "nk_gs_create: signs must be +1 or -1");
        ++rowptr[(size_t)l2g[i] + 1];
    }
    for (int64_t g = 0; g < nglobal; ++g) rowptr[(size_t)g + 1] += rowptr[(size_t)g];
    std::vector<int> col((size_t)nlocal), l32((size_t)nlocal);
    {
        std::vector<long long> fill(rowptr.begin(), rowptr.end() - 1);
        for (int64_t i = 0; i < nlocal; ++i) {
            col[(size_t)fill[(size_t)l2g[i]]++] = (int)i;
            l32[(size_t)i] = (int)l2g[i];
        }
    }
    nk_gs* gs = new (std::nothrow) nk_gs;
    if (!gs) return sfail(NK_ERR_ALLOC, "nk_gs_create: out of memory");
    gs->nelem = nelem;
    gs->nglobal = nglobal;
    gs->nlocal = nlocal;
    gs->nm = nm_local;
    *out = gs;
    if (nlocal == 0) return NK_OK;
    cudaError_t e = cudaMalloc(&gs->d_l2g, (size_t)nlocal * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&gs->d_col, (size_t)nlocal * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&gs->d_rowptr, ((size_t)nglobal + 1) * sizeof(long long));
    if (e == cudaSuccess && sign) e = cudaMalloc(&gs->d_sgn, (size_t)nlocal);
    if (e == cudaSuccess) e = cudaMemcpy(gs->d_l2g, l32.data(), (size_t)nlocal * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(gs->d_col, col.data(), (size_t)nlocal * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(gs->d_rowptr, rowptr.data(), ((size_t)nglobal + 1) * sizeof(long long), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && sign) e = cudaMemcpy(gs->d_sgn, sign, (size_t)nlocal, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        const std::string msg = std::string("nk_gs_create: ") + cudaGetErrorString(e);
        nk_gs_destroy(gs);
        *out = nullptr;
        return sfail(NK_ERR_CUDA, msg);
    }
    return NK_OK;
}

extern "C" nk_status nk_gs_destroy(nk_gs* gs)
{
    if (!gs) return NK_OK;
    for (void* p : {(void*)gs->d_free, (void*)gs->d_l2g, (void*)gs->d_sgn, (void*)gs->d_rowptr, (void*)gs->d_col, (void*)gs->d_lin, (void*)gs->d_lout,
                    (void*)gs->d_r, (void*)gs->d_p, (void*)gs->d_Ap, (void*)gs->d_partial, (void*)gs->d_sc, (void*)gs->d_z, (void*)gs->d_diag,
                    (void*)gs->d_ldiag})
        if (p) cudaFree(p);
    delete gs;
    return NK_OK;
}

extern "C" int64_t nk_gs_num_global(const nk_gs* gs) { return gs ? gs->nglobal : -1; }

extern "C" nk_status nk_gs_set_constrained(nk_gs* gs, int64_t n, const int64_t* dofs)
{
    if (!gs || n < 0 || (n > 0 && !dofs)) return sfail(NK_ERR_INVALID_ARG, "nk_gs_set_constrained: bad arguments");
    std::lock_guard<std::mutex> lk(gs->mu);
    gs->diag_geom = nullptr;                       // the cached Jacobi diagonal belongs to the old constraint set
    if (n == 0) {
        if (gs->d_free) cudaFree(gs->d_free);
        gs->d_free = nullptr;
        return NK_OK;
    }
    std::vector<unsigned char> f((size_t)gs->nglobal, 1);
    for (int64_t i = 0; i < n; ++i) {
        if (dofs[i] < 0 || dofs[i] >= gs->nglobal) return sfail(NK_ERR_INVALID_ARG, "nk_gs_set_constrained: dof out of range");
        f[(size_t)dofs[i]] = 0;
    }
    cudaError_t e = cudaSuccess;
    if (!gs->d_free) e = cudaMalloc(&gs->d_free, (size_t)gs->nglobal);
    if (e == cudaSuccess) e = cudaMemcpy(gs->d_free, f.data(), (size_t)gs->nglobal, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return sfail(NK_ERR_CUDA, std::string("nk_gs_set_constrained: ") + cudaGetErrorString(e));
    return NK_OK;
}

static int grid_for(long long n)
{
    long long b = (n + 255) / 256;
    return (int)(b < 1 ? 1 : b > 148LL * 16 ? 148LL * 16 : b);
}

extern "C" nk_status nk_gs_gather(const nk_gs* gs, const double* global, double* local, void* stream)
{
    if (!gs || (gs->nlocal > 0 && (!global || !local))) return sfail(NK_ERR_INVALID_ARG, "nk_gs_gather: NULL argument");
    if (gs->nlocal == 0) return NK_OK;
    gather_kernel<<<grid_for(gs->nlocal), 256, 0, (cudaStream_t)stream>>>(gs->d_l2g, gs->d_sgn, nullptr, global, local, gs->nlocal);
    nk_count_launches_(1);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, std::string("nk_gs_gather: ") + cudaGetErrorString(e));
}

extern "C" nk_status nk_gs_scatter_add(const nk_gs* gs, const double* local, double* global, void* stream)
{
    if (!gs || (gs->nglobal > 0 && (!global || (gs->nlocal > 0 && !local)))) return sfail(NK_ERR_INVALID_ARG, "nk_gs_scatter_add: NULL argument");
    if (gs->nglobal == 0) return NK_OK;
    scatter_kernel<<<grid_for(gs->nglobal), 256, 0, (cudaStream_t)stream>>>(gs->d_rowptr, gs->d_col, gs->d_sgn, local, global, gs->nglobal);
    nk_count_launches_(1);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, std::string("nk_gs_scatter_add: ") + cudaGetErrorString(e));
}

static nk_status ensure_work(nk_gs* gs)
{
    if (gs->d_lin) return NK_OK;
    cudaError_t e = cudaSuccess;
    double** bufs[] = {&gs->d_lin, &gs->d_lout, &gs->d_r, &gs->d_p, &gs->d_Ap, &gs->d_partial, &gs->d_sc, &gs->d_z, &gs->d_diag, &gs->d_ldiag};
    const size_t sizes[] = {(size_t)gs->nlocal, (size_t)gs->nlocal, (size_t)gs->nglobal, (size_t)gs->nglobal, (size_t)gs->nglobal,
                            (size_t)kRedBlocks, (size_t)S_COUNT, (size_t)gs->nglobal, (size_t)gs->nglobal, (size_t)gs->nlocal};
    constexpr int NB = 10;
    double* got[NB] = {};
    for (int i = 0; i < NB && e == cudaSuccess; ++i) e = cudaMalloc(&got[i], (sizes[i] ? sizes[i] : 1) * sizeof(double));
    if (e != cudaSuccess) {
        for (double* p : got)
            if (p) cudaFree(p);
        cudaGetLastError();
        return sfail(NK_ERR_ALLOC, "nk_gs: cudaMalloc of the work space failed");
    }
    for (int i = 0; i < NB; ++i) *bufs[i] = got[i];
    return NK_OK;
}

// out = A in on the caller's stream, A = Q^T H Q, or with constrained dofs A = P Q^T H Q P + (I - P) (P = projector on
// the free dofs: identity rows and columns at the constrained ones); work space of gs (callers hold gs->mu)
static nk_status assembled_apply(const nk_basis* b, const nk_geom* g, nk_gs* gs, double lambda, const double* in, double* out, void* stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    gather_kernel<<<grid_for(gs->nlocal), 256, 0, s>>>(gs->d_l2g, gs->d_sgn, gs->d_free, in, gs->d_lin, gs->nlocal);
    nk_status st = nk_helmholtz_apply(b, g, lambda, gs->d_lin, gs->d_lout, stream);
    if (st != NK_OK) return st;
    scatter_kernel<<<grid_for(gs->nglobal), 256, 0, s>>>(gs->d_rowptr, gs->d_col, gs->d_sgn, gs->d_lout, out, gs->nglobal, gs->d_free, in);
    nk_count_launches_(2);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, std::string("assembled apply: ") + cudaGetErrorString(e));
}

extern "C" nk_status nk_assembled_helmholtz_apply(const nk_basis* b, const nk_geom* g, const nk_gs* gsc, double lambda, const double* in,
                                                  double* out, void* stream)
{
    if (!b || !g || !gsc || !in || !out) return sfail(NK_ERR_INVALID_ARG, "nk_assembled_helmholtz_apply: NULL argument");
    nk_gs* gs = const_cast<nk_gs*>(gsc);
    if (gs->nelem != nk_geom_num_elements(g) || gs->nm != nk_basis_num_modes(b))
        return sfail(NK_ERR_SHAPE_MISMATCH, "nk_assembled_helmholtz_apply: the map does not belong to this block");
    if (in == out) return sfail(NK_ERR_INVALID_ARG, "nk_assembled_helmholtz_apply: in and out alias");
    if (gs->nglobal == 0) return NK_OK;
    std::lock_guard<std::mutex> lk(gs->mu);
    nk_status st = ensure_work(gs);
    if (st != NK_OK) return st;
    return assembled_apply(b, g, gs, lambda, in, out, stream);
}

// diag(A) = Q^T diag(H^e): the elemental diagonals by Nm applications of the elemental operator to unit vectors
// (entry m of H^e e_m, all elements at once); cached per (geometry, lambda)
static nk_status assembled_diagonal(const nk_basis* b, const nk_geom* g, nk_gs* gs, double lambda, void* stream)
{
    if (gs->diag_geom == (const void*)g && gs->diag_lambda == lambda) return NK_OK;
    cudaStream_t s = (cudaStream_t)stream;
    const int gl = grid_for(gs->nlocal);
    for (int m = 0; m < gs->nm; ++m) {
        unit_mode<<<gl, 256, 0, s>>>(gs->d_lin, gs->nelem, gs->nm, m);
        nk_status st = nk_helmholtz_apply(b, g, lambda, gs->d_lin, gs->d_lout, stream);
        if (st != NK_OK) return st;
        take_mode<<<grid_for(gs->nelem), 256, 0, s>>>(gs->d_ldiag, gs->d_lout, gs->nelem, gs->nm, m);
        nk_count_launches_(2);
    }
    // signs square to one: the plain transposed sum (a map without signs)
    scatter_kernel<<<grid_for(gs->nglobal), 256, 0, s>>>(gs->d_rowptr, gs->d_col, nullptr, gs->d_ldiag, gs->d_diag, gs->nglobal, gs->d_free, nullptr);
    nk_count_launches_(1);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return sfail(NK_ERR_CUDA, std::string("nk_cg_solve: diagonal: ") + cudaGetErrorString(e));
    gs->diag_geom = (const void*)g;
    gs->diag_lambda = lambda;
    return NK_OK;
}

extern "C" nk_status nk_cg_solve(const nk_basis* b, const nk_geom* g, const nk_gs* gsc, double lambda, const double* rhs, double* x,
                                 int precond, double rtol, int maxit, int* iters_out, double* relres_out, void* stream)
{
    if (precond != NK_PRECOND_NONE && precond != NK_PRECOND_JACOBI) return sfail(NK_ERR_INVALID_ARG, "nk_cg_solve: unknown preconditioner");
    if (!b || !g || !gsc || !rhs || !x) return sfail(NK_ERR_INVALID_ARG, "nk_cg_solve: NULL argument");
    if (!(rtol >= 0.0) || maxit < 0) return sfail(NK_ERR_INVALID_ARG, "nk_cg_solve: rtol >= 0 and maxit >= 0 required");
    nk_gs* gs = const_cast<nk_gs*>(gsc);
    if (gs->nelem != nk_geom_num_elements(g) || gs->nm != nk_basis_num_modes(b))
        return sfail(NK_ERR_SHAPE_MISMATCH, "nk_cg_solve: the map does not belong to this block");
    if (rhs == x) return sfail(NK_ERR_INVALID_ARG, "nk_cg_solve: rhs and x alias");
    if (iters_out) *iters_out = 0;
    if (relres_out) *relres_out = 0.0;
    if (gs->nglobal == 0) return NK_OK;
    std::lock_guard<std::mutex> lk(gs->mu);
    nk_status st = ensure_work(gs);
    if (st != NK_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    const long long n = gs->nglobal;
    const int gv = grid_for(n);
    double h[S_COUNT];
    auto dot = [&](const double* a_, const double* b_, int which) {
        dot_partial<<<kRedBlocks, kRedThreads, 0, s>>>(a_, b_, n, gs->d_partial);
        dot_final<<<1, kRedThreads, 0, s>>>(gs->d_partial, kRedBlocks, gs->d_sc, which);
        nk_count_launches_(2);
    };
    auto read_scalars = [&]() -> cudaError_t {
        cudaError_t e = cudaMemcpyAsync(h, gs->d_sc, sizeof h, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        return e;
    };
    const bool pc = precond == NK_PRECOND_JACOBI;
    if (pc) {
        st = assembled_diagonal(b, g, gs, lambda, stream);
        if (st != NK_OK) return st;
    }
    double* z = pc ? gs->d_z : gs->d_r;          // without a preconditioner z IS r
    // ||b||
    dot(rhs, rhs, S_NORM2);
    cudaError_t e = read_scalars();
    if (e != cudaSuccess) return sfail(NK_ERR_CUDA, std::string("nk_cg_solve: ") + cudaGetErrorString(e));
    const double bnorm = std::sqrt(h[S_NORM2]);
    if (!(bnorm > 0.0)) {   // b = 0: the solution is 0
        e = cudaMemsetAsync(x, 0, (size_t)n * sizeof(double), s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, "nk_cg_solve: memset");
    }
    // r = b - A x0 ; z = M^-1 r ; p = z ; rz = r.z
    st = assembled_apply(b, g, gs, lambda, x, gs->d_Ap, stream);
    if (st != NK_OK) return st;
    init_rp<<<gv, 256, 0, s>>>(gs->d_r, gs->d_p, rhs, gs->d_Ap, n);
    nk_count_launches_(1);
    if (pc) {
        jacobi_apply<<<gv, 256, 0, s>>>(z, gs->d_r, gs->d_diag, n);
        e = cudaMemcpyAsync(gs->d_p, z, (size_t)n * sizeof(double), cudaMemcpyDeviceToDevice, s);
        if (e != cudaSuccess) return sfail(NK_ERR_CUDA, "nk_cg_solve: copy");
        nk_count_launches_(1);
    }
    dot(gs->d_r, z, S_RR);
    dot(gs->d_r, gs->d_r, S_NORM2);
    e = read_scalars();
    if (e != cudaSuccess) return sfail(NK_ERR_CUDA, std::string("nk_cg_solve: ") + cudaGetErrorString(e));
    double rel = std::sqrt(h[S_NORM2]) / bnorm;
    int it = 0;
    while (it < maxit && rel > rtol) {
        st = assembled_apply(b, g, gs, lambda, gs->d_p, gs->d_Ap, stream);
        if (st != NK_OK) return st;
        dot(gs->d_p, gs->d_Ap, S_PAP);                         // alpha = rz / pAp
        update_xr<<<gv, 256, 0, s>>>(x, gs->d_r, gs->d_p, gs->d_Ap, gs->d_sc, n);
        if (pc) jacobi_apply<<<gv, 256, 0, s>>>(z, gs->d_r, gs->d_diag, n);
        dot(gs->d_r, z, S_RRNEW);                              // beta = rz_new / rz ; rz = rz_new
        update_p<<<gv, 256, 0, s>>>(gs->d_p, z, gs->d_sc, n);  // p = z + beta p
        if (pc) dot(gs->d_r, gs->d_r, S_NORM2);
        nk_count_launches_(pc ? 3 : 2);
        e = read_scalars();
        if (e != cudaSuccess) return sfail(NK_ERR_CUDA, std::string("nk_cg_solve: ") + cudaGetErrorString(e));
        ++it;
        if (!(h[S_PAP] > 0.0)) return sfail(NK_ERR_INVALID_ARG, "nk_cg_solve: p.Ap <= 0 (the operator is not positive definite: lambda > 0 needed)");
        rel = std::sqrt(pc ? h[S_NORM2] : h[S_RR]) / bnorm;
    }
    if (iters_out) *iters_out = it;
    if (relres_out) *relres_out = rel;
    return NK_OK;
}

// =========================== partitioned solve (several ranks, one sub-mesh each) ===========================
// A mesh split over ranks by elements (contiguous element ranges) shares the dofs on the cut: every
// rank holds them in its own numbering and the assembled operator needs their contributions from all ranks.  That sum is
// the one data-path exchange of this library ("first consumer of multi-GPU"):
//     y = A x:   local Q^T H Q on the rank's elements, then  y[shared] <- sum over ranks  (pack, all-reduce, unpack)
//     <a, b>:    sum_i w_i a_i b_i with w_i = 1 / (number of ranks holding dof i), then a scalar all-reduce
// for vectors that are CONSISTENT (equal on every rank that holds a dof).  The all-reduce itself is the caller's
// (a C callback: torch.distributed / NCCL over NVLink in the Python binding); everything else runs in the kernels below.
namespace {
enum { S_TMP0 = 6, S_TMP1 = 7 };
__global__ void pack_kernel(const int* __restrict__ sdof, const int* __restrict__ sslot, const unsigned char* __restrict__ free,
                            const double* __restrict__ vec, double* __restrict__ ibuf, long long ns)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ns; i += (long long)gridDim.x * blockDim.x) {
        const int d = sdof[i];
        ibuf[sslot[i]] = (!free || free[d]) ? vec[d] : 0.0;     // constrained dofs keep their identity row: nothing to sum
    }
}
__global__ void unpack_kernel(const int* __restrict__ sdof, const int* __restrict__ sslot, const unsigned char* __restrict__ free,
                              double* __restrict__ vec, const double* __restrict__ ibuf, long long ns)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ns; i += (long long)gridDim.x * blockDim.x) {
        const int d = sdof[i];
        if (!free || free[d]) vec[d] = ibuf[sslot[i]];
    }
}
__global__ void __launch_bounds__(kRedThreads) dot_partial_w(const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ w,
                                                              long long n, double* __restrict__ partial)
{
    double v = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) v = fma(w[i] * a[i], b[i], v);
    const double s = block_sum(v);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}
__global__ void __launch_bounds__(kRedThreads) sum_final(const double* __restrict__ partial, int nb, double* __restrict__ sc, int slot)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < nb; i += blockDim.x) v += partial[i];
    const double s = block_sum(v);
    if (threadIdx.x == 0) sc[slot] = s;
}
// the scalar updates of CG once the reduced sums sit in sc[S_TMP0], sc[S_TMP1]
__global__ void cg_scalars(double* __restrict__ sc, int which)
{
    if (which == S_RR) {                  // start: rz, rr
        sc[S_RR] = sc[S_TMP0];
        sc[S_NORM2] = sc[S_TMP1];
    } else if (which == S_PAP) {          // alpha = rz / pAp
        sc[S_PAP] = sc[S_TMP0];
        sc[S_ALPHA] = sc[S_TMP0] != 0.0 ? sc[S_RR] / sc[S_TMP0] : 0.0;
    } else {                              // beta = rz_new / rz ; rz = rz_new ; rr
        sc[S_RRNEW] = sc[S_TMP0];
        sc[S_BETA] = sc[S_RR] != 0.0 ? sc[S_TMP0] / sc[S_RR] : 0.0;
        sc[S_RR] = sc[S_TMP0];
        sc[S_NORM2] = sc[S_TMP1];
    }
}
} // namespace

struct nk_part {
    nk_gs* gs = nullptr;
    int64_t ns = 0, ni = 0;
    int *d_sdof = nullptr, *d_sslot = nullptr;
    double *d_w = nullptr, *d_ibuf = nullptr, *d_diag = nullptr;     // weights [nglobal], interface vector [ni], exchanged diag(A)
    const void* diag_geom = nullptr;
    double diag_lambda = 0.0;
    nk_allreduce_fn fn = nullptr;
    void* user = nullptr;
};

extern "C" nk_status nk_part_destroy(nk_part* p)
{
    if (!p) return NK_OK;
    for (void* q : {(void*)p->d_sdof, (void*)p->d_sslot, (void*)p->d_w, (void*)p->d_ibuf, (void*)p->d_diag})
        if (q) cudaFree(q);
    delete p;
    return NK_OK;
}

extern "C" nk_status nk_part_create(nk_gs* gs, int64_t n_shared, const int64_t* shared_dof, const int64_t* shared_slot, const int32_t* shared_mult,
                                    int64_t n_interface, nk_allreduce_fn allreduce, void* user, nk_part** out)
{
    if (!out) return sfail(NK_ERR_INVALID_ARG, "nk_part_create: out is NULL");
    *out = nullptr;
    if (!gs || !allreduce || n_shared < 0 || n_interface < 0 || n_shared > n_interface ||
        (n_shared > 0 && (!shared_dof || !shared_slot || !shared_mult)))
        return sfail(NK_ERR_INVALID_ARG, "nk_part_create: bad arguments");
    std::vector<int> sd((size_t)n_shared), ss((size_t)n_shared);
    std::vector<double> w((size_t)gs->nglobal, 1.0);
    std::vector<unsigned char> seen((size_t)n_interface, 0);
    for (int64_t i = 0; i < n_shared; ++i) {
        if (shared_dof[i] < 0 || shared_dof[i] >= gs->nglobal || shared_slot[i] < 0 || shared_slot[i] >= n_interface || shared_mult[i] < 2)
            return sfail(NK_ERR_INVALID_ARG, "nk_part_create: shared dof / slot out of range, or multiplicity < 2");
        if (seen[(size_t)shared_slot[i]] || w[(size_t)shared_dof[i]] != 1.0)
            return sfail(NK_ERR_INVALID_ARG, "nk_part_create: a shared dof or an interface slot is listed twice");
        seen[(size_t)shared_slot[i]] = 1;
        sd[(size_t)i] = (int)shared_dof[i];
        ss[(size_t)i] = (int)shared_slot[i];
        w[(size_t)shared_dof[i]] = 1.0 / (double)shared_mult[i];
    }
    nk_part* p = new (std::nothrow) nk_part;
    if (!p) return sfail(NK_ERR_ALLOC, "nk_part_create: out of memory");
    p->gs = gs;
    p->ns = n_shared;
    p->ni = n_interface;
    p->fn = allreduce;
    p->user = user;
    cudaError_t e = cudaMalloc(&p->d_w, (size_t)(gs->nglobal ? gs->nglobal : 1) * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_diag, (size_t)(gs->nglobal ? gs->nglobal : 1) * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_ibuf, (size_t)(n_interface ? n_interface : 1) * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_sdof, (size_t)(n_shared ? n_shared : 1) * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_sslot, (size_t)(n_shared ? n_shared : 1) * sizeof(int));
    if (e == cudaSuccess && gs->nglobal) e = cudaMemcpy(p->d_w, w.data(), (size_t)gs->nglobal * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && n_shared) e = cudaMemcpy(p->d_sdof, sd.data(), (size_t)n_shared * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && n_shared) e = cudaMemcpy(p->d_sslot, ss.data(), (size_t)n_shared * sizeof(int), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        const std::string msg = std::string("nk_part_create: ") + cudaGetErrorString(e);
        nk_part_destroy(p);
        return sfail(e == cudaErrorMemoryAllocation ? NK_ERR_ALLOC : NK_ERR_CUDA, msg);
    }
    *out = p;
    return NK_OK;
}

// vec[shared] <- sum over ranks of vec[shared] (free dofs only); every rank must call it (the all-reduce is collective)
static nk_status part_exchange(nk_part* p, double* vec, void* stream)
{
    if (p->ni == 0) return NK_OK;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = cudaMemsetAsync(p->d_ibuf, 0, (size_t)p->ni * sizeof(double), s);
    if (e != cudaSuccess) return sfail(NK_ERR_CUDA, std::string("partition exchange: ") + cudaGetErrorString(e));
    if (p->ns > 0) {
        pack_kernel<<<grid_for(p->ns), 256, 0, s>>>(p->d_sdof, p->d_sslot, p->gs->d_free, vec, p->d_ibuf, p->ns);
        nk_count_launches_(1);
    }
    if (p->fn(p->user, p->d_ibuf, p->ni, stream) != 0) return sfail(NK_ERR_CUDA, "partition exchange: the all-reduce callback failed");
    if (p->ns > 0) {
        unpack_kernel<<<grid_for(p->ns), 256, 0, s>>>(p->d_sdof, p->d_sslot, p->gs->d_free, vec, p->d_ibuf, p->ns);
        nk_count_launches_(1);
    }
    e = cudaGetLastError();
    return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, std::string("partition exchange: ") + cudaGetErrorString(e));
}

static nk_status part_check(const char* name, const nk_basis* b, const nk_geom* g, const nk_part* p)
{
    if (!b || !g || !p) return sfail(NK_ERR_INVALID_ARG, std::string(name) + ": NULL argument");
    if (p->gs->nelem != nk_geom_num_elements(g) || p->gs->nm != nk_basis_num_modes(b))
        return sfail(NK_ERR_SHAPE_MISMATCH, std::string(name) + ": the map does not belong to this block");
    return NK_OK;
}

extern "C" nk_status nk_part_exchange_sum(nk_part* p, double* vec, void* stream)
{
    if (!p || (!vec && p->gs->nglobal > 0)) return sfail(NK_ERR_INVALID_ARG, "nk_part_exchange_sum: NULL argument");
    std::lock_guard<std::mutex> lk(p->gs->mu);
    return part_exchange(p, vec, stream);
}

extern "C" nk_status nk_part_assembled_helmholtz_apply(const nk_basis* b, const nk_geom* g, nk_part* p, double lambda, const double* in,
                                                       double* out, void* stream)
{
    nk_status st = part_check("nk_part_assembled_helmholtz_apply", b, g, p);
    if (st != NK_OK) return st;
    if (!in || !out || in == out) return sfail(NK_ERR_INVALID_ARG, "nk_part_assembled_helmholtz_apply: NULL or aliased vectors");
    nk_gs* gs = p->gs;
    std::lock_guard<std::mutex> lk(gs->mu);
    st = ensure_work(gs);
    if (st != NK_OK) return st;
    if (gs->nglobal > 0) {
        st = assembled_apply(b, g, gs, lambda, in, out, stream);
        if (st != NK_OK) return st;
    }
    return part_exchange(p, out, stream);
}

extern "C" nk_status nk_part_cg_solve(const nk_basis* b, const nk_geom* g, nk_part* p, double lambda, const double* rhs, double* x, int precond,
                                      double rtol, int maxit, int* iters_out, double* relres_out, void* stream)
{
    if (precond != NK_PRECOND_NONE && precond != NK_PRECOND_JACOBI) return sfail(NK_ERR_INVALID_ARG, "nk_part_cg_solve: unknown preconditioner");
    nk_status st = part_check("nk_part_cg_solve", b, g, p);
    if (st != NK_OK) return st;
    if (!rhs || !x || rhs == x) return sfail(NK_ERR_INVALID_ARG, "nk_part_cg_solve: NULL or aliased vectors");
    if (!(rtol >= 0.0) || maxit < 0) return sfail(NK_ERR_INVALID_ARG, "nk_part_cg_solve: rtol >= 0 and maxit >= 0 required");
    if (iters_out) *iters_out = 0;
    if (relres_out) *relres_out = 0.0;
    nk_gs* gs = p->gs;
    std::lock_guard<std::mutex> lk(gs->mu);
    st = ensure_work(gs);
    if (st != NK_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    const long long n = gs->nglobal;        // a rank may hold no element: it still takes part in every collective
    const int gv = grid_for(n > 0 ? n : 1);
    double h[S_COUNT];
    auto dotw = [&](const double* a_, const double* b_, int slot) {
        dot_partial_w<<<kRedBlocks, kRedThreads, 0, s>>>(a_, b_, p->d_w, n, gs->d_partial);
        sum_final<<<1, kRedThreads, 0, s>>>(gs->d_partial, kRedBlocks, gs->d_sc, slot);
        nk_count_launches_(2);
    };
    auto reduce = [&](int count, int which) -> nk_status {     // all-reduce sc[S_TMP0 .. S_TMP0 + count), then the scalar updates
        if (p->fn(p->user, gs->d_sc + S_TMP0, count, stream) != 0) return sfail(NK_ERR_CUDA, "nk_part_cg_solve: the all-reduce callback failed");
        if (which >= 0) {
            cg_scalars<<<1, 1, 0, s>>>(gs->d_sc, which);
            nk_count_launches_(1);
        }
        return NK_OK;
    };
    auto read_scalars = [&]() -> nk_status {
        cudaError_t e = cudaMemcpyAsync(h, gs->d_sc, sizeof h, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, std::string("nk_part_cg_solve: ") + cudaGetErrorString(e));
    };
    auto apply = [&](const double* in, double* out) -> nk_status {
        if (n > 0) {
            nk_status a = assembled_apply(b, g, gs, lambda, in, out, stream);
            if (a != NK_OK) return a;
        }
        return part_exchange(p, out, stream);
    };
    const bool pc = precond == NK_PRECOND_JACOBI;
    if (pc && !(p->diag_geom == (const void*)g && p->diag_lambda == lambda)) {
        // diag(A) of the WHOLE mesh: the rank's own Q^T diag(H^e), summed over the ranks on the shared dofs
        if (n > 0) {
            st = assembled_diagonal(b, g, gs, lambda, stream);
            if (st != NK_OK) return st;
            cudaError_t e = cudaMemcpyAsync(p->d_diag, gs->d_diag, (size_t)n * sizeof(double), cudaMemcpyDeviceToDevice, s);
            if (e != cudaSuccess) return sfail(NK_ERR_CUDA, "nk_part_cg_solve: copy of the diagonal");
        }
        st = part_exchange(p, p->d_diag, stream);
        if (st != NK_OK) return st;
        p->diag_geom = (const void*)g;
        p->diag_lambda = lambda;
    }
    double* z = pc ? gs->d_z : gs->d_r;
    // ||b||
    dotw(rhs, rhs, S_TMP0);
    st = reduce(1, -1);
    if (st == NK_OK) st = read_scalars();
    if (st != NK_OK) return st;
    const double bnorm = std::sqrt(h[S_TMP0]);
    if (!(bnorm > 0.0)) {
        cudaError_t e = n > 0 ? cudaMemsetAsync(x, 0, (size_t)n * sizeof(double), s) : cudaSuccess;
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, "nk_part_cg_solve: memset");
    }
    st = apply(x, gs->d_Ap);
    if (st != NK_OK) return st;
    init_rp<<<gv, 256, 0, s>>>(gs->d_r, gs->d_p, rhs, gs->d_Ap, n);
    nk_count_launches_(1);
    if (pc) {
        jacobi_apply<<<gv, 256, 0, s>>>(z, gs->d_r, p->d_diag, n);
        cudaError_t e = n > 0 ? cudaMemcpyAsync(gs->d_p, z, (size_t)n * sizeof(double), cudaMemcpyDeviceToDevice, s) : cudaSuccess;
        if (e != cudaSuccess) return sfail(NK_ERR_CUDA, "nk_part_cg_solve: copy");
        nk_count_launches_(1);
    }
    dotw(gs->d_r, z, S_TMP0);
    dotw(gs->d_r, gs->d_r, S_TMP1);
    st = reduce(2, S_RR);
    if (st == NK_OK) st = read_scalars();
    if (st != NK_OK) return st;
    double rel = std::sqrt(h[S_NORM2]) / bnorm;
    int it = 0;
    while (it < maxit && rel > rtol) {          // rel is the same on every rank: all ranks leave the loop together
        st = apply(gs->d_p, gs->d_Ap);
        if (st != NK_OK) return st;
        dotw(gs->d_p, gs->d_Ap, S_TMP0);
        st = reduce(1, S_PAP);
        if (st != NK_OK) return st;
        update_xr<<<gv, 256, 0, s>>>(x, gs->d_r, gs->d_p, gs->d_Ap, gs->d_sc, n);
        if (pc) jacobi_apply<<<gv, 256, 0, s>>>(z, gs->d_r, p->d_diag, n);
        dotw(gs->d_r, z, S_TMP0);
        dotw(gs->d_r, gs->d_r, S_TMP1);
        st = reduce(2, S_RRNEW);
        if (st != NK_OK) return st;
        update_p<<<gv, 256, 0, s>>>(gs->d_p, z, gs->d_sc, n);
        nk_count_launches_(pc ? 3 : 2);
        st = read_scalars();
        if (st != NK_OK) return st;
        ++it;
        if (!(h[S_PAP] > 0.0)) return sfail(NK_ERR_INVALID_ARG, "nk_part_cg_solve: p.Ap <= 0 (the operator is not positive definite)");
        rel = std::sqrt(h[S_NORM2]) / bnorm;
    }
    if (iters_out) *iters_out = it;
    if (relres_out) *relres_out = rel;
    return NK_OK;
}


// =========================== the entry point that allocates nothing ===========================
// nk_assembled_helmholtz_apply_static (nk.h): nk_assembled_helmholtz_apply with the two local work vectors (Q in and
// H Q in, [nelem][Nm] each) in a file-scope device array instead of cudaMalloc'ed work space of the nk_gs handle, for
// callers that cannot allocate (CUDA graph capture, serving loops).  2 x NK_STATIC_MAX_LOCAL_DOFS doubles = 16 MiB,
// held by every GPU that loads the library until the process exits.
// In HOST code the name nk_static_scratch is a host-side stand-in, not a device address: the kernels get the address
// cudaGetSymbolAddress returns, asked for once per device with that device current (static_scratch below).
static __device__ __align__(256) double nk_static_scratch[2 * (size_t)NK_STATIC_MAX_LOCAL_DOFS];

namespace {
// device address of nk_static_scratch on the CURRENT device (cached per device ordinal)
nk_status static_scratch(double** out)
{
    enum { kMaxDevices = 64 };
    static std::mutex mu;
    static double* addr[kMaxDevices] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return sfail(NK_ERR_CUDA, std::string("nk_assembled_helmholtz_apply_static: cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return sfail(NK_ERR_UNSUPPORTED, "nk_assembled_helmholtz_apply_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lk(mu);
    if (!addr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, nk_static_scratch);
        if (e != cudaSuccess || !p)
            return sfail(NK_ERR_CUDA, std::string("nk_assembled_helmholtz_apply_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        addr[dev] = p;
    }
    *out = addr[dev];
    return NK_OK;
}
} // namespace

extern "C" int nk_helmholtz_apply_allocates_(const nk_basis* b, const nk_geom* g);   // nk_api.cu

extern "C" int64_t nk_static_max_local_dofs(void) { return (int64_t)NK_STATIC_MAX_LOCAL_DOFS; }

extern "C" nk_status nk_assembled_helmholtz_apply_static(const nk_basis* b, const nk_geom* g, const nk_gs* gs, double lambda, const double* in,
                                                         double* out, void* stream)
{
    const char* me = "nk_assembled_helmholtz_apply_static";
    if (!b || !g || !gs || !in || !out) return sfail(NK_ERR_INVALID_ARG, std::string(me) + ": NULL argument");
    if (gs->nelem != nk_geom_num_elements(g) || gs->nm != nk_basis_num_modes(b))
        return sfail(NK_ERR_SHAPE_MISMATCH, std::string(me) + ": the map does not belong to this block");
    if (in == out) return sfail(NK_ERR_INVALID_ARG, std::string(me) + ": in and out alias");
    if (gs->nlocal > (int64_t)NK_STATIC_MAX_LOCAL_DOFS)
        return sfail(NK_ERR_UNSUPPORTED, std::string(me) + ": " + std::to_string((long long)gs->nlocal) + " local dofs (nelem x Nm) exceed the static work "
                     "space of NK_STATIC_MAX_LOCAL_DOFS = " + std::to_string((long long)NK_STATIC_MAX_LOCAL_DOFS) +
                     "; use nk_assembled_helmholtz_apply (it allocates its work space on first use)");
    if (gs->nglobal == 0) return NK_OK;
    if (nk_helmholtz_apply_allocates_(b, g))
        return sfail(NK_ERR_UNSUPPORTED, std::string(me) + ": the elemental operator of this block would still build device tables (reference-matrix "
                     "form: first use on this basis, or a kernel specialised at run time); call nk_helmholtz_apply once on the block at set-up, "
                     "or select form 1 (nk_set_affine_simplex_form)");
    double* w = nullptr;
    nk_status st = static_scratch(&w);
    if (st != NK_OK) return st;
    double* lin = w;
    double* lout = w + (size_t)NK_STATIC_MAX_LOCAL_DOFS;
    // Nothing in the array has to start at zero: the gather writes lin[0, nlocal), the elemental kernel writes
    // lout[0, nlocal), and nothing beyond nlocal is read; what an earlier call left behind is never seen.
    cudaStream_t s = (cudaStream_t)stream;
    gather_kernel<<<grid_for(gs->nlocal), 256, 0, s>>>(gs->d_l2g, gs->d_sgn, gs->d_free, in, lin, gs->nlocal);
    st = nk_helmholtz_apply(b, g, lambda, lin, lout, stream);
    if (st != NK_OK) return st;
    scatter_kernel<<<grid_for(gs->nglobal), 256, 0, s>>>(gs->d_rowptr, gs->d_col, gs->d_sgn, lout, out, gs->nglobal, gs->d_free, in);
    nk_count_launches_(2);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? NK_OK : sfail(NK_ERR_CUDA, std::string(me) + ": " + cudaGetErrorString(e));
}
