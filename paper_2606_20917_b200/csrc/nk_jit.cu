// nk_jit.cu -- run-time specialisation of both kernel families with NVRTC.
//
// The paper generates and JIT-compiles one kernel per (shape, P, Q) at run time and reports "< 1 second" for it
// (P:27-29).  This library instantiates its kernels ahead of time for Q = P+2; what falls outside that table is
// specialised at run time from the SAME sources, embedded in the library at build time:
//   * the reference-matrix kernels depend on ONE number, the modes per element Nm: csrc/nk_dense.cuh is compiled for an
//     Nm outside the prebuilt table (prisms, hexes of order >= 2, ... when nk_set_affine_simplex_form(2) asks for the
//     reference-matrix form there), cached per (device, Nm, operator);
//   * the sum-factorised kernel template nk_kernel<shape, P, deformed, op, Q> (nk_kernel_body.cuh and its stage files) is
//     compiled for a (shape, P, Q) outside the table -- any P+1 <= Q <= 12, tets and prisms of order 9 and 10 -- one
//     instantiation per first use, cached per (device, shape, P, Q, deformed, operator); second half of this file.
// Cubins are loaded through the driver API.
// libnvrtc and libcuda are opened with dlopen: libnk.so has no link-time dependency on either, loads on a machine
// without a driver, and nk_jit_compile_check() compiles without a GPU.
#include <dlfcn.h>

#include <chrono>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <tuple>
#include <utility>
#include <vector>

#include <cuda.h>
#include <nvrtc.h>

#include "nk_dense_launch.h"
#include "nk_launch.h"

namespace nk {
namespace {

// the text of csrc/nk_dense.cuh, embedded at build time (paper_2606_20917_b200/build.py writes build/nk_dense_src.inc)
const char kDenseSource[] =
#include "nk_dense_src.inc"
    ;
// the sum-factorised kernel template: nk_kernels.cuh, nk_kernel_body.cuh and the nk_stage_*.inc files it includes, each
// as {name, text} (build/nk_sumfac_src.inc); NVRTC resolves the #include lines from this list
struct SrcFile {
    const char *name, *text;
};
const SrcFile kSumfacSources[] = {
#include "nk_sumfac_src.inc"
};

struct Api {
    void *rtc = nullptr, *drv = nullptr;
    decltype(&nvrtcCreateProgram) CreateProgram = nullptr;
    decltype(&nvrtcDestroyProgram) DestroyProgram = nullptr;
    decltype(&nvrtcCompileProgram) CompileProgram = nullptr;
    decltype(&nvrtcGetProgramLogSize) GetProgramLogSize = nullptr;
    decltype(&nvrtcGetProgramLog) GetProgramLog = nullptr;
    decltype(&nvrtcAddNameExpression) AddNameExpression = nullptr;
    decltype(&nvrtcGetLoweredName) GetLoweredName = nullptr;
    decltype(&nvrtcGetCUBINSize) GetCUBINSize = nullptr;
    decltype(&nvrtcGetCUBIN) GetCUBIN = nullptr;
    decltype(&cuModuleLoadData) ModuleLoadData = nullptr;
    decltype(&cuModuleGetFunction) ModuleGetFunction = nullptr;
    decltype(&cuFuncSetAttribute) FuncSetAttribute = nullptr;
    decltype(&cuOccupancyMaxActiveBlocksPerMultiprocessor) Occupancy = nullptr;
    decltype(&cuLaunchKernel) LaunchKernel = nullptr;
    decltype(&cuGetErrorString) GetErrorString = nullptr;
    std::string why;
};

template <class F>
bool sym(void* lib, const char* name, F& f)
{
    f = reinterpret_cast<F>(dlsym(lib, name));
    return f != nullptr;
}

std::mutex g_mu;
Api g_api;
bool g_rtc_tried = false, g_drv_tried = false;
long long g_compiled = 0;
double g_compile_ms = 0.0;

bool load_rtc(std::string* err)
{
    if (!g_rtc_tried) {
        g_rtc_tried = true;
        for (const char* n : {"libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so"}) {
            g_api.rtc = dlopen(n, RTLD_NOW | RTLD_LOCAL);
            if (g_api.rtc) break;
        }
        Api& a = g_api;
        if (!a.rtc) {
            a.why = "libnvrtc not found (dlopen)";
        } else if (!(sym(a.rtc, "nvrtcCreateProgram", a.CreateProgram) && sym(a.rtc, "nvrtcDestroyProgram", a.DestroyProgram) &&
                     sym(a.rtc, "nvrtcCompileProgram", a.CompileProgram) && sym(a.rtc, "nvrtcGetProgramLogSize", a.GetProgramLogSize) &&
                     sym(a.rtc, "nvrtcGetProgramLog", a.GetProgramLog) && sym(a.rtc, "nvrtcAddNameExpression", a.AddNameExpression) &&
                     sym(a.rtc, "nvrtcGetLoweredName", a.GetLoweredName) && sym(a.rtc, "nvrtcGetCUBINSize", a.GetCUBINSize) &&
                     sym(a.rtc, "nvrtcGetCUBIN", a.GetCUBIN))) {
            a.why = "libnvrtc lacks an entry point";
            a.rtc = nullptr;
        }
    }
    if (!g_api.rtc && err) *err = g_api.why;
    return g_api.rtc != nullptr;
}

bool load_drv(std::string* err)
{
    if (!g_drv_tried) {
        g_drv_tried = true;
        Api& a = g_api;
        a.drv = dlopen("libcuda.so.1", RTLD_NOW | RTLD_LOCAL);
        if (!a.drv) {
            a.why = "libcuda.so.1 not found (no driver on this machine)";
        } else if (!(sym(a.drv, "cuModuleLoadData", a.ModuleLoadData) && sym(a.drv, "cuModuleGetFunction", a.ModuleGetFunction) &&
                     sym(a.drv, "cuFuncSetAttribute", a.FuncSetAttribute) &&
                     sym(a.drv, "cuOccupancyMaxActiveBlocksPerMultiprocessor", a.Occupancy) &&
                     sym(a.drv, "cuLaunchKernel", a.LaunchKernel) && sym(a.drv, "cuGetErrorString", a.GetErrorString))) {
            a.why = "libcuda lacks an entry point";
            a.drv = nullptr;
        }
    }
    if (!g_api.drv && err) *err = g_api.why;
    return g_api.drv != nullptr;
}

// launch configuration of a run-time specialisation, chosen by the rules the prebuilt table was tuned to
struct Plan {
    bool streamed = false;
    int warps = 0, minb = 1, ksc = 1, stages = 2;
    size_t smem = 0;
    int threads = 0;
    std::string name;   // name expression of the instantiation
};

Plan make_plan(int nm, int c0, int nc)
{
    Plan p;
    const int NK = (nm + 3) / 4, NTF = nm / 8, R = nm % 8;
    const bool REM = (R > 0 && R < nc);
    const int NTS = NTF + ((R > 0 && !REM) ? 1 : 0), NRT = REM ? R : 0;
    const size_t resident = dense_pack_size(nm, nc) * sizeof(double);
    char buf[160];
    if (resident <= (size_t)176 * 1024) {
        p.warps = nm >= 32 ? 16 : 8;
        const size_t per_block = resident + 1024;
        int byshm = (int)((size_t)220 * 1024 / per_block);
        p.minb = p.warps == 16 ? 1 : (byshm < 1 ? 1 : byshm > 4 ? 4 : byshm);
        p.smem = resident;
        p.threads = p.warps * 32;
        snprintf(buf, sizeof buf, "nk::nk_dense_kernel<%d, %d, %d, %d, %d>", nm, c0, nc, p.warps, p.minb);
    } else {
        p.streamed = true;
        p.warps = 4;
        p.stages = 2;
        const int widest = NTS > NRT ? NTS : NRT;
        p.ksc = 1;
        for (int k = 1; k <= NK; ++k)
            if (NK % k == 0 && (size_t)k * widest * 256 <= (size_t)32 * 1024) p.ksc = k;
        const size_t stage = (size_t)p.ksc * widest * 32 * sizeof(double);
        const int ustride = (4 * NK) % 8 == 4 ? 4 * NK : 4 * NK + 4;
        const size_t slab = (size_t)(8 * ustride + 64) * sizeof(double);
        p.smem = p.stages * stage + p.warps * slab + 2 * p.stages * sizeof(unsigned long long);
        p.minb = 2 * (p.smem + 1024) <= (size_t)227 * 1024 ? 2 : 1;
        p.threads = (p.warps + 1) * 32;
        snprintf(buf, sizeof buf, "nk::nk_dense_stream_kernel<%d, %d, %d, %d, %d, %d, %d>", nm, c0, nc, p.warps, p.ksc, p.stages, p.minb);
    }
    p.name = buf;
    return p;
}

// NVRTC: source (+ headers) -> cubin of ONE instantiation, named by the expression `name`; needs no device
bool compile_source(const char* src, const char* src_name, int nheaders, const char* const* header_text,
                    const char* const* header_names, const std::string& name, std::vector<char>& cubin, std::string& lowered,
                    double& ms, std::string& err)
{
    if (!load_rtc(&err)) return false;
    Api& a = g_api;
    const auto t0 = std::chrono::steady_clock::now();
    nvrtcProgram prog = nullptr;
    if (a.CreateProgram(&prog, src, src_name, nheaders, header_text, header_names) != NVRTC_SUCCESS) {
        err = "nvrtcCreateProgram failed";
        return false;
    }
    bool ok = a.AddNameExpression(prog, name.c_str()) == NVRTC_SUCCESS;
    // -default-device: lambdas and helpers without an execution-space annotation are device functions (as under nvcc)
    const char* opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "-default-device"};
    nvrtcResult r = ok ? a.CompileProgram(prog, 4, opts) : NVRTC_ERROR_INVALID_INPUT;
    if (r != NVRTC_SUCCESS) {
        size_t n = 0;
        a.GetProgramLogSize(prog, &n);
        std::string log(n, '\0');
        if (n) a.GetProgramLog(prog, &log[0]);
        err = "NVRTC could not compile " + name + ": " + log.substr(0, 600);
        a.DestroyProgram(&prog);
        return false;
    }
    const char* ln = nullptr;
    size_t nb = 0;
    ok = a.GetLoweredName(prog, name.c_str(), &ln) == NVRTC_SUCCESS && ln && a.GetCUBINSize(prog, &nb) == NVRTC_SUCCESS && nb > 0;
    if (ok) {
        lowered = ln;
        cubin.resize(nb);
        ok = a.GetCUBIN(prog, cubin.data()) == NVRTC_SUCCESS;
    }
    a.DestroyProgram(&prog);
    ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    if (!ok) err = "NVRTC produced no cubin for " + name;
    return ok;
}
bool compile(const Plan& p, std::vector<char>& cubin, std::string& lowered, double& ms, std::string& err)
{
    return compile_source(kDenseSource, "nk_dense.cuh", 0, nullptr, nullptr, p.name, cubin, lowered, ms, err);
}

struct Loaded {
    CUfunction fn = nullptr;
    Plan plan;
    int blocks_per_sm = 1, sms = 0;
};
std::map<std::tuple<int, int, int>, Loaded> g_cache;   // (device, Nm, kind)

std::string drv_error(CUresult r)
{
    const char* s = nullptr;
    if (g_api.GetErrorString) g_api.GetErrorString(r, &s);
    return s ? s : "unknown driver error";
}

} // namespace

bool dense_jit_compile_check(int nmodes, int kind, double* ms, size_t* cubin_bytes, std::string* err)
{
    std::lock_guard<std::mutex> lk(g_mu);
    const Plan p = make_plan(nmodes, dense_c0(kind), dense_nc(kind));
    std::vector<char> cubin;
    std::string lowered, e;
    double t = 0.0;
    if (!compile(p, cubin, lowered, t, e)) {
        if (err) *err = e;
        return false;
    }
    if (ms) *ms = t;
    if (cubin_bytes) *cubin_bytes = cubin.size();
    return true;
}

void dense_jit_stats(long long* kernels, double* total_ms)
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (kernels) *kernels = g_compiled;
    if (total_ms) *total_ms = g_compile_ms;
}

bool dense_jit_launch(int nmodes, int kind, const DenseArgs& a, cudaStream_t stream, int* launched, std::string* err)
{
    *launched = 0;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaFree(nullptr) != cudaSuccess) {   // the primary context must exist and be current
        *err = "no CUDA device";
        return false;
    }
    std::lock_guard<std::mutex> lk(g_mu);
    const auto key = std::make_tuple(dev, nmodes, kind);
    auto it = g_cache.find(key);
    if (it == g_cache.end()) {
        if (!load_drv(err)) return false;
        Loaded L;
        L.plan = make_plan(nmodes, dense_c0(kind), dense_nc(kind));
        std::vector<char> cubin;
        std::string lowered;
        double ms = 0.0;
        if (!compile(L.plan, cubin, lowered, ms, *err)) return false;
        CUmodule mod = nullptr;
        CUresult r = g_api.ModuleLoadData(&mod, cubin.data());
        if (r == CUDA_SUCCESS) r = g_api.ModuleGetFunction(&L.fn, mod, lowered.c_str());
        if (r == CUDA_SUCCESS) r = g_api.FuncSetAttribute(L.fn, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)L.plan.smem);
        if (r == CUDA_SUCCESS) r = g_api.FuncSetAttribute(L.fn, CU_FUNC_ATTRIBUTE_PREFERRED_SHARED_MEMORY_CARVEOUT, 100);
        int bps = 0;
        if (r == CUDA_SUCCESS) r = g_api.Occupancy(&bps, L.fn, L.plan.threads, L.plan.smem);
        if (r != CUDA_SUCCESS) {
            *err = "loading the run-time kernel " + L.plan.name + ": " + drv_error(r);
            return false;
        }
        L.blocks_per_sm = bps < 1 ? 1 : bps;
        if (cudaDeviceGetAttribute(&L.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || L.sms < 1) L.sms = 1;
        g_compiled += 1;
        g_compile_ms += ms;
        it = g_cache.emplace(key, L).first;
    }
    const Loaded& L = it->second;
    if (a.e1 <= a.e0 || a.nfields < 1) return true;
    const long long per_tile = L.plan.streamed ? 8LL * L.plan.warps : 8LL;
    const long long ntiles = ((a.e1 - a.e0 + per_tile - 1) / per_tile) * a.nfields;
    if (ntiles >= 0x7fffffffLL) {
        *err = "too many tiles";
        return false;
    }
    long long grid = (long long)L.sms * L.blocks_per_sm;
    const long long need = L.plan.streamed ? ntiles : (ntiles + L.plan.warps - 1) / L.plan.warps;
    if (grid > need) grid = need;
    DenseArgs args = a;
    void* params[] = {&args};
    const CUresult r = g_api.LaunchKernel(L.fn, (unsigned)grid, 1, 1, (unsigned)L.plan.threads, 1, 1, (unsigned)L.plan.smem, (CUstream)stream,
                                          params, nullptr);
    if (r != CUDA_SUCCESS) {
        *err = "launching " + L.plan.name + ": " + drv_error(r);
        return false;
    }
    *launched = 1;
    return true;
}


// =====================================================================================================================
// Sum-factorised kernels (nk_kernel_body.cuh) for a (shape, P, Q) outside the prebuilt table: tets / prisms of order 9 and 10,
// any Q != P+2 (P+1 <= Q <= 12).  The kernel template takes Q as a parameter and its launch rules (Tune / TuneOp) are
// functions of Q, so the host reads the configuration of any triple from the same templates (table below, no GPU needed)
// and NVRTC instantiates exactly one nk_kernel<shape, P, deformed, op, Q> per first use.
// =====================================================================================================================
namespace {

template <int SHAPE, int P, int Q, int DEF, int... OPS>
void fill_ops(JitInfo& o, std::integer_sequence<int, OPS...>)
{
    ((o.op[DEF][OPS] = JitOpCfg{TuneOp<SHAPE, P, DEF, OPS, Q>::E, TuneOp<SHAPE, P, DEF, OPS, Q>::NT, TuneOp<SHAPE, P, DEF, OPS, Q>::MINB,
                                (size_t)TuneOp<SHAPE, P, DEF, OPS, Q>::smem_grid}),
     ...);
}
template <int SHAPE, int P, int Q>
void fill_info(JitInfo& o)
{
    o.shape = SHAPE;
    o.P = P;
    o.Q = Q;
    o.E[0] = Tune<SHAPE, P, 0, Q>::E;
    o.E[1] = Tune<SHAPE, P, 1, Q>::E;
    fill_ops<SHAPE, P, Q, 0>(o, std::make_integer_sequence<int, OP_COUNT>{});
    fill_ops<SHAPE, P, Q, 1>(o, std::make_integer_sequence<int, OP_COUNT>{});
    o.tabs_bytes = sizeof(DenseTabs<P + 1, Q, SHAPE == K_HEX>);
    o.sx_bytes = sizeof(typename SimplexTabsFor<SHAPE, P + 1, Q>::type);
    o.sx_dup = k_sx_dup(SHAPE, P + 1, Q);
    static_assert(sizeof(DenseTabs<P + 1, Q, SHAPE == K_HEX>) == sizeof(double) * k_dense_doubles(P + 1, Q, SHAPE == K_HEX), "k_dense_doubles out of date");
}
// Q = P+1 .. kJitMaxQ
template <int SHAPE, int P, int... DQ>
bool pick_q(int Q, JitInfo& o, std::integer_sequence<int, DQ...>)
{
    return ((Q == P + 1 + DQ ? (fill_info<SHAPE, P, P + 1 + DQ>(o), true) : false) || ...);
}
template <int SHAPE, int... PM1>
bool pick_p(int P, int Q, JitInfo& o, std::integer_sequence<int, PM1...>)
{
    return ((P == PM1 + 1 ? pick_q<SHAPE, PM1 + 1>(Q, o, std::make_integer_sequence<int, kJitMaxQ - PM1 - 1>{}) : false) || ...);
}

struct SumfacLoaded {
    CUfunction fn = nullptr;
    int blocks_per_sm = 1;
};
std::map<std::tuple<int, int, int, int, int, int>, SumfacLoaded> g_sumfac_cache;   // (device, shape, P, Q, def, op)

std::string sumfac_name(int shape, int P, int Q, int def, int op)
{
    char buf[96];
    snprintf(buf, sizeof buf, "nk::nk_kernel<%d, %d, %d, %d, %d>", shape, P, def, op, Q);
    return buf;
}
bool sumfac_compile(const std::string& name, std::vector<char>& cubin, std::string& lowered, double& ms, std::string& err)
{
    constexpr int N = (int)(sizeof(kSumfacSources) / sizeof(kSumfacSources[0]));
    const char *text[N], *names[N];
    for (int i = 0; i < N; ++i) {
        text[i] = kSumfacSources[i].text;
        names[i] = kSumfacSources[i].name;
    }
    return compile_source("#include \"nk_kernel_body.cuh\"\n", "nk_jit_sumfac.cu", N, text, names, name, cubin, lowered, ms, err);
}

} // namespace

bool sumfac_jit_info(int shape, int P, int Q, JitInfo* out, std::string* why)
{
    JitInfo o;
    std::memset(&o, 0, sizeof o);
    bool ok = false;
    if (P >= 1 && P <= kJitMaxP && Q >= P + 1 && Q <= kJitMaxQ) {
        const auto ps = std::make_integer_sequence<int, kJitMaxP>{};
        ok = shape == K_HEX ? pick_p<K_HEX>(P, Q, o, ps) : shape == K_TET ? pick_p<K_TET>(P, Q, o, ps) : shape == K_PRISM ? pick_p<K_PRISM>(P, Q, o, ps) : false;
    }
    if (!ok) {
        if (why) *why = "run-time specialisation covers 1 <= P <= 10 and P+1 <= Q <= 12";
        return false;
    }
    if (o.tabs_bytes + o.sx_bytes + sizeof(KArgs) > 32000) {
        if (why) *why = "the basis tables of this (shape, P, Q) exceed the 32 KB kernel-parameter space";
        return false;
    }
    for (int d = 0; d < 2; ++d)
        for (int k = 0; k < OP_COUNT; ++k)
            if (o.op[d][k].smem > (size_t)227 * 1024 || o.op[d][k].threads > 1024) {
                if (why) *why = "this (shape, P, Q) needs more shared memory or threads than a block can have";
                return false;
            }
    if (out) *out = o;
    return true;
}

bool sumfac_jit_compile_check(int shape, int P, int Q, int def, int op, double* ms, size_t* cubin_bytes, std::string* err)
{
    std::string e;
    JitInfo info;
    if (def < 0 || def > 1 || op < 0 || op >= OP_COUNT || !sumfac_jit_info(shape, P, Q, &info, &e)) {
        if (err) *err = e.empty() ? "bad deformed flag / operator" : e;
        return false;
    }
    std::lock_guard<std::mutex> lk(g_mu);
    std::vector<char> cubin;
    std::string lowered;
    double t = 0.0;
    if (!sumfac_compile(sumfac_name(shape, P, Q, def, op), cubin, lowered, t, e)) {
        if (err) *err = e;
        return false;
    }
    if (ms) *ms = t;
    if (cubin_bytes) *cubin_bytes = cubin.size();
    return true;
}

bool sumfac_jit_launch(const JitInfo& info, int def, int op, const double* tabs_flat, const double* sx_flat, const KArgs& a, int num_sms,
                       cudaStream_t stream, std::string* err)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaFree(nullptr) != cudaSuccess) {   // the primary context must exist and be current
        *err = "no CUDA device";
        return false;
    }
    const JitOpCfg& cfg = info.op[def][op];
    std::lock_guard<std::mutex> lk(g_mu);
    const auto key = std::make_tuple(dev, info.shape, info.P, info.Q, def, op);
    auto it = g_sumfac_cache.find(key);
    if (it == g_sumfac_cache.end()) {
        if (!load_drv(err)) return false;
        const std::string name = sumfac_name(info.shape, info.P, info.Q, def, op);
        std::vector<char> cubin;
        std::string lowered;
        double ms = 0.0;
        if (!sumfac_compile(name, cubin, lowered, ms, *err)) return false;
        SumfacLoaded L;
        CUmodule mod = nullptr;
        CUresult r = g_api.ModuleLoadData(&mod, cubin.data());
        if (r == CUDA_SUCCESS) r = g_api.ModuleGetFunction(&L.fn, mod, lowered.c_str());
        if (r == CUDA_SUCCESS) r = g_api.FuncSetAttribute(L.fn, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)cfg.smem);
        if (r == CUDA_SUCCESS) r = g_api.FuncSetAttribute(L.fn, CU_FUNC_ATTRIBUTE_PREFERRED_SHARED_MEMORY_CARVEOUT, 100);
        int bps = 0;
        if (r == CUDA_SUCCESS) r = g_api.Occupancy(&bps, L.fn, cfg.threads, cfg.smem);
        if (r != CUDA_SUCCESS) {
            *err = "loading the run-time kernel " + name + ": " + drv_error(r);
            return false;
        }
        L.blocks_per_sm = bps < 1 ? 1 : bps;
        g_compiled += 1;
        g_compile_ms += ms;
        it = g_sumfac_cache.emplace(key, L).first;
    }
    const SumfacLoaded& L = it->second;
    if (a.grid_groups <= 0) return true;
    KArgs b = a;
    // L2 prefetch distance: the rule of the prebuilt kernels (nk_inst.cu)
    b.pf_dist = (int)((long long)num_sms * L.blocks_per_sm * (L.blocks_per_sm == 1 ? 2 : 12) / 100) + 1;
    const long long units = (long long)a.grid_groups * (a.nfields > 1 ? a.nfields : 1);
    if (units > 0x7fffffffLL) {
        *err = "too many groups";
        return false;
    }
    // kernel parameters: DenseTabs and SimplexTabs are the flat tables themselves (all doubles, declaration order)
    static const double no_sx[4] = {0.0, 0.0, 0.0, 0.0};
    void* params[] = {const_cast<double*>(tabs_flat), const_cast<double*>(info.shape == K_HEX ? no_sx : sx_flat), &b};
    const CUresult r = g_api.LaunchKernel(L.fn, (unsigned)units, 1, 1, (unsigned)cfg.threads, 1, 1, (unsigned)cfg.smem, (CUstream)stream, params, nullptr);
    if (r != CUDA_SUCCESS) {
        *err = "launching " + sumfac_name(info.shape, info.P, info.Q, def, op) + ": " + drv_error(r);
        return false;
    }
    return true;
}

} // namespace nk
