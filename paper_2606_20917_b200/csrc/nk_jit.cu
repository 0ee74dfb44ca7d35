// nk_jit.cu -- run-time specialisation of the reference-matrix kernels with NVRTC (first part).
//
// The paper generates and JIT-compiles one kernel per (shape, P, Q) at run time and reports "< 1 second" for it
// (P:27-29).  This library instantiates its kernels ahead of time; what it specialises at run time is the
// kernel family that depends on ONE number, the modes per element Nm: csrc/nk_dense.cuh is compiled by NVRTC for an Nm
// outside the prebuilt table (prisms, hexes of order >= 2, ... when nk_set_affine_simplex_form(2) asks for the
// reference-matrix form there), loaded through the driver API and cached per (device, Nm, operator).
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
#include <vector>

#include <cuda.h>
#include <nvrtc.h>

#include "nk_dense_launch.h"

namespace nk {
namespace {

// the text of csrc/nk_dense.cuh, embedded at build time (paper_2606_20917_b200/build.py writes build/nk_dense_src.inc)
const char kDenseSource[] =
#include "nk_dense_src.inc"
    ;

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

// NVRTC: source -> cubin of ONE instantiation; needs no device
bool compile(const Plan& p, std::vector<char>& cubin, std::string& lowered, double& ms, std::string& err)
{
    if (!load_rtc(&err)) return false;
    Api& a = g_api;
    const auto t0 = std::chrono::steady_clock::now();
    nvrtcProgram prog = nullptr;
    if (a.CreateProgram(&prog, kDenseSource, "nk_dense.cuh", 0, nullptr, nullptr) != NVRTC_SUCCESS) {
        err = "nvrtcCreateProgram failed";
        return false;
    }
    bool ok = a.AddNameExpression(prog, p.name.c_str()) == NVRTC_SUCCESS;
    const char* opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo"};
    nvrtcResult r = ok ? a.CompileProgram(prog, 3, opts) : NVRTC_ERROR_INVALID_INPUT;
    if (r != NVRTC_SUCCESS) {
        size_t n = 0;
        a.GetProgramLogSize(prog, &n);
        std::string log(n, '\0');
        if (n) a.GetProgramLog(prog, &log[0]);
        err = "NVRTC could not compile " + p.name + ": " + log.substr(0, 600);
        a.DestroyProgram(&prog);
        return false;
    }
    const char* ln = nullptr;
    size_t nb = 0;
    ok = a.GetLoweredName(prog, p.name.c_str(), &ln) == NVRTC_SUCCESS && ln && a.GetCUBINSize(prog, &nb) == NVRTC_SUCCESS && nb > 0;
    if (ok) {
        lowered = ln;
        cubin.resize(nb);
        ok = a.GetCUBIN(prog, cubin.data()) == NVRTC_SUCCESS;
    }
    a.DestroyProgram(&prog);
    ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    if (!ok) err = "NVRTC produced no cubin for " + p.name;
    return ok;
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

} // namespace nk
