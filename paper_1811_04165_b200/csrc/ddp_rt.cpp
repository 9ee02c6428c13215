// CUDA side of libddp: driver/NVRTC loading, kernel compilation + caching, launches of the four
// kernels, workspace binding and the CUDA-event timing harness (fitness function of the tuners).
//
// libcuda and libnvrtc are dlopen'ed on first use so that the library loads (and its host-only
// entry points work) on a machine without a GPU; every compute / hardware-tune call then returns
// DDP_E_CUDA -- there is no CPU fallback (BJ:north_star).
//
// Kernels come from ONE parameterised template each (ddp_kernels.cuh).  A configuration's code
// shape (samples/DMs per thread, unroll, staging, vector width, max threads) is instantiated either
// ahead of time (ddp_aot.cubin built by nvcc, looked up by name) or at tune time by NVRTC from the
// template text embedded in this library; cubins are cached in memory and optionally on disk.
#include <cuda.h>
#include <dlfcn.h>
#include <nvrtc.h>
#include <unistd.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <thread>

#include "ddp_internal.h"

extern const char* const ddp_kernel_source;  // generated: ddp_params.h + ddp_kernels.cuh as one string

#define DDP_MAX_DEVICES 16
#define DDP_STR2(x) #x
#define DDP_STR(x) DDP_STR2(x)

// ------------------------------------------------------------------------------------ dynamic API
namespace {
struct Api {
    bool tried = false, ok = false;
    std::string why;
    void* hcuda = nullptr;
    void* hnvrtc = nullptr;
#define DRV(name) decltype(&name) p_##name = nullptr;
    DRV(cuInit)
    DRV(cuDeviceGet)
    DRV(cuDeviceGetCount)
    DRV(cuDeviceGetAttribute)
    DRV(cuDevicePrimaryCtxRetain)
    DRV(cuCtxGetCurrent)
    DRV(cuCtxSetCurrent)
    DRV(cuModuleLoadData)
    DRV(cuModuleUnload)
    DRV(cuModuleGetFunction)
    DRV(cuFuncSetAttribute)
    DRV(cuFuncGetAttribute)
    DRV(cuLaunchKernel)
    DRV(cuMemcpyHtoDAsync)
    DRV(cuMemcpyDtoHAsync)
    DRV(cuMemsetD32Async)
    DRV(cuEventCreate)
    DRV(cuEventRecord)
    DRV(cuEventSynchronize)
    DRV(cuEventElapsedTime)
    DRV(cuEventDestroy)
    DRV(cuStreamSynchronize)
    DRV(cuGetErrorString)
    DRV(cuOccupancyMaxActiveBlocksPerMultiprocessor)
    DRV(cuMemcpy2DAsync)
    DRV(cuStreamCreate)
    DRV(cuStreamDestroy)
    DRV(cuStreamWaitEvent)
#undef DRV
#define RTC(name) decltype(&name) p_##name = nullptr;
    RTC(nvrtcCreateProgram)
    RTC(nvrtcCompileProgram)
    RTC(nvrtcGetCUBINSize)
    RTC(nvrtcGetCUBIN)
    RTC(nvrtcGetProgramLogSize)
    RTC(nvrtcGetProgramLog)
    RTC(nvrtcDestroyProgram)
    RTC(nvrtcGetErrorString)
#undef RTC
    bool nvrtc_ok = false;
    CUcontext ctx[DDP_MAX_DEVICES] = {nullptr};
    bool inited = false;
};
Api g_api;
std::mutex g_api_mu;

bool load_nvrtc_locked() {
    if (g_api.nvrtc_ok) return true;
    if (g_api.hnvrtc == nullptr) {
        const char* names[] = {"libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so"};
        for (const char* n : names) {
            g_api.hnvrtc = dlopen(n, RTLD_NOW | RTLD_LOCAL);
            if (g_api.hnvrtc) break;
        }
        if (!g_api.hnvrtc) return false;
    }
    bool ok = true;
#define RTC(name)                                                                   \
    g_api.p_##name = (decltype(&name))dlsym(g_api.hnvrtc, DDP_STR(name));           \
    ok = ok && g_api.p_##name != nullptr;
    RTC(nvrtcCreateProgram)
    RTC(nvrtcCompileProgram)
    RTC(nvrtcGetCUBINSize)
    RTC(nvrtcGetCUBIN)
    RTC(nvrtcGetProgramLogSize)
    RTC(nvrtcGetProgramLog)
    RTC(nvrtcDestroyProgram)
    RTC(nvrtcGetErrorString)
#undef RTC
    g_api.nvrtc_ok = ok;
    return ok;
}

// Loads libcuda and initialises the driver; false (with g_api.why) when there is no usable GPU.
bool load_cuda_locked() {
    if (g_api.tried) return g_api.ok;
    g_api.tried = true;
    g_api.hcuda = dlopen("libcuda.so.1", RTLD_NOW | RTLD_LOCAL);
    if (!g_api.hcuda) {
        g_api.why = "libcuda.so.1 not found (no NVIDIA driver on this machine)";
        return false;
    }
    bool ok = true;
#define DRV(name)                                                                  \
    g_api.p_##name = (decltype(&name))dlsym(g_api.hcuda, DDP_STR(name));            \
    ok = ok && g_api.p_##name != nullptr;
    DRV(cuInit)
    DRV(cuDeviceGet)
    DRV(cuDeviceGetCount)
    DRV(cuDeviceGetAttribute)
    DRV(cuDevicePrimaryCtxRetain)
    DRV(cuCtxGetCurrent)
    DRV(cuCtxSetCurrent)
    DRV(cuModuleLoadData)
    DRV(cuModuleUnload)
    DRV(cuModuleGetFunction)
    DRV(cuFuncSetAttribute)
    DRV(cuFuncGetAttribute)
    DRV(cuLaunchKernel)
    DRV(cuMemcpyHtoDAsync)
    DRV(cuMemcpyDtoHAsync)
    DRV(cuMemsetD32Async)
    DRV(cuEventCreate)
    DRV(cuEventRecord)
    DRV(cuEventSynchronize)
    DRV(cuEventElapsedTime)
    DRV(cuEventDestroy)
    DRV(cuStreamSynchronize)
    DRV(cuGetErrorString)
    DRV(cuOccupancyMaxActiveBlocksPerMultiprocessor)
    DRV(cuMemcpy2DAsync)
    DRV(cuStreamCreate)
    DRV(cuStreamDestroy)
    DRV(cuStreamWaitEvent)
#undef DRV
    if (!ok) {
        g_api.why = "libcuda.so.1 lacks a required driver entry point";
        return false;
    }
    if (g_api.p_cuInit(0) != CUDA_SUCCESS) {
        g_api.why = "cuInit failed (no CUDA device)";
        return false;
    }
    int n = 0;
    if (g_api.p_cuDeviceGetCount(&n) != CUDA_SUCCESS || n <= 0) {
        g_api.why = "no CUDA device";
        return false;
    }
    g_api.ok = true;
    return true;
}

std::string cu_err(CUresult r) {
    const char* s = nullptr;
    if (g_api.p_cuGetErrorString && g_api.p_cuGetErrorString(r, &s) == CUDA_SUCCESS && s) return s;
    return "CUDA error " + std::to_string((int)r);
}

// Makes the primary context of `device` current on the calling thread (the one torch uses).
ddp_status ensure_ctx(const ddp_plan* p, int device) {
    std::lock_guard<std::mutex> lk(g_api_mu);
    if (!load_cuda_locked()) return ddp_fail(p, DDP_E_CUDA, g_api.why);
    if (device < 0 || device >= DDP_MAX_DEVICES) return ddp_fail(p, DDP_E_ARG, "device ordinal out of range");
    if (!g_api.ctx[device]) {
        CUdevice dev;
        CUresult r = g_api.p_cuDeviceGet(&dev, device);
        if (r != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, "cuDeviceGet: " + cu_err(r));
        r = g_api.p_cuDevicePrimaryCtxRetain(&g_api.ctx[device], dev);
        if (r != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, "cuDevicePrimaryCtxRetain: " + cu_err(r));
    }
    CUcontext cur = nullptr;
    g_api.p_cuCtxGetCurrent(&cur);
    if (cur != g_api.ctx[device]) {
        CUresult r = g_api.p_cuCtxSetCurrent(g_api.ctx[device]);
        if (r != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, "cuCtxSetCurrent: " + cu_err(r));
    }
    return DDP_OK;
}
}  // namespace

// ------------------------------------------------------------------------------------ kernel registry
struct DdpCompiled {
    std::string name;
    std::vector<char> cubin;  // device image (from NVRTC or the disk cache); empty for AOT functions
    bool aot = false;         // function of ddp_aot.cubin (looked up per device in the AOT module)
    // A CUmodule / CUfunction belongs to the context that loaded it: one slot per device ordinal.
    CUmodule mod[DDP_MAX_DEVICES] = {nullptr};
    CUfunction fn[DDP_MAX_DEVICES] = {nullptr};
    bool loaded[DDP_MAX_DEVICES] = {false};
    int smem_opt_in[DDP_MAX_DEVICES];  // largest dynamic shared size already granted by cuFuncSetAttribute
    bool failed = false;
    std::string log;
    int regs = 0;
    DdpCompiled() {
        for (int d = 0; d < DDP_MAX_DEVICES; ++d) smem_opt_in[d] = -1;
    }
};

namespace {
std::mutex g_reg_mu;
std::unordered_map<std::string, DdpCompiled*> g_reg;
std::atomic<int64_t> g_ncompiles{0};
std::mutex g_load_mu;  // serialises module loads and the per-device AOT initialisation
CUmodule g_aot_mod[DDP_MAX_DEVICES] = {nullptr};
bool g_aot_tried[DDP_MAX_DEVICES] = {false};

enum CodeKind { CK_DEDISP_U8 = 0, CK_DEDISP_U32 = 1, CK_INTEG = 2, CK_SNR = 3, CK_DEDISP_U16 = 4, CK_ISNR = 5 };
CodeKind code_kind(const ddp_plan* p, ddp_kernel k) {
    switch (k) {
        case DDP_K_DIRECT:
        case DDP_K_SUB1: return p->in_bytes == 2 ? CK_DEDISP_U16 : CK_DEDISP_U8;  // INPUT_BITS = 16: the uint16 code shapes
        case DDP_K_SUB2: return p->info.sub_elem_bytes == 2 ? CK_DEDISP_U16 : CK_DEDISP_U32;
        case DDP_K_INTEGRATE: return CK_INTEG;
        case DDP_K_ISNR: return CK_ISNR;
        default: return CK_SNR;
    }
}
bool is_dedisp(CodeKind ck) { return ck == CK_DEDISP_U8 || ck == CK_DEDISP_U32 || ck == CK_DEDISP_U16; }
const char* kind_tag(CodeKind ck) {
    static const char* t[] = {"ddp_dedisp_u8", "ddp_dedisp_u32", "ddp_integ", "ddp_snr", "ddp_dedisp_u16", "ddp_isnr"};
    return t[ck];
}
const char* kind_type(CodeKind ck) { return ck == CK_DEDISP_U8 ? "ddp_u8" : (ck == CK_DEDISP_U16 ? "ddp_u16" : "ddp_u32"); }
// Code-shape flags of the dedispersion template (ddp_kernels.cuh, ddp_dedisp_entry):
//   bit 0  WIDE   the packed uint8 kernel flushes its 16-bit lanes every 256 rows: only when the
//                 reduction is longer than that (direct dedispersion);
//   bit 1  OUT16  subband step 1 writes the narrow (uint16) intermediate;
//   bits 2-3      packed uint16 kernel (step 2): log2 of how many subband words are summed in 16-bit
//                 lanes before they are split, the largest of {1, 2, 4} that cannot overflow;
//   bit 4  SINGLE packed uint8 kernel with one buffer of shifted copies (two do not fit in 227 KB);
//   bit 5  REGSPLIT merged kernel with 512 consumer threads: setmaxnreg hands the producers' spare registers to them;
//   bit 6  DIAG   packed uint8 kernel, subband step 1: time tiles aligned to the input, per-trial output shift.
int code_flags(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    const CodeKind ck = code_kind(p, k);
    int f = 0;
    if (ck == CK_DEDISP_U8 && c.staging != 0 && ddp_kgeom(p, k).nred > 257) f |= 1;  // 257 * 255 = 65535 still fits the lanes
    if (k == DDP_K_SUB1 && p->info.sub_elem_bytes == 2) f |= 2;
    if (ck == CK_DEDISP_U8 && ddp_u8_single_buffered(p, k, c)) f |= 16;
    if (ck == CK_DEDISP_U8 && ddp_merge_group(c) && c.threads_t * c.threads_dm >= 512) f |= 32;  // REGSPLIT
    if (ck == CK_DEDISP_U8 && ddp_sub1_diag(p, k, c)) f |= 64;  // DIAG: input-aligned time tiles, per-trial output shift
    if (ck == CK_DEDISP_U16 && c.staging != 0 && k == DDP_K_SUB2) {  // uint16 INPUT samples can be 65535: no lane sums there
        const int64_t room = 65535 / (255 * (int64_t)p->cps);
        f |= (room >= 4 ? 2 : (room >= 2 ? 1 : 0)) << 2;
    }
    return f;
}
// threads_t x threads_dm is a launch parameter; the code shape only sees it through
// __launch_bounds__, whose register cap is the same (255) for every block of <= 256 threads.
int maxt_bucket(const ddp_kcfg& c) {
    int t = c.threads_t * c.threads_dm;
    if (ddp_merge_group(c)) t += ddp_merge_producer_threads(c);  // the merged kernel adds its producer warps to the block
    return t <= 256 ? 256 : t;
}
std::string kernel_name(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    char b[160];
    const CodeKind ck = code_kind(p, k);
    if (is_dedisp(ck))
        std::snprintf(b, sizeof b, "%s_s%d_d%d_u%d_g%d_v%d_t%d_w%d", kind_tag(ck), c.samples_per_thread,
                      c.dms_per_thread, c.unroll, c.staging, c.vec_bytes, maxt_bucket(c), code_flags(p, k, c));
    else if (ck == CK_ISNR)
        std::snprintf(b, sizeof b, "%s%s_s%d_d%d_t%d", kind_tag(ck), p->integ_mode == DDP_INTEG_SLIDING ? "_slide" : "",
                      c.samples_per_thread, c.dms_per_thread, maxt_bucket(c));
    else  // integrate reads `unroll` at run time (tiles per block): not part of its code shape
        std::snprintf(b, sizeof b, "%s_s%d_d%d_u%d_g%d_v%d_t%d", kind_tag(ck), c.samples_per_thread,
                      c.dms_per_thread, ck == CK_INTEG ? 1 : c.unroll, c.staging, c.vec_bytes, maxt_bucket(c));
    return b;
}
std::string define_line(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, const std::string& name) {
    char b[320];
    const int maxt = maxt_bucket(c);
    const CodeKind ck = code_kind(p, k);
    switch (ck) {
        case CK_DEDISP_U8:
        case CK_DEDISP_U16:
        case CK_DEDISP_U32:
            std::snprintf(b, sizeof b, "\nDDP_DEFINE_DEDISP(%s, %s, %d, %d, %d, %d, %d, %d, %d)\n", name.c_str(), kind_type(ck),
                          c.samples_per_thread, c.dms_per_thread, c.unroll, c.staging, c.vec_bytes, maxt, code_flags(p, k, c));
            break;
        case CK_ISNR:
            std::snprintf(b, sizeof b, "\nDDP_DEFINE_ISNR%s(%s, %d, %d, %d)\n", p->integ_mode == DDP_INTEG_SLIDING ? "_SLIDE" : "",
                          name.c_str(), c.samples_per_thread, c.dms_per_thread, maxt);
            break;
        case CK_INTEG:
            std::snprintf(b, sizeof b, "\nDDP_DEFINE_INTEG(%s, %d, %d, %d, %d, %d, %d)\n", name.c_str(),
                          c.samples_per_thread, c.dms_per_thread, 1, c.staging, c.vec_bytes, maxt);
            break;
        default:
            std::snprintf(b, sizeof b, "\nDDP_DEFINE_SNR(%s, %d, %d, %d, %d, %d, %d)\n", name.c_str(),
                          c.samples_per_thread, c.dms_per_thread, c.unroll, c.staging, c.vec_bytes, maxt);
            break;
    }
    return b;
}

bool read_file(const std::string& path, std::vector<char>& out) {
    FILE* f = std::fopen(path.c_str(), "rb");
    if (!f) return false;
    std::fseek(f, 0, SEEK_END);
    const long n = std::ftell(f);
    std::fseek(f, 0, SEEK_SET);
    if (n <= 0) {
        std::fclose(f);
        return false;
    }
    out.resize((size_t)n);
    const size_t got = std::fread(out.data(), 1, (size_t)n, f);
    std::fclose(f);
    return got == (size_t)n;
}
void write_file_atomic(const std::string& path, const std::vector<char>& data) {
    char suffix[64];
    std::snprintf(suffix, sizeof suffix, ".tmp%d_%p", (int)getpid(), (void*)&data);
    const std::string tmp = path + suffix;
    FILE* f = std::fopen(tmp.c_str(), "wb");
    if (!f) return;
    const size_t put = std::fwrite(data.data(), 1, data.size(), f);
    std::fclose(f);
    if (put == data.size())
        std::rename(tmp.c_str(), path.c_str());
    else
        std::remove(tmp.c_str());
}

// NVRTC: template text + one DDP_DEFINE_* line -> sm_100a cubin.  Host only, thread safe.
// With DDP_KEEP_SOURCE=1 in the environment and a cache directory, the generated translation unit is
// also written to <cache_dir>/<name>.cu and compiled under that path, so that profilers (ncu
// --import-source) can map SASS back to the template text.
bool nvrtc_compile(const std::string& name, const std::string& define, const std::string& cache_dir,
                   std::vector<char>& cubin, std::string& log) {
    {
        std::lock_guard<std::mutex> lk(g_api_mu);
        if (!load_nvrtc_locked()) {
            log = "libnvrtc.so.12 not available";
            return false;
        }
    }
    const std::string src = std::string(ddp_kernel_source) + define;
    std::string unit = name + ".cu";
    const char* keep = std::getenv("DDP_KEEP_SOURCE");
    if (keep && keep[0] == '1' && !cache_dir.empty()) {
        unit = cache_dir + "/" + unit;
        write_file_atomic(unit, std::vector<char>(src.begin(), src.end()));
    }
    nvrtcProgram prog = nullptr;
    nvrtcResult r = g_api.p_nvrtcCreateProgram(&prog, src.c_str(), unit.c_str(), 0, nullptr, nullptr);
    if (r != NVRTC_SUCCESS) {
        log = std::string("nvrtcCreateProgram: ") + g_api.p_nvrtcGetErrorString(r);
        return false;
    }
    // DDP_NVRTC_DEFINES="NAME=VALUE NAME2=VALUE2": development hook for template experiments
    std::vector<std::string> extra;
    if (const char* d = std::getenv("DDP_NVRTC_DEFINES")) {
        std::string all = d, cur;
        for (char ch : all + " ") {
            if (ch == ' ') {
                if (!cur.empty()) extra.push_back("-D" + cur);
                cur.clear();
            } else {
                cur += ch;
            }
        }
    }
    std::vector<const char*> opts = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo", "--device-int128"};
    for (const std::string& e : extra) opts.push_back(e.c_str());
    r = g_api.p_nvrtcCompileProgram(prog, (int)opts.size(), opts.data());
    g_ncompiles.fetch_add(1);
    if (r != NVRTC_SUCCESS) {
        size_t n = 0;
        g_api.p_nvrtcGetProgramLogSize(prog, &n);
        log.assign(n, '\0');
        if (n) g_api.p_nvrtcGetProgramLog(prog, &log[0]);
        log = std::string("nvrtcCompileProgram: ") + g_api.p_nvrtcGetErrorString(r) + "\n" + log;
        g_api.p_nvrtcDestroyProgram(&prog);
        return false;
    }
    size_t n = 0;
    g_api.p_nvrtcGetCUBINSize(prog, &n);
    cubin.resize(n);
    g_api.p_nvrtcGetCUBIN(prog, cubin.data());
    g_api.p_nvrtcDestroyProgram(&prog);
    return n > 0;
}

std::string lib_dir() {
    Dl_info info;
    if (dladdr((void*)&ddp_rt_compile_count, &info) && info.dli_fname) {
        std::string s = info.dli_fname;
        const size_t k = s.rfind('/');
        return k == std::string::npos ? "." : s.substr(0, k);
    }
    return ".";
}

// Disk-cache tag: FNV-1a of the template text, so that cubins of an older template are never reused.
const std::string& source_tag() {
    static const std::string tag = [] {
        uint64_t h = 1469598103934665603ull;
        for (const char* c = ddp_kernel_source; *c; ++c) h = (h ^ (unsigned char)*c) * 1099511628211ull;
        if (const char* d = std::getenv("DDP_NVRTC_DEFINES"))
            for (const char* c = d; *c; ++c) h = (h ^ (unsigned char)*c) * 1099511628211ull;
        char b[24];
        std::snprintf(b, sizeof b, "%016llx", (unsigned long long)h);
        return std::string(b);
    }();
    return tag;
}

// Registry entry with a device image (or a failure record); no CUDA context needed.
DdpCompiled* obtain_image(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    const std::string name = kernel_name(p, k, c);
    {
        std::lock_guard<std::mutex> lk(g_reg_mu);
        auto it = g_reg.find(name);
        if (it != g_reg.end()) return it->second;
    }
    DdpCompiled* K = new DdpCompiled();
    K->name = name;
    bool have = false;
    const std::string path = p->cache_dir.empty() ? std::string() : p->cache_dir + "/" + name + "." + source_tag() + ".cubin";
    if (!path.empty()) have = read_file(path, K->cubin);
    if (!have) {
        have = nvrtc_compile(name, define_line(p, k, c, name), p->cache_dir, K->cubin, K->log);
        if (have && !path.empty()) write_file_atomic(path, K->cubin);
    }
    K->failed = !have;
    std::lock_guard<std::mutex> lk(g_reg_mu);
    auto it = g_reg.find(name);
    if (it != g_reg.end()) {  // another thread won the race
        delete K;
        return it->second;
    }
    g_reg[name] = K;
    return K;
}

// AOT module of the plan's device (ddp_aot.cubin beside the library), loaded once per device.
CUmodule aot_module_locked(int dev) {
    if (!g_aot_tried[dev]) {
        g_aot_tried[dev] = true;
        std::vector<char> img;
        if (read_file(lib_dir() + "/ddp_aot.cubin", img)) {
            if (g_api.p_cuModuleLoadData(&g_aot_mod[dev], img.data()) != CUDA_SUCCESS) g_aot_mod[dev] = nullptr;
        }
    }
    return g_aot_mod[dev];
}

// Loads the kernel into the context of the plan's device (current on the calling thread).
ddp_status load_kernel(const ddp_plan* p, DdpCompiled* K) {
    const int dev = p->device;
    std::lock_guard<std::mutex> lk(g_load_mu);
    if (K->loaded[dev]) return DDP_OK;
    if (K->failed) return ddp_fail(p, DDP_E_COMPILE, K->name + ": " + K->log);
    CUresult r;
    if (K->aot) {
        CUmodule m = aot_module_locked(dev);
        if (!m || g_api.p_cuModuleGetFunction(&K->fn[dev], m, K->name.c_str()) != CUDA_SUCCESS || !K->fn[dev])
            return ddp_fail(p, DDP_E_COMPILE, K->name + ": not in ddp_aot.cubin on this device");
    } else {
        if (K->cubin.empty()) return ddp_fail(p, DDP_E_COMPILE, K->name + ": no device image");
        r = g_api.p_cuModuleLoadData(&K->mod[dev], K->cubin.data());
        if (r != CUDA_SUCCESS) {
            K->failed = true;
            K->log = "cuModuleLoadData: " + cu_err(r);
            return ddp_fail(p, DDP_E_COMPILE, K->name + ": " + K->log);
        }
        r = g_api.p_cuModuleGetFunction(&K->fn[dev], K->mod[dev], K->name.c_str());
        if (r != CUDA_SUCCESS) {
            K->failed = true;
            K->log = "cuModuleGetFunction: " + cu_err(r);
            return ddp_fail(p, DDP_E_COMPILE, K->name + ": " + K->log);
        }
    }
    g_api.p_cuFuncGetAttribute(&K->regs, CU_FUNC_ATTRIBUTE_NUM_REGS, K->fn[dev]);
    K->loaded[dev] = true;
    return DDP_OK;
}

// AOT lookup: a function of this exact name in ddp_aot.cubin needs no NVRTC at all.
DdpCompiled* obtain_aot(const ddp_plan* p, const std::string& name) {
    {
        std::lock_guard<std::mutex> lk(g_load_mu);
        CUmodule m = aot_module_locked(p->device);
        if (!m) return nullptr;
        CUfunction fn = nullptr;
        if (g_api.p_cuModuleGetFunction(&fn, m, name.c_str()) != CUDA_SUCCESS || !fn) return nullptr;
    }
    DdpCompiled* K = new DdpCompiled();
    K->name = name;
    K->aot = true;
    std::lock_guard<std::mutex> lk(g_reg_mu);
    auto it = g_reg.find(name);
    if (it != g_reg.end()) {
        delete K;
        return it->second;
    }
    g_reg[name] = K;
    return K;
}

// Ready-to-launch kernel of configuration c (context current).
ddp_status get_kernel(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, DdpCompiled** out) {
    const std::string name = kernel_name(p, k, c);
    DdpCompiled* K = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_reg_mu);
        auto it = g_reg.find(name);
        if (it != g_reg.end()) K = it->second;
    }
    if (!K) K = obtain_aot(p, name);
    if (!K) K = obtain_image(p, k, c);
    ddp_status s = load_kernel(p, K);
    if (s != DDP_OK) return s;
    const int dev = p->device;
    const int smem = (int)ddp_smem_bytes(p, k, c);
    if (smem > 48 * 1024 && smem > K->smem_opt_in[dev]) {
        CUresult r = g_api.p_cuFuncSetAttribute(K->fn[dev], CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, smem);
        if (r != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, K->name + ": shared-memory opt-in: " + cu_err(r));
        K->smem_opt_in[dev] = smem;
    }
    *out = K;
    return DDP_OK;
}
}  // namespace

int64_t ddp_rt_compile_count() { return g_ncompiles.load(); }

// Compiles (NVRTC, all host cores) every not-yet-known code shape of the list; pure host work.
void ddp_rt_precompile(const ddp_plan* p, const std::vector<std::pair<ddp_kernel, ddp_kcfg>>& list) {
    std::vector<std::pair<ddp_kernel, ddp_kcfg>> todo;
    {
        std::lock_guard<std::mutex> lk(g_reg_mu);
        std::unordered_map<std::string, int> seen;
        for (const auto& e : list) {
            const std::string name = kernel_name(p, e.first, e.second);
            if (g_reg.count(name) || seen.count(name)) continue;
            seen[name] = 1;
            todo.push_back(e);
        }
    }
    if (todo.empty()) return;
    unsigned nt = std::thread::hardware_concurrency();
    if (nt == 0) nt = 4;
    nt = std::min<unsigned>(nt, 32);
    nt = std::min<unsigned>(nt, (unsigned)todo.size());
    std::atomic<size_t> next{0};
    auto work = [&]() {
        for (;;) {
            const size_t i = next.fetch_add(1);
            if (i >= todo.size()) break;
            obtain_image(p, todo[i].first, todo[i].second);
        }
    };
    std::vector<std::thread> th;
    for (unsigned t = 1; t < nt; ++t) th.emplace_back(work);
    work();
    for (auto& t : th) t.join();
}

// ------------------------------------------------------------------------------------ per-plan state
namespace {
struct PlanRt {
    std::vector<CUevent> ev;  // event pool of the timing harness
    CUstream copy_stream = nullptr;  // ddp_search_host_batches: uploads run beside the compute stream
    CUevent ev_in[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr};
};
PlanRt* rt_of(ddp_plan* p) {
    if (!p->rt) p->rt = new PlanRt();
    return (PlanRt*)p->rt;
}
inline int64_t round_up64(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
}  // namespace

void ddp_rt_release(ddp_plan* p) {
    if (!p || !p->rt) return;
    PlanRt* R = (PlanRt*)p->rt;
    if (g_api.ok)
        for (CUevent e : R->ev) g_api.p_cuEventDestroy(e);
    if (g_api.ok) {
        for (int b = 0; b < 2; ++b) {
            if (R->ev_in[b]) g_api.p_cuEventDestroy(R->ev_in[b]);
            if (R->ev_done[b]) g_api.p_cuEventDestroy(R->ev_done[b]);
        }
        if (R->copy_stream) g_api.p_cuStreamDestroy(R->copy_stream);
    }
    delete R;
    p->rt = nullptr;
}

ddp_status ddp_rt_activate(ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    {
        std::lock_guard<std::mutex> lk(g_api_mu);
        if (!load_cuda_locked()) {  // host-only machine: validity was checked, nothing to compile for
            p->active[k] = nullptr;
            return DDP_OK;
        }
    }
    ddp_status s = ensure_ctx(p, p->device);
    if (s != DDP_OK) return s;
    DdpCompiled* K = nullptr;
    s = get_kernel(p, k, c, &K);
    if (s != DDP_OK) return s;
    p->active[k] = K;
    return DDP_OK;
}

extern "C" ddp_status ddp_plan_bind_workspace(ddp_plan* plan, void* d_workspace, size_t bytes, void* stream) {
    if (!plan) return DDP_E_ARG;
    if (!d_workspace) return ddp_fail(plan, DDP_E_WORKSPACE, "workspace pointer is NULL");
    if (bytes < (size_t)plan->info.workspace_bytes) return ddp_fail(plan, DDP_E_WORKSPACE, "workspace too small");
    if (((uintptr_t)d_workspace & 255u) != 0) return ddp_fail(plan, DDP_E_WORKSPACE, "workspace not 256-byte aligned");
    ddp_status s = ensure_ctx(plan, plan->device);
    if (s != DDP_OK) return s;
    char* base = (char*)d_workspace;
    size_t off = 0;
    auto upload = [&](const std::vector<int32_t>& t, int32_t** dst) -> CUresult {
        *dst = (int32_t*)(base + off);
        off += (size_t)round_up64((int64_t)t.size() * 4, 256);
        return g_api.p_cuMemcpyHtoDAsync((CUdeviceptr)*dst, t.data(), t.size() * 4, (CUstream)stream);
    };
    CUresult r = CUDA_SUCCESS;
    if (plan->subband) {
        r = upload(plan->d1, &plan->d_d1);
        if (r == CUDA_SUCCESS) r = upload(plan->d2, &plan->d_d2);
        plan->d_sub = (uint32_t*)(base + off);
        off += (size_t)round_up64((int64_t)plan->ncoarse * plan->nsub * plan->info.sub_stride * plan->info.sub_elem_bytes, 256);
    } else {
        r = upload(plan->delay, &plan->d_delay);
    }
    plan->d_merge = (unsigned char*)(base + off);
    plan->merge_resident[0] = -1;
    off += (size_t)plan->merge_capacity;
    plan->d_rowmap = nullptr;
    plan->d_zero_row = nullptr;
    if (!plan->chan_mask.empty() && r == CUDA_SUCCESS) {  // DD.7m: masked channels read a row of zeros
        plan->rowmap_host.resize(plan->nchan);
        for (int c = 0; c < plan->nchan; ++c) plan->rowmap_host[c] = plan->chan_mask[c] ? c : -1;
        r = upload(plan->rowmap_host, &plan->d_rowmap);
        plan->d_zero_row = (unsigned char*)(base + off);
        if (r == CUDA_SUCCESS)
            r = g_api.p_cuMemsetD32Async((CUdeviceptr)plan->d_zero_row, 0u,
                                         (size_t)round_up64(plan->info.in_stride_min * plan->in_bytes, 256) / 4,
                                         (CUstream)stream);
    }
    if (r != CUDA_SUCCESS) return ddp_fail(plan, DDP_E_CUDA, "delay table upload: " + cu_err(r));
    plan->ws = d_workspace;
    plan->ws_bytes = bytes;
    return DDP_OK;
}

extern "C" ddp_status ddp_plan_subband_buffer(const ddp_plan* plan, void** d_sub) {
    if (!plan || !d_sub) return DDP_E_ARG;
    *d_sub = (plan->subband && plan->ws) ? (void*)plan->d_sub : nullptr;
    return DDP_OK;
}

// ------------------------------------------------------------------------------------ launches
namespace {
struct IoView {  // what one pipeline pass touches
    const uint8_t* d_in;
    size_t in_stride;
    uint32_t* d_out;
    size_t out_stride;
    uint32_t* d_integ;
    float* d_snr;
    uint32_t* d_argmax;
    CUstream stream;
};

ddp_status check_io_dedisp(const ddp_plan* p, const uint8_t* d_in, size_t in_stride, const uint32_t* d_out,
                           size_t out_stride) {
    if (!d_in || !d_out) return ddp_fail(p, DDP_E_ARG, "NULL device pointer");
    if (!p->ws) return ddp_fail(p, DDP_E_WORKSPACE, "ddp_plan_bind_workspace has not been called");
    if ((int64_t)in_stride < p->info.in_stride_min || in_stride % 16 != 0 || ((uintptr_t)d_in & 15u))
        return ddp_fail(p, DDP_E_SHAPE, "in_stride < in_stride_min, not a multiple of 16, or d_in misaligned");
    if ((int64_t)out_stride < p->info.out_stride_min || out_stride % 4 != 0 || ((uintptr_t)d_out & 15u))
        return ddp_fail(p, DDP_E_SHAPE, "out_stride < out_stride_min, not a multiple of 4, or d_out misaligned");
    return DDP_OK;
}

ddp_status launch(const ddp_plan* p, DdpCompiled* K, unsigned gx, unsigned gy, unsigned gz, unsigned bx, unsigned by,
                  size_t smem, CUstream st, void* params) {
    if (gx == 0 || gy == 0 || gz == 0 || gy > 65535u || gz > 65535u)
        return ddp_fail(p, DDP_E_CONFIG, K->name + ": grid outside the launch limits");
    void* args[] = {params};
    CUresult r = g_api.p_cuLaunchKernel(K->fn[p->device], gx, gy, gz, bx, by, 1, (unsigned)smem, st, args, nullptr);
    if (r != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, K->name + ": cuLaunchKernel: " + cu_err(r));
    return DDP_OK;
}

inline unsigned cdiv(int64_t a, int64_t b) { return (unsigned)((a + b - 1) / b); }

// One dedispersion-type launch (ddp_params.h: out[g][i][t] = sum_r in[g][r][t + delay[g][i][r]]).
ddp_status launch_dedisp(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, DdpCompiled* K, const IoView& io) {
    DdpDedispParams q;
    std::memset(&q, 0, sizeof q);
    const ddp_plan_info& I = p->info;
    unsigned groups = 1;
    switch (k) {
        case DDP_K_DIRECT:
            q.in = io.d_in;
            q.out = io.d_out;
            q.delay = p->d_delay;
            q.in_row_stride = (long long)io.in_stride;
            q.in_group_stride = 0;
            q.in_row_len = (long long)io.in_stride;
            q.out_dm_stride = (long long)io.out_stride;
            q.out_group_stride = 0;
            q.delay_dm_stride = p->nchan;
            q.delay_group_off = 0;
            q.nred = p->nchan;
            q.ndm = p->ndm;
            q.ns = p->ns;
            break;
        case DDP_K_SUB1:  // g = subband, i = coarse DM, r = channel of the subband (SB.1)
            q.in = io.d_in;
            q.out = p->d_sub;  // uint16 or uint32 elements (info.sub_elem_bytes); strides below are in elements
            q.delay = p->d_d1;
            q.in_row_stride = (long long)io.in_stride;
            q.in_group_stride = (long long)io.in_stride * p->cps;
            q.in_row_len = (long long)io.in_stride;
            q.out_dm_stride = (long long)I.sub_stride * p->nsub;
            q.out_group_stride = (long long)I.sub_stride;
            q.delay_dm_stride = p->nchan;
            q.delay_group_off = p->cps;
            q.nred = p->cps;
            q.ndm = p->ncoarse;
            q.ns = (int)I.nsamp_sub;
            groups = (unsigned)p->nsub;
            break;
        default:  // DDP_K_SUB2: g = coarse DM, i = fine DM, r = subband
            q.in = p->d_sub;
            q.out = io.d_out;
            q.delay = p->d_d2;
            q.in_row_stride = (long long)I.sub_stride;
            q.in_group_stride = (long long)I.sub_stride * p->nsub;
            q.in_row_len = (long long)I.sub_stride;
            q.out_dm_stride = (long long)io.out_stride;
            q.out_group_stride = (long long)io.out_stride * p->nfine;
            q.delay_dm_stride = p->nsub;
            q.delay_group_off = 0;
            q.nred = p->nsub;
            q.ndm = p->nfine;
            q.ns = p->ns;
            groups = (unsigned)p->ncoarse;
            break;
    }
    q.win = c.staging ? ddp_dedisp_win(p, k, c) : 0;
    q.one = 1;
    if (p->d_rowmap && k != DDP_K_SUB2) {  // channel mask: the zero row is in_stride_min long, which covers every needed sample
        q.rowmap = p->d_rowmap;
        q.zero_row = p->d_zero_row;
        q.in_row_len = std::min<long long>(q.in_row_len, (long long)I.in_stride_min);
    }
    const int64_t TT = (int64_t)c.threads_t * c.samples_per_thread;
    const int64_t TD = (int64_t)c.threads_dm * c.dms_per_thread;
    if (const int G = ddp_merge_group(c)) {
        // merged staging: a persistent kernel over (tile, segment of <= 256 reduction rows) units
        const DdpMergeGeom mg = ddp_merge_geom(p, k, c);
        q.vmax = mg.vcap;
        q.lw = mg.lw;
        q.le = mg.le;
        q.rows_max = mg.rows_max;
        q.meta_rw = mg.rw;
        // the (kernel, TD, G) table must be the resident one: upload it on the launch stream when it is not
        const int TDm = (int)TD, which = k == DDP_K_DIRECT ? 0 : 1;
        const DdpMergeTable& T = ddp_merge_table(p, k, TDm, G);
        ddp_plan* pm = const_cast<ddp_plan*>(p);
        if (p->merge_resident[0] != which || p->merge_resident[1] != TDm || p->merge_resident[2] != G) {
            const std::vector<unsigned char>& blob = ddp_merge_table_blob(p, k, TDm, G);
            if (blob.empty() || (int64_t)blob.size() > p->merge_capacity)
                return ddp_fail(p, DDP_E_WORKSPACE, "merged-staging table does not fit");
            CUresult r = g_api.p_cuMemcpyHtoDAsync((CUdeviceptr)p->d_merge, blob.data(), blob.size(), io.stream);
            if (r != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, "merged-staging table upload: " + cu_err(r));
            pm->merge_resident[0] = which;
            pm->merge_resident[1] = TDm;
            pm->merge_resident[2] = G;
        }
        q.meta = p->d_merge;
        q.meta_ngg = T.ngg;
        q.meta_gg0_stride = k == DDP_K_SUB1 ? p->cps / G : 0;
        q.n_ttiles = (int)cdiv(q.ns, TT);
        q.n_dtiles = (int)cdiv(q.ndm, TD);
        const bool wide = q.nred > 257;  // code_flags bit 0
        q.nseg = wide ? (q.nred + 255) / 256 : 1;
        const int64_t nunits = (int64_t)groups * q.n_dtiles * q.n_ttiles * q.nseg;
        if (nunits > 0x7fffffff) return ddp_fail(p, DDP_E_CONFIG, K->name + ": too many work units");
        q.nunits = (int)nunits;
        const size_t smem = ddp_smem_bytes(p, k, c);
        q.threads_t = c.threads_t;
        q.threads_dm = c.threads_dm;
        const int threads = c.threads_t * c.threads_dm + ddp_merge_producer_threads(c);  // consumers + producer warps
        int per_sm = 0, nsm = 0;
        CUdevice dev;
        if (g_api.p_cuDeviceGet(&dev, p->device) != CUDA_SUCCESS ||
            g_api.p_cuDeviceGetAttribute(&nsm, CU_DEVICE_ATTRIBUTE_MULTIPROCESSOR_COUNT, dev) != CUDA_SUCCESS ||
            g_api.p_cuOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, K->fn[p->device], threads, smem) != CUDA_SUCCESS ||
            per_sm < 1 || nsm < 1)
            return ddp_fail(p, DDP_E_CUDA, K->name + ": occupancy query failed");
        if (wide) {  // the segments of a tile add into the output with RED.ADD: it starts from zero
            const size_t words = k == DDP_K_DIRECT ? (size_t)p->ndm * io.out_stride
                                                   : (size_t)p->ncoarse * p->nsub * (size_t)I.sub_stride;
            CUresult r = g_api.p_cuMemsetD32Async((CUdeviceptr)q.out, 0u, words, io.stream);
            if (r != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, "zeroing the output: " + cu_err(r));
        }
        const int64_t grid = std::min<int64_t>(nunits, (int64_t)per_sm * nsm);
        return launch(p, K, (unsigned)grid, 1, 1, (unsigned)threads, 1u, smem, io.stream, &q);
    }
    int shift_max = 0;  // DIAG: the tile grid also covers the samples the last trial of a tile owns beyond the first one's
    ddp_sub1_diag(p, k, c, nullptr, &shift_max);
    return launch(p, K, cdiv((int64_t)q.ns + shift_max, TT), cdiv(q.ndm, TD), groups, (unsigned)c.threads_t, (unsigned)c.threads_dm,
                  ddp_smem_bytes(p, k, c), io.stream, &q);
}

ddp_status launch_integ(const ddp_plan* p, const ddp_kcfg& c, DdpCompiled* K, const IoView& io) {
    DdpIntegParams q;
    std::memset(&q, 0, sizeof q);
    const ddp_plan_info& I = p->info;
    q.in = io.d_out;
    q.out = io.d_integ;
    q.in_stride = (long long)io.out_stride;
    int np = 0;
    for (int k = 0; k < p->nwidths; ++k) {
        if (p->widths[k] == 1) continue;
        q.plane_off[np] = I.plane_offset[k];
        q.plane_stride[np] = I.plane_stride[k];
        q.plane_len[np] = (int)I.plane_len[k];
        q.width[np] = p->widths[k];
        ++np;
    }
    if (np == 0) return DDP_OK;  // only w = 1: nothing to integrate
    q.nplanes = np;
    for (int m = 0; m < DDP_MAXW; ++m) q.lvl_plane[m] = -1;
    for (int k = 0; k < np; ++k) {
            int m = 0;
            while ((1 << m) < q.width[k]) ++m;
        q.lvl_plane[m] = k;
        if (m > q.max_lvl) q.max_lvl = m;
    }
    q.ndm = p->ndm;
    q.ns = p->ns;
    q.tiles_per_block = c.unroll;
    const int64_t TT = (int64_t)c.threads_t * c.samples_per_thread;
    const int64_t TD = (int64_t)c.threads_dm * c.dms_per_thread;
    return launch(p, K, cdiv(p->ns, TT * c.unroll), cdiv(p->ndm, TD), 1, (unsigned)c.threads_t, (unsigned)c.threads_dm,
                  ddp_smem_bytes(p, DDP_K_INTEGRATE, c), io.stream, &q);
}

ddp_status launch_snr(const ddp_plan* p, const ddp_kcfg& c, DdpCompiled* K, const IoView& io) {
    DdpSnrParams q;
    std::memset(&q, 0, sizeof q);
    const ddp_plan_info& I = p->info;
    for (int k = 0; k < p->nwidths; ++k) {
        if (p->widths[k] == 1) {
            q.base[k] = io.d_out;
            q.stride[k] = (long long)io.out_stride;
        } else {
            q.base[k] = io.d_integ + I.plane_offset[k];
            q.stride[k] = I.plane_stride[k];
        }
        q.n[k] = (int)I.plane_len[k];
    }
    q.snr = io.d_snr;
    q.argmax = io.d_argmax;
    q.nwidths = p->nwidths;
    q.ndm = p->ndm;
    q.ddof = p->ddof;
    const int64_t TD = (int64_t)c.threads_dm * c.dms_per_thread;
    return launch(p, K, 1, cdiv(p->ndm, TD), (unsigned)p->nwidths, (unsigned)c.threads_t, (unsigned)c.threads_dm,
                  ddp_smem_bytes(p, DDP_K_SNR, c), io.stream, &q);
}

// Fused integration + S/N (ddp_isnr_body): level m = width 2^m; planes only when io.d_integ is given.
ddp_status launch_isnr(const ddp_plan* p, const ddp_kcfg& c, DdpCompiled* K, const IoView& io) {
    DdpIsnrParams q;
    std::memset(&q, 0, sizeof q);
    const ddp_plan_info& I = p->info;
    q.in = io.d_out;
    q.planes = io.d_integ;
    q.in_stride = (long long)io.out_stride;
    for (int m = 0; m < DDP_MAXW; ++m) q.lvl_k[m] = -1;
    for (int k = 0; k < p->nwidths; ++k) {
        int m = 0;
        while ((1 << m) < p->widths[k]) ++m;
        if (m >= DDP_MAXW) return ddp_fail(p, DDP_E_CONFIG, "fused kernel: width too large");
        q.lvl_k[m] = k;
        if (m > q.max_lvl) q.max_lvl = m;
        q.n[k] = (int)I.plane_len[k];
        q.plane_off[k] = p->widths[k] == 1 ? 0 : I.plane_offset[k];
        q.plane_stride[k] = p->widths[k] == 1 ? 0 : I.plane_stride[k];
    }
    q.snr = io.d_snr;
    q.argmax = io.d_argmax;
    q.nwidths = p->nwidths;
    q.ndm = p->ndm;
    q.ns = p->ns;
    q.ddof = p->ddof;
    const int64_t TD = (int64_t)c.threads_dm * c.dms_per_thread;
    if (p->integ_mode == DDP_INTEG_SLIDING) {  // ddp_isnr_slide_body: a grid row per 4 widths, no planes
        if (io.d_integ) return ddp_fail(p, DDP_E_ARG, "sliding boxcar sums are never materialised: d_integ must be NULL");
        for (int k = 0; k < p->nwidths; ++k) q.width[k] = p->widths[k];
        q.slide_nb = ddp_slide_nb(p, c);
        return launch(p, K, cdiv(p->ndm, TD), cdiv(p->nwidths, 4), 1, 32u, (unsigned)c.threads_dm,
                      ddp_smem_bytes(p, DDP_K_ISNR, c), io.stream, &q);
    }
    return launch(p, K, cdiv(p->ndm, TD), 1, 1, 32u, (unsigned)c.threads_dm, ddp_smem_bytes(p, DDP_K_ISNR, c), io.stream, &q);
}

ddp_status launch_kernel(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, DdpCompiled* K, const IoView& io) {
    switch (k) {
        case DDP_K_DIRECT:
        case DDP_K_SUB1:
        case DDP_K_SUB2: return launch_dedisp(p, k, c, K, io);
        case DDP_K_INTEGRATE: return launch_integ(p, c, K, io);
        case DDP_K_ISNR: return launch_isnr(p, c, K, io);
        default: return launch_snr(p, c, K, io);
    }
}

// The plan's active kernel of k (compiled on first use).
ddp_status active_kernel(ddp_plan* p, ddp_kernel k, DdpCompiled** K) {
    if (!p->active[k]) {
        ddp_status s = get_kernel(p, k, p->kcfg[k], &p->active[k]);
        if (s != DDP_OK) return s;
    }
    *K = p->active[k];
    return DDP_OK;
}
}  // namespace

// ------------------------------------------------------------------------------------ compute calls
extern "C" ddp_status ddp_dedisperse(ddp_plan* plan, const uint8_t* d_in, size_t in_stride, uint32_t* d_out,
                                     size_t out_stride, void* stream) {
    if (!plan) return DDP_E_ARG;
    ddp_status s = ensure_ctx(plan, plan->device);
    if (s != DDP_OK) return s;
    s = check_io_dedisp(plan, d_in, in_stride, d_out, out_stride);
    if (s != DDP_OK) return s;
    IoView io{d_in, in_stride, d_out, out_stride, nullptr, nullptr, nullptr, (CUstream)stream};
    DdpCompiled* K = nullptr;
    if (!plan->subband) {
        if ((s = active_kernel(plan, DDP_K_DIRECT, &K)) != DDP_OK) return s;
        return launch_dedisp(plan, DDP_K_DIRECT, plan->kcfg[DDP_K_DIRECT], K, io);
    }
    if ((s = active_kernel(plan, DDP_K_SUB1, &K)) != DDP_OK) return s;
    if ((s = launch_dedisp(plan, DDP_K_SUB1, plan->kcfg[DDP_K_SUB1], K, io)) != DDP_OK) return s;
    if ((s = active_kernel(plan, DDP_K_SUB2, &K)) != DDP_OK) return s;
    return launch_dedisp(plan, DDP_K_SUB2, plan->kcfg[DDP_K_SUB2], K, io);
}

extern "C" ddp_status ddp_integrate(ddp_plan* plan, const uint32_t* d_dedisp, size_t stride, uint32_t* d_integ,
                                    void* stream) {
    if (!plan) return DDP_E_ARG;
    ddp_status s = ensure_ctx(plan, plan->device);
    if (s != DDP_OK) return s;
    if (plan->integ_mode != DDP_INTEG_DECIMATE)
        return ddp_fail(plan, DDP_E_CONFIG, "sliding boxcar plan: the sums are not materialised, use ddp_integrate_snr");
    if (!d_dedisp || (!d_integ && plan->info.integ_elems > 0)) return ddp_fail(plan, DDP_E_ARG, "NULL device pointer");
    if ((int64_t)stride < plan->info.out_stride_min || stride % 4 != 0 || ((uintptr_t)d_dedisp & 15u) ||
        ((uintptr_t)d_integ & 15u))
        return ddp_fail(plan, DDP_E_SHAPE, "stride < out_stride_min, not a multiple of 4, or misaligned pointer");
    IoView io{nullptr, 0, (uint32_t*)d_dedisp, stride, d_integ, nullptr, nullptr, (CUstream)stream};
    DdpCompiled* K = nullptr;
    if ((s = active_kernel(plan, DDP_K_INTEGRATE, &K)) != DDP_OK) return s;
    return launch_integ(plan, plan->kcfg[DDP_K_INTEGRATE], K, io);
}

extern "C" ddp_status ddp_snr(ddp_plan* plan, const uint32_t* d_dedisp, size_t stride, const uint32_t* d_integ,
                              float* d_snr, uint32_t* d_argmax, void* stream) {
    if (!plan) return DDP_E_ARG;
    ddp_status s = ensure_ctx(plan, plan->device);
    if (s != DDP_OK) return s;
    if (plan->integ_mode != DDP_INTEG_DECIMATE)
        return ddp_fail(plan, DDP_E_CONFIG, "sliding boxcar plan: use ddp_integrate_snr");
    if (!d_dedisp || !d_snr || (!d_integ && plan->info.integ_elems > 0))
        return ddp_fail(plan, DDP_E_ARG, "NULL device pointer");
    if ((int64_t)stride < plan->info.out_stride_min || stride % 4 != 0 || ((uintptr_t)d_dedisp & 15u) ||
        ((uintptr_t)d_integ & 15u))
        return ddp_fail(plan, DDP_E_SHAPE, "stride < out_stride_min, not a multiple of 4, or misaligned pointer");
    IoView io{nullptr, 0, (uint32_t*)d_dedisp, stride, (uint32_t*)d_integ, d_snr, d_argmax, (CUstream)stream};
    DdpCompiled* K = nullptr;
    if ((s = active_kernel(plan, DDP_K_SNR, &K)) != DDP_OK) return s;
    return launch_snr(plan, plan->kcfg[DDP_K_SNR], K, io);
}

extern "C" ddp_status ddp_integrate_snr(ddp_plan* plan, const uint32_t* d_dedisp, size_t stride, uint32_t* d_integ,
                                        float* d_snr, uint32_t* d_argmax, void* stream) {
    if (!plan) return DDP_E_ARG;
    ddp_status s = ensure_ctx(plan, plan->device);
    if (s != DDP_OK) return s;
    if (!d_dedisp || !d_snr) return ddp_fail(plan, DDP_E_ARG, "NULL device pointer");
    if ((int64_t)stride < plan->info.out_stride_min || stride % 4 != 0 || ((uintptr_t)d_dedisp & 15u) ||
        ((uintptr_t)d_integ & 15u))
        return ddp_fail(plan, DDP_E_SHAPE, "stride < out_stride_min, not a multiple of 4, or misaligned pointer");
    IoView io{nullptr, 0, (uint32_t*)d_dedisp, stride, d_integ, d_snr, d_argmax, (CUstream)stream};
    DdpCompiled* K = nullptr;
    if ((s = active_kernel(plan, DDP_K_ISNR, &K)) != DDP_OK) return s;
    return launch_isnr(plan, plan->kcfg[DDP_K_ISNR], K, io);
}

// One whole search through HOST buffers: H2D of the filterbank, dedisperse -> integrate -> snr, D2H of
// the S/N table (and argmax), stream synchronised before returning.
extern "C" ddp_status ddp_search_host(ddp_plan* plan, const uint8_t* h_in, size_t in_stride, uint8_t* d_in,
                                      uint32_t* d_out, size_t out_stride, uint32_t* d_integ, float* d_snr,
                                      uint32_t* d_argmax, float* h_snr, uint32_t* h_argmax, void* stream) {
    if (!plan) return DDP_E_ARG;
    if (!h_in || !h_snr || !d_in || !d_snr) return ddp_fail(plan, DDP_E_ARG, "NULL pointer");
    if (h_argmax && !d_argmax) return ddp_fail(plan, DDP_E_ARG, "h_argmax given without d_argmax");
    ddp_status s = ensure_ctx(plan, plan->device);
    if (s != DDP_OK) return s;
    CUstream st = (CUstream)stream;
    CUresult r = g_api.p_cuMemcpyHtoDAsync((CUdeviceptr)d_in, h_in, in_stride * (size_t)plan->nchan * (size_t)plan->in_bytes, st);
    if (r != CUDA_SUCCESS) return ddp_fail(plan, DDP_E_CUDA, "H2D copy: " + cu_err(r));
    if ((s = ddp_dedisperse(plan, d_in, in_stride, d_out, out_stride, stream)) != DDP_OK) return s;
    if (d_integ && plan->integ_mode == DDP_INTEG_DECIMATE) {
        if ((s = ddp_integrate(plan, d_out, out_stride, d_integ, stream)) != DDP_OK) return s;
        if ((s = ddp_snr(plan, d_out, out_stride, d_integ, d_snr, d_argmax, stream)) != DDP_OK) return s;
    } else if ((s = ddp_integrate_snr(plan, d_out, out_stride, nullptr, d_snr, d_argmax, stream)) != DDP_OK) {
        return s;
    }
    const size_t n = (size_t)plan->ndm * plan->nwidths;
    r = g_api.p_cuMemcpyDtoHAsync(h_snr, (CUdeviceptr)d_snr, n * sizeof(float), st);
    if (r == CUDA_SUCCESS && h_argmax) r = g_api.p_cuMemcpyDtoHAsync(h_argmax, (CUdeviceptr)d_argmax, n * 4, st);
    if (r != CUDA_SUCCESS) return ddp_fail(plan, DDP_E_CUDA, "D2H copy: " + cu_err(r));
    r = g_api.p_cuStreamSynchronize(st);
    if (r != CUDA_SUCCESS) return ddp_fail(plan, DDP_E_CUDA, "stream synchronize: " + cu_err(r));
    return DDP_OK;
}

// Consecutive batches of one observation ("10 batches").  Batch b searches the samples
// [b*ns, b*ns + ns + max_delay) of every channel.  Only the ns NEW samples of a batch cross the bus: the max_delay
// samples it shares with the previous batch are carried over on the device (copy from the other input buffer), and
// the upload of batch b+1 runs on a second stream while batch b is searched.
extern "C" ddp_status ddp_search_host_batches(ddp_plan* plan, const uint8_t* h_in, size_t h_stride, int nbatches,
                                              uint8_t* d_in0, uint8_t* d_in1, size_t in_stride, uint32_t* d_out,
                                              size_t out_stride, float* d_snr, uint32_t* d_argmax, float* h_snr,
                                              uint32_t* h_argmax, void* stream) {
    if (!plan) return DDP_E_ARG;
    if (!h_in || !h_snr || !d_in0 || !d_in1 || !d_out || !d_snr || nbatches < 1) return ddp_fail(plan, DDP_E_ARG, "NULL pointer or no batch");
    if (h_argmax && !d_argmax) return ddp_fail(plan, DDP_E_ARG, "h_argmax given without d_argmax");
    ddp_status s = ensure_ctx(plan, plan->device);
    if (s != DDP_OK) return s;
    const ddp_plan_info& I = plan->info;
    const size_t ns = (size_t)plan->ns, carry = (size_t)I.max_delay, eb = (size_t)plan->in_bytes;  // eb: bytes per sample
    if (h_stride < (size_t)nbatches * ns + carry) return ddp_fail(plan, DDP_E_SHAPE, "h_stride shorter than nbatches * nsamp_out + max_delay");
    if ((s = check_io_dedisp(plan, d_in0, in_stride, d_out, out_stride)) != DDP_OK) return s;
    if ((uintptr_t)d_in1 & 15u) return ddp_fail(plan, DDP_E_SHAPE, "d_in1 misaligned");
    PlanRt* R = rt_of(plan);
    if (!R->copy_stream) {
        CUresult r = g_api.p_cuStreamCreate(&R->copy_stream, CU_STREAM_NON_BLOCKING);
        for (int b = 0; b < 2 && r == CUDA_SUCCESS; ++b) {
            r = g_api.p_cuEventCreate(&R->ev_in[b], CU_EVENT_DISABLE_TIMING);
            if (r == CUDA_SUCCESS) r = g_api.p_cuEventCreate(&R->ev_done[b], CU_EVENT_DISABLE_TIMING);
        }
        if (r != CUDA_SUCCESS) return ddp_fail(plan, DDP_E_CUDA, "copy stream / events: " + cu_err(r));
    }
    CUstream st = (CUstream)stream, cs = R->copy_stream;
    uint8_t* d_in[2] = {d_in0, d_in1};
    const size_t n = (size_t)plan->ndm * plan->nwidths;
    auto copy2d = [&](bool from_host, const void* src, size_t spitch, uint8_t* dst, size_t width) -> CUresult {
        CUDA_MEMCPY2D c;
        std::memset(&c, 0, sizeof c);
        if (from_host) { c.srcMemoryType = CU_MEMORYTYPE_HOST; c.srcHost = src; }
        else { c.srcMemoryType = CU_MEMORYTYPE_DEVICE; c.srcDevice = (CUdeviceptr)src; }
        c.srcPitch = spitch * eb;
        c.dstMemoryType = CU_MEMORYTYPE_DEVICE;
        c.dstDevice = (CUdeviceptr)dst;
        c.dstPitch = in_stride * eb;
        c.WidthInBytes = width * eb;
        c.Height = (size_t)plan->nchan;
        return g_api.p_cuMemcpy2DAsync(&c, cs);
    };
    // the caller's earlier work on `stream` (e.g. the previous use of the buffers) comes first
    CUresult r = g_api.p_cuEventRecord(R->ev_done[1], st);
    if (r == CUDA_SUCCESS) r = g_api.p_cuStreamWaitEvent(cs, R->ev_done[1], 0);
    for (int b = 0; b < nbatches && r == CUDA_SUCCESS; ++b) {
        uint8_t* cur = d_in[b & 1];
        if (b >= 2) r = g_api.p_cuStreamWaitEvent(cs, R->ev_done[b & 1], 0);  // the search of batch b - 2 has left this buffer
        if (r != CUDA_SUCCESS) break;
        if (b == 0) {
            r = copy2d(true, h_in, h_stride, cur, ns + carry);
        } else {  // carried samples from the other buffer (device to device), then the new ones
            if (carry) r = copy2d(false, d_in[(b - 1) & 1] + ns * eb, in_stride, cur, carry);
            if (r == CUDA_SUCCESS) r = copy2d(true, h_in + ((size_t)b * ns + carry) * eb, h_stride, cur + carry * eb, ns);
        }
        if (r == CUDA_SUCCESS) r = g_api.p_cuEventRecord(R->ev_in[b & 1], cs);
        if (r == CUDA_SUCCESS) r = g_api.p_cuStreamWaitEvent(st, R->ev_in[b & 1], 0);
        if (r != CUDA_SUCCESS) break;
        if ((s = ddp_dedisperse(plan, cur, in_stride, d_out, out_stride, stream)) != DDP_OK) return s;
        if ((s = ddp_integrate_snr(plan, d_out, out_stride, nullptr, d_snr, d_argmax, stream)) != DDP_OK) return s;
        r = g_api.p_cuMemcpyDtoHAsync(h_snr + (size_t)b * n, (CUdeviceptr)d_snr, n * sizeof(float), st);
        if (r == CUDA_SUCCESS && h_argmax) r = g_api.p_cuMemcpyDtoHAsync(h_argmax + (size_t)b * n, (CUdeviceptr)d_argmax, n * 4, st);
        if (r == CUDA_SUCCESS) r = g_api.p_cuEventRecord(R->ev_done[b & 1], st);
    }
    if (r != CUDA_SUCCESS) return ddp_fail(plan, DDP_E_CUDA, "batched search: " + cu_err(r));
    r = g_api.p_cuStreamSynchronize(st);
    if (r == CUDA_SUCCESS) r = g_api.p_cuStreamSynchronize(cs);
    if (r != CUDA_SUCCESS) return ddp_fail(plan, DDP_E_CUDA, "stream synchronize: " + cu_err(r));
    return DDP_OK;
}

// ------------------------------------------------------------------------------------ timing harness
// Fitness of a joint configuration ("run time of the whole pipeline"; BJ:cfg4 "summed CUDA-event
// time of the four kernels, median of 5 runs"): warm-up passes, then `reps` timed passes of the
// plan's kernels in pipeline order on the caller's buffers, one CUDA event between consecutive
// kernels; *ms = median over passes of the summed kernel times.  A configuration that fails to
// compile or launch costs +inf (the analogue of the paper's 3-minute penalty) and still
// counts as an evaluation.  Compile time is not part of the fitness (P:205 excludes T_data likewise).
static double median_of(std::vector<double> v) {
    std::sort(v.begin(), v.end());
    const size_t n = v.size();
    return n == 0 ? 0.0 : (n % 2 ? v[n / 2] : 0.5 * (v[n / 2 - 1] + v[n / 2]));
}

ddp_status ddp_rt_time_pipeline_mask(ddp_plan* p, const ddp_tune_io* io, const ddp_kcfg cfg[DDP_NSLOTS], unsigned slot_mask,
                                     double best_so_far, double* ms, double kernel_ms[DDP_NSLOTS], int64_t* n_timings) {
    const double inf = std::numeric_limits<double>::infinity();
    for (int s = 0; s < DDP_NSLOTS; ++s) kernel_ms[s] = 0.0;
    *ms = inf;
    ddp_status st = ensure_ctx(p, p->device);
    if (st != DDP_OK) return st;
    if (!io->d_in || !io->d_out || !io->d_snr || (!io->d_integ && p->info.integ_elems > 0))
        return ddp_fail(p, DDP_E_ARG, "tune io: NULL device buffer");
    st = check_io_dedisp(p, io->d_in, io->in_stride, io->d_out, io->out_stride);
    if (st != DDP_OK) return st;

    ddp_kernel kern[DDP_NSLOTS];
    DdpCompiled* K[DDP_NSLOTS] = {nullptr, nullptr, nullptr, nullptr};
    int nk = 0, slot_of[DDP_NSLOTS];
    for (int s = 0; s < DDP_NSLOTS; ++s) {
        const ddp_kernel k = ddp_slot_kernel(p, s);
        if (k == DDP_K_COUNT || !(slot_mask & (1u << s))) continue;
        if (!ddp_kcfg_valid(p, k, cfg[s], nullptr)) return DDP_OK;  // +inf
        if (get_kernel(p, k, cfg[s], &K[nk]) != DDP_OK) return DDP_OK;  // compile failure: +inf
        kern[nk] = k;
        slot_of[nk] = s;
        ++nk;
    }
    const int reps = io->reps > 0 ? io->reps : 5;
    const int warm = io->warmup > 0 ? io->warmup : (io->warmup < 0 ? 0 : 1);  // 0 = default 1, negative = none
    PlanRt* R = rt_of(p);
    const size_t need = (size_t)reps * (nk + 1);
    while (R->ev.size() < need) {
        CUevent e;
        if (g_api.p_cuEventCreate(&e, CU_EVENT_DEFAULT) != CUDA_SUCCESS) return ddp_fail(p, DDP_E_CUDA, "cuEventCreate");
        R->ev.push_back(e);
    }
    CUstream stream = (CUstream)io->stream;
    IoView v{io->d_in, io->in_stride, io->d_out, io->out_stride, io->d_integ, io->d_snr, io->d_argmax, stream};
    auto pass = [&](CUevent* ev) -> bool {
        if (io->d_flush && io->flush_bytes >= 4)
            g_api.p_cuMemsetD32Async((CUdeviceptr)io->d_flush, 0u, io->flush_bytes / 4, stream);
        if (ev) g_api.p_cuEventRecord(ev[0], stream);
        for (int i = 0; i < nk; ++i) {
            if (launch_kernel(p, kern[i], cfg[slot_of[i]], K[i], v) != DDP_OK) return false;
            if (ev) g_api.p_cuEventRecord(ev[i + 1], stream);
        }
        return true;
    };
    for (int w = 0; w < warm; ++w)
        if (!pass(nullptr)) {
            g_api.p_cuStreamSynchronize(stream);
            return DDP_OK;  // launch failure: +inf
        }
    std::vector<double> total;
    std::vector<std::vector<double>> per(nk);
    int done = 0;
    auto collect = [&](int upto) -> bool {
        for (; done < upto; ++done) {
            CUevent* ev = &R->ev[(size_t)done * (nk + 1)];
            if (g_api.p_cuEventSynchronize(ev[nk]) != CUDA_SUCCESS) return false;
            double sum = 0.0;
            for (int i = 0; i < nk; ++i) {
                float t = 0.f;
                if (g_api.p_cuEventElapsedTime(&t, ev[i], ev[i + 1]) != CUDA_SUCCESS) return false;
                per[i].push_back((double)t);
                sum += (double)t;
            }
            total.push_back(sum);
        }
        return true;
    };
    int issued = 0;
    for (int r = 0; r < reps; ++r) {
        if (!pass(&R->ev[(size_t)r * (nk + 1)])) {
            g_api.p_cuStreamSynchronize(stream);
            return DDP_OK;
        }
        ++issued;
        if (r == 0 && io->cutoff_factor > 0.0 && std::isfinite(best_so_far)) {
            if (!collect(1)) return ddp_fail(p, DDP_E_CUDA, "event timing failed (kernel fault?)");
            if (total[0] > io->cutoff_factor * best_so_far) break;  // hopeless: keep the single sample
        }
    }
    if (!collect(issued)) return ddp_fail(p, DDP_E_CUDA, "event timing failed (kernel fault?)");
    *ms = median_of(total);
    for (int i = 0; i < nk; ++i) kernel_ms[slot_of[i]] = median_of(per[i]);
    if (n_timings) *n_timings += (int64_t)total.size() * nk;
    return DDP_OK;
}

// NVRTC-only entry used by build steps and tests on machines without a GPU: compiles the code shape
// of (k, cfg) for sm_100a (into the plan's cache_dir when set).  DDP_E_COMPILE with the log on failure.
extern "C" ddp_status ddp_compile_kcfg(ddp_plan* plan, ddp_kernel k, const ddp_kcfg* cfg) {
    if (!plan || !cfg || k < 0 || k >= DDP_K_COUNT) return DDP_E_ARG;
    std::string why;
    if (!ddp_kcfg_valid(plan, k, *cfg, &why)) return ddp_fail(plan, DDP_E_CONFIG, why);
    DdpCompiled* K = obtain_image(plan, k, *cfg);
    if (K->failed) return ddp_fail(plan, DDP_E_COMPILE, K->name + ": " + K->log);
    return DDP_OK;
}
