// ddp_static.cu -- the allocation-free entry point of include/ddp_static.h (libddp_static.so; CUDA runtime API,
// statically linked).  Two-step subband dedispersion whose intermediate S lives in a file-scope device array.
// The kernels are two instantiations of the library's dedispersion template (ddp_kernels.cuh, generic direct-load
// body): step 1 uint8 -> uint32, step 2 uint32 -> uint32.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/ddp_static.h"
#include "ddp_params.h"
#include "ddp_kernels.cuh"

// The scratch.  In HOST code this name is a stand-in, not a device address: it is only ever handed to
// cudaGetSymbolAddress (below); kernels get the resolved pointer.
static __device__ __align__(256) unsigned char ddp_static_scratch[DDP_STATIC_SCRATCH_BYTES];

// step 1: 8 samples x 2 coarse trials per thread, one channel per iteration (divides every subband length)
#define DDP_ST1_SPT 8
#define DDP_ST1_DPT 2
#define DDP_ST1_TX 32
#define DDP_ST1_TY 8
// step 2: 4 samples x 4 fine trials per thread
#define DDP_ST2_SPT 4
#define DDP_ST2_DPT 4
#define DDP_ST2_TX 64
#define DDP_ST2_TY 4
DDP_DEFINE_DEDISP(ddp_static_step1, ddp_u8, DDP_ST1_SPT, DDP_ST1_DPT, 1, 0, 8, 256, 0)
DDP_DEFINE_DEDISP(ddp_static_step2, ddp_u32, DDP_ST2_SPT, DDP_ST2_DPT, 1, 0, 16, 256, 0)

namespace {

thread_local char g_err[256] = "";
int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

// Device address of the scratch array, resolved once per device with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_ptr[kMaxDevices] = {nullptr};

int scratch_of_current_device(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(DDP_STATIC_E_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(DDP_STATIC_E_CUDA, "device ordinal %d outside 0..%d", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, ddp_static_scratch);
        if (e != cudaSuccess || !p)
            return fail(DDP_STATIC_E_CUDA, "cudaGetSymbolAddress(ddp_static_scratch) on device %d: %s", dev, cudaGetErrorString(e));
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return DDP_STATIC_OK;
}

inline long long round_up(long long a, long long b) { return (a + b - 1) / b * b; }
inline unsigned cdiv(long long a, long long b) { return (unsigned)((a + b - 1) / b); }

}  // namespace

extern "C" size_t ddp_static_scratch_bytes(void) { return (size_t)DDP_STATIC_SCRATCH_BYTES; }
extern "C" const char* ddp_static_last_error(void) { return g_err; }

extern "C" int ddp_static_subband_dedisperse(const uint8_t* d_in, size_t in_stride, int nchan, int n_subbands,
                                             const int32_t* d_d1, int n_coarse, int max_d1,
                                             const int32_t* d_d2, int n_fine, int max_d2,
                                             int nsamp_out, uint32_t* d_out, size_t out_stride, void* stream) {
    g_err[0] = 0;
    if (!d_in || !d_d1 || !d_d2 || !d_out) return fail(DDP_STATIC_E_ARG, "NULL device pointer");
    if (nchan <= 0 || n_subbands <= 0 || n_coarse <= 0 || n_fine <= 0 || nsamp_out <= 0 || max_d1 < 0 || max_d2 < 0)
        return fail(DDP_STATIC_E_ARG, "non-positive size or negative delay bound");
    if (nchan % n_subbands != 0) return fail(DDP_STATIC_E_ARG, "n_subbands = %d does not divide nchan = %d", n_subbands, nchan);
    if ((long long)nsamp_out + max_d1 + max_d2 + 64 >= (1ll << 31)) return fail(DDP_STATIC_E_ARG, "sample count outside int32");
    if ((long long)n_coarse * n_fine >= (1ll << 31)) return fail(DDP_STATIC_E_ARG, "trial count outside int32");
    if (255.0 * (double)nchan >= 4294967296.0) return fail(DDP_STATIC_E_ARG, "uint32 sums could overflow");
    const long long need_in = round_up((long long)nsamp_out + max_d1 + max_d2 + 32, 16);
    if ((long long)in_stride < need_in || in_stride % 16 != 0 || ((uintptr_t)d_in & 15u))
        return fail(DDP_STATIC_E_SHAPE, "in_stride %zu: need >= %lld, a multiple of 16, d_in 16-byte aligned", in_stride, need_in);
    if ((long long)out_stride < round_up(nsamp_out, 4) || out_stride % 4 != 0 || ((uintptr_t)d_out & 15u))
        return fail(DDP_STATIC_E_SHAPE, "out_stride %zu: need >= %lld, a multiple of 4, d_out 16-byte aligned", out_stride,
                    round_up(nsamp_out, 4));
    const int cps = nchan / n_subbands;
    const long long nsamp_sub = (long long)nsamp_out + max_d2;           // samples of S that step 2 reads
    const long long sub_stride = round_up(nsamp_sub + 32, 32);             // row stride of S in the scratch (elements)
    const long long per_coarse = (long long)n_subbands * sub_stride * 4;   // bytes of one coarse trial's intermediate
    if (per_coarse > (long long)DDP_STATIC_SCRATCH_BYTES)
        return fail(DDP_STATIC_E_TOO_LARGE,
                    "one coarse trial needs %lld bytes of intermediate (%d subbands x %lld samples x 4), the static scratch holds %u",
                    per_coarse, n_subbands, sub_stride, (unsigned)DDP_STATIC_SCRATCH_BYTES);
    void* scratch = nullptr;
    int rc = scratch_of_current_device(&scratch);
    if (rc != DDP_STATIC_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int group = (int)std::min<long long>((long long)DDP_STATIC_SCRATCH_BYTES / per_coarse, (long long)n_coarse);

    for (int a0 = 0; a0 < n_coarse; a0 += group) {
        const int na = std::min(group, n_coarse - a0);
        // ---- step 1: g = subband, i = coarse trial a0 + i, r = channel of the subband  ->  S in the scratch
        DdpDedispParams q;
        std::memset(&q, 0, sizeof q);
        q.in = d_in;
        q.out = (unsigned int*)scratch;
        q.delay = d_d1 + (size_t)a0 * nchan;
        q.in_row_stride = (long long)in_stride;
        q.in_group_stride = (long long)in_stride * cps;
        q.in_row_len = (long long)in_stride;
        q.out_dm_stride = sub_stride * n_subbands;
        q.out_group_stride = sub_stride;
        q.delay_dm_stride = nchan;
        q.delay_group_off = cps;
        q.nred = cps;
        q.ndm = na;
        q.ns = (int)nsamp_sub;
        q.one = 1;
        {
            const dim3 block(DDP_ST1_TX, DDP_ST1_TY);
            const dim3 grid(cdiv(nsamp_sub, DDP_ST1_TX * DDP_ST1_SPT), cdiv(na, DDP_ST1_TY * DDP_ST1_DPT), (unsigned)n_subbands);
            if (grid.y > 65535u || grid.z > 65535u) return fail(DDP_STATIC_E_ARG, "grid outside the launch limits (step 1)");
            ddp_static_step1<<<grid, block, 0, st>>>(q);
        }
        // ---- step 2: g = coarse trial of the group, i = fine trial, r = subband  ->  out rows (a0 + g) * n_fine + i
        DdpDedispParams w;
        std::memset(&w, 0, sizeof w);
        w.in = scratch;
        w.out = d_out + (size_t)a0 * n_fine * out_stride;
        w.delay = d_d2;
        w.in_row_stride = sub_stride;
        w.in_group_stride = sub_stride * n_subbands;
        w.in_row_len = sub_stride;
        w.out_dm_stride = (long long)out_stride;
        w.out_group_stride = (long long)out_stride * n_fine;
        w.delay_dm_stride = n_subbands;
        w.delay_group_off = 0;
        w.nred = n_subbands;
        w.ndm = n_fine;
        w.ns = nsamp_out;
        w.one = 1;
        {
            const dim3 block(DDP_ST2_TX, DDP_ST2_TY);
            const dim3 grid(cdiv(nsamp_out, DDP_ST2_TX * DDP_ST2_SPT), cdiv(n_fine, DDP_ST2_TY * DDP_ST2_DPT), (unsigned)na);
            if (grid.y > 65535u || grid.z > 65535u) return fail(DDP_STATIC_E_ARG, "grid outside the launch limits (step 2)");
            ddp_static_step2<<<grid, block, 0, st>>>(w);
        }
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(DDP_STATIC_E_CUDA, "kernel launch: %s", cudaGetErrorString(e));
    }
    return DDP_STATIC_OK;
}
