// Instruction-rate micro-benchmarks behind the dedispersion add roofline (
// "the per-SM integer-add rate of sm_100 is not in MEASURED_PEAKS.json and must be
// measured on the box").  Standalone: build.py compiles it with nvcc for sm_100a into `ddp_ubench`;
// `ddp_ubench` prints one JSON object with, per instruction mix, thread-operations per clock per SM:
// "thread_ops_per_clk_per_sm_wall" = all thread-operations of the launch / CUDA-event time / (SMs x the
// device's SM clock) -- the figure to use (B200, 1965 MHz: IADD3 126-127, LOP3 / PRMT / IMAD / IDP.4A 63.7) --
// and "thread_ops_per_clk_per_sm" from clock64 deltas inside the kernel, which on B200 comes out 1.34x
// higher than the wall-clock figure for every mix (cause not investigated) and is kept only for
// comparison.  Nothing of the search is computed here.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <vector>

#define CK(x)                                                                          \
    do {                                                                               \
        cudaError_t e_ = (x);                                                          \
        if (e_ != cudaSuccess) {                                                       \
            std::fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_));              \
            std::exit(1);                                                              \
        }                                                                              \
    } while (0)

enum Mix { M_IADD3, M_LOP3, M_PRMT, M_IMAD, M_IMADWIDE, M_DP4A, M_LOOP_NOLDS, M_LDS32, M_LOOP,
           M_LOP3_IADD3, M_LOP3_PRMT_2IADD3, M_T_NOLDS, M_T, M_COUNT };
static const char* kNames[M_COUNT] = {"iadd3", "lop3", "prmt", "imad", "imad_wide", "idp4a",
                                      "lop3_prmt_2imad", "lds32", "lds32_lop3_prmt_2imad",
                                      "lop3_iadd3", "lop3_prmt_2iadd3", "lop3_iadd3_imadwide", "lds32_lop3_iadd3_imadwide"};
// thread-operations per loop body (8 independent chains x 8 repeats of the pattern)
static const int kOpsPerBody[M_COUNT] = {64, 64, 64, 64, 64, 64, 64 * 4, 64, 64 * 5, 64 * 2, 64 * 4, 64 * 3, 64 * 4};

template <int MIX>
__global__ void __launch_bounds__(512, 2) ubench(unsigned* out, unsigned long long* cycles, int iters, unsigned one,
                                               unsigned seed) {
    __shared__ unsigned sm[2048];
    for (int i = threadIdx.x; i < 2048; i += blockDim.x) sm[i] = seed * (unsigned)i + 12345u;
    __syncthreads();
    unsigned a[8], b[8], c[8];
    unsigned long long w[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        a[k] = seed + threadIdx.x * 8 + k;
        b[k] = a[k] ^ 0x9e3779b9u;
        w[k] = a[k];
        c[k] = b[k] + 3u;
    }
    const unsigned lp = (unsigned)__cvta_generic_to_shared(sm + (threadIdx.x & 511));
    const long long c0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if constexpr (MIX == M_IADD3) {
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(a[k]) : "r"(b[k]));
                } else if constexpr (MIX == M_LOP3) {
                    asm volatile("lop3.b32 %0, %0, %1, 0x00ff00ff, 0x6a;" : "+r"(a[k]) : "r"(b[k]));
                } else if constexpr (MIX == M_PRMT) {
                    asm volatile("prmt.b32 %0, %0, %1, 0x4341;" : "+r"(a[k]) : "r"(b[k]));
                } else if constexpr (MIX == M_IMAD) {
                    asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[k]) : "r"(b[k]), "r"(one));
                } else if constexpr (MIX == M_IMADWIDE) {
                    asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(w[k]) : "r"(b[k]), "r"(one));
                } else if constexpr (MIX == M_DP4A) {
                    asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(a[k]) : "r"(b[k]), "r"(one));
                } else if constexpr (MIX == M_LOOP_NOLDS || MIX == M_LOOP || MIX == M_LDS32) {
                    unsigned x = b[k];
                    if constexpr (MIX != M_LOOP_NOLDS) {
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(x) : "r"(lp + 128u * ((r * 8 + k) & 31)));
                    }
                    if constexpr (MIX == M_LDS32) {
                        asm volatile("add.u32 %0, %0, %1;" : "+r"(a[k]) : "r"(x));  // LDS + IADD3
                    } else {
                        unsigned e, o;
                        asm volatile("and.b32 %0, %1, 0x00ff00ff;" : "=r"(e) : "r"(x));
                        asm volatile("prmt.b32 %0, %1, 0, 0x4341;" : "=r"(o) : "r"(x));
                        asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[k]) : "r"(e), "r"(one));
                        asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(b[k]) : "r"(o), "r"(one));
                    }
                } else if constexpr (MIX == M_LOP3_IADD3) {
                    unsigned e;
                    asm volatile("and.b32 %0, %1, 0x00ff00ff;" : "=r"(e) : "r"(b[k]));
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(a[k]) : "r"(e));
                } else if constexpr (MIX == M_LOP3_PRMT_2IADD3) {
                    unsigned e, o;
                    asm volatile("and.b32 %0, %1, 0x00ff00ff;" : "=r"(e) : "r"(b[k]));
                    asm volatile("prmt.b32 %0, %1, 0, 0x4341;" : "=r"(o) : "r"(b[k]));
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(a[k]) : "r"(e));
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(c[k]) : "r"(o));
                } else if constexpr (MIX == M_T_NOLDS || MIX == M_T) {
                    unsigned x = b[k], e;
                    if constexpr (MIX == M_T) {
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(x) : "r"(lp + 128u * ((r * 8 + k) & 31)));
                    }
                    asm volatile("and.b32 %0, %1, 0x00ff00ff;" : "=r"(e) : "r"(x));
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(a[k]) : "r"(e));
                    asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(w[k]) : "r"(x), "r"(one));
                }
            }
        }
    }
    const long long c1 = clock64();
    unsigned acc = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) acc += a[k] + b[k] + c[k] + (unsigned)w[k] + (unsigned)(w[k] >> 32);
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(c1 - c0);
}

static double g_clock_hz = 0.0;  // SM clock used for the wall-clock figure (cudaDeviceProp::clockRate)
static double g_wall[M_COUNT];

template <int MIX>
static void run(int nsm, int iters, unsigned* d_out, unsigned long long* d_cyc, double* ops_clk_sm, double* ms_out) {
    const int blocks = 2 * nsm, threads = 512;  // two co-resident blocks per SM: 8 warps per scheduler
    ubench<MIX><<<blocks, threads>>>(d_out, d_cyc, 16, 1u, 7u);  // warm-up
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    CK(cudaEventRecord(e0));
    ubench<MIX><<<blocks, threads>>>(d_out, d_cyc, iters, 1u, 7u);
    CK(cudaEventRecord(e1));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    std::vector<unsigned long long> cyc(blocks);
    CK(cudaMemcpy(cyc.data(), d_cyc, blocks * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    double mean = 0.0;
    for (auto c : cyc) mean += (double)c;
    mean /= blocks;
    *ops_clk_sm = 2.0 * (double)kOpsPerBody[MIX] * iters * threads / mean;  // two blocks share an SM
    g_wall[MIX] = (double)blocks * threads * (double)kOpsPerBody[MIX] * iters / (ms * 1e-3) / (nsm * g_clock_hz);
    *ms_out = ms;
    CK(cudaEventDestroy(e0));
    CK(cudaEventDestroy(e1));
}

int main(int argc, char** argv) {
    const int iters = argc > 1 ? std::atoi(argv[1]) : 4096;
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    const int nsm = prop.multiProcessorCount;
    g_clock_hz = (double)prop.clockRate * 1e3;
    unsigned* d_out;
    unsigned long long* d_cyc;
    CK(cudaMalloc(&d_out, (size_t)nsm * 1024 * sizeof(unsigned)));
    CK(cudaMalloc(&d_cyc, (size_t)2 * nsm * sizeof(unsigned long long)));
    double r[M_COUNT], ms[M_COUNT];
    run<M_IADD3>(nsm, iters, d_out, d_cyc, &r[M_IADD3], &ms[M_IADD3]);
    run<M_LOP3>(nsm, iters, d_out, d_cyc, &r[M_LOP3], &ms[M_LOP3]);
    run<M_PRMT>(nsm, iters, d_out, d_cyc, &r[M_PRMT], &ms[M_PRMT]);
    run<M_IMAD>(nsm, iters, d_out, d_cyc, &r[M_IMAD], &ms[M_IMAD]);
    run<M_IMADWIDE>(nsm, iters, d_out, d_cyc, &r[M_IMADWIDE], &ms[M_IMADWIDE]);
    run<M_DP4A>(nsm, iters, d_out, d_cyc, &r[M_DP4A], &ms[M_DP4A]);
    run<M_LOOP_NOLDS>(nsm, iters, d_out, d_cyc, &r[M_LOOP_NOLDS], &ms[M_LOOP_NOLDS]);
    run<M_LDS32>(nsm, iters, d_out, d_cyc, &r[M_LDS32], &ms[M_LDS32]);
    run<M_LOOP>(nsm, iters, d_out, d_cyc, &r[M_LOOP], &ms[M_LOOP]);
    run<M_LOP3_IADD3>(nsm, iters, d_out, d_cyc, &r[M_LOP3_IADD3], &ms[M_LOP3_IADD3]);
    run<M_LOP3_PRMT_2IADD3>(nsm, iters, d_out, d_cyc, &r[M_LOP3_PRMT_2IADD3], &ms[M_LOP3_PRMT_2IADD3]);
    run<M_T_NOLDS>(nsm, iters, d_out, d_cyc, &r[M_T_NOLDS], &ms[M_T_NOLDS]);
    run<M_T>(nsm, iters, d_out, d_cyc, &r[M_T], &ms[M_T]);
    std::printf("{\"device\": \"%s\", \"sms\": %d, \"iters\": %d, \"thread_ops_per_clk_per_sm\": {", prop.name, nsm, iters);
    for (int m = 0; m < M_COUNT; ++m) std::printf("%s\"%s\": %.2f", m ? ", " : "", kNames[m], r[m]);
    std::printf("}, \"sm_clock_mhz\": %.0f, \"thread_ops_per_clk_per_sm_wall\": {", g_clock_hz / 1e6);
    for (int m = 0; m < M_COUNT; ++m) std::printf("%s\"%s\": %.2f", m ? ", " : "", kNames[m], g_wall[m]);
    std::printf("}, \"kernel_ms\": {");
    for (int m = 0; m < M_COUNT; ++m) std::printf("%s\"%s\": %.4f", m ? ", " : "", kNames[m], ms[m]);
    std::printf("}}\n");
    return 0;
}
