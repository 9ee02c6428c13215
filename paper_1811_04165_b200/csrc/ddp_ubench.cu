// Instruction-rate micro-benchmarks behind the dedispersion add roofline (
// "the per-SM integer-add rate of sm_100 is not in MEASURED_PEAKS.json and must be
// measured on the box").  Standalone: build.py compiles it with nvcc for sm_100a into `ddp_ubench`
// and then CHECKS THE SASS of every kernel (cuobjdump): the loop body must hold exactly NCH
// instructions of the opcode(s) under test plus the loop counter, compare and branch -- ptxas fuses
// dependent `add.u32` pairs into one three-input IADD3 and merges or hoists anything that is not
// loop carried, which is how round 1 misread "127 adds per clock" as "127 IADD3 per clock".
//
// Construction that cannot be folded: NCH independent dependency chains per thread, ONE instruction
// per chain per iteration of a loop that is not unrolled (`#pragma unroll 1`), every instruction
// loop carried through its own chain register.  Mixes alternate two opcodes chain by chain, so a
// mix that reaches ~2x the single-opcode rate shows that the two opcodes issue to different pipes.
//
// One block of 512 threads per SM (a 120 KB dynamic shared-memory request keeps a second block off
// the SM); the SM clock is measured inside the kernel (clock64 against globaltimer), so the rates do
// not depend on what nvidia-smi reports.  Output: one JSON object; per kernel
//   "inst_per_clk_per_sm"  thread-instructions of the loop body (NCH + 3) x iterations x threads /
//                          (kernel time x measured SM clock), per SM
//   "adds_per_clk_per_sm"  for the add kernels: scalar 32-bit additions performed, same denominator.
// Nothing of the search is computed here.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#define CK(x)                                                                          \
    do {                                                                               \
        cudaError_t e_ = (x);                                                          \
        if (e_ != cudaSuccess) {                                                       \
            std::fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_));              \
            std::exit(1);                                                              \
        }                                                                              \
    } while (0)

#define NCH 96      // independent chains per thread = instructions under test per loop iteration
#define THREADS 512
#define SMEM_WORDS 8192

enum Mix {
    M_IADD_2IN,    // a += b                      -> IADD3 with one zero input (one add per instruction)
    M_IADD3_3IN,   // a += b; a += c (two PTX adds, fused by ptxas) -> IADD3, three live inputs (two adds)
    M_LOP3,        // a = a ^ b ^ c
    M_PRMT,        // a = prmt(a, b, sel)
    M_IMAD,        // a = b * one + a             -> IMAD
    M_IDP4A,       // a = dp4a(b, one, a)         -> IDP.4A
    M_IMAD_IMM,    // a = b * 3 + a               -> IMAD with an immediate multiplier
    M_IADD3_IMAD,  // even chains IADD3 (three inputs), odd chains IMAD
    M_LOP3_IMAD,
    M_PRMT_IMAD,
    M_LOP3_IDP4A,
    M_PRMT_IDP4A,
    M_LOP3_PRMT,   // both on the alu pipe: must NOT exceed the single-opcode rate
    M_LDS32,       // x = lds[x]: loop-carried, conflict-free 32-bit shared loads
    M_LDS32_IADD3, // even chains LDS.32, odd chains IADD3 (three inputs)
    M_COUNT
};
static const char* kNames[M_COUNT] = {"iadd_2in", "iadd3_3in", "lop3", "prmt", "imad", "idp4a", "imad_imm", "iadd3_imad",
                                      "lop3_imad", "prmt_imad", "lop3_idp4a", "prmt_idp4a", "lop3_prmt", "lds32",
                                      "lds32_iadd3"};
// scalar 32-bit additions per loop iteration (0 = not an add kernel)
static const int kAdds[M_COUNT] = {NCH, 2 * NCH, 0, 0, NCH, NCH, NCH, 2 * (NCH / 2) + NCH / 2, 0, 0, 0, 0, 0, 0, 0};

__device__ __forceinline__ unsigned long long gtimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

template <int MIX>
__device__ __forceinline__ void chain_op(unsigned& a, int k, unsigned b, unsigned c, unsigned one, unsigned sbase) {
    const bool odd = (k & 1) != 0;
    if constexpr (MIX == M_IADD_2IN) {
        asm volatile("add.u32 %0, %0, %1;" : "+r"(a) : "r"(b));
    } else if constexpr (MIX == M_IADD3_3IN) {
        asm volatile("add.u32 %0, %0, %1;\n\tadd.u32 %0, %0, %2;" : "+r"(a) : "r"(b), "r"(c));
    } else if constexpr (MIX == M_LOP3) {
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(c));
    } else if constexpr (MIX == M_PRMT) {
        asm volatile("prmt.b32 %0, %0, %1, 0x4341;" : "+r"(a) : "r"(b));
    } else if constexpr (MIX == M_IMAD) {
        asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(one));
    } else if constexpr (MIX == M_IDP4A) {
        asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(one));
    } else if constexpr (MIX == M_IMAD_IMM) {
        asm volatile("mad.lo.u32 %0, %1, 3, %0;" : "+r"(a) : "r"(b));
    } else if constexpr (MIX == M_IADD3_IMAD) {
        if (odd) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(one));
        else asm volatile("add.u32 %0, %0, %1;\n\tadd.u32 %0, %0, %2;" : "+r"(a) : "r"(b), "r"(c));
    } else if constexpr (MIX == M_LOP3_IMAD) {
        if (odd) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(one));
        else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(c));
    } else if constexpr (MIX == M_PRMT_IMAD) {
        if (odd) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(one));
        else asm volatile("prmt.b32 %0, %0, %1, 0x4341;" : "+r"(a) : "r"(b));
    } else if constexpr (MIX == M_LOP3_IDP4A) {
        if (odd) asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(one));
        else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(c));
    } else if constexpr (MIX == M_PRMT_IDP4A) {
        if (odd) asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(one));
        else asm volatile("prmt.b32 %0, %0, %1, 0x4341;" : "+r"(a) : "r"(b));
    } else if constexpr (MIX == M_LOP3_PRMT) {
        if (odd) asm volatile("prmt.b32 %0, %0, %1, 0x4341;" : "+r"(a) : "r"(b));
        else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(c));
    } else if constexpr (MIX == M_LDS32) {
        asm volatile("ld.shared.u32 %0, [%0];" : "+r"(a) : : "memory");
    } else if constexpr (MIX == M_LDS32_IADD3) {
        if (odd) asm volatile("add.u32 %0, %0, %1;\n\tadd.u32 %0, %0, %2;" : "+r"(a) : "r"(b), "r"(c));
        else asm volatile("ld.shared.u32 %0, [%0];" : "+r"(a) : : "memory");
    }
    (void)sbase;
}

template <int MIX>
__global__ void __launch_bounds__(THREADS, 1) ubench(unsigned* out, unsigned long long* stamps, int iters, unsigned one,
                                                     unsigned seed) {
    extern __shared__ __align__(16) unsigned sm[];
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(sm);
    // sm[i] = shared-memory BYTE ADDRESS of word (i + 32 * 37) mod SMEM_WORDS: a permutation that keeps
    // the bank (i mod 32), so a warp whose lanes start in distinct banks never conflicts.
    for (int i = threadIdx.x; i < SMEM_WORDS; i += blockDim.x) sm[i] = sbase + 4u * ((i + 32 * 37) % SMEM_WORDS);
    __syncthreads();
    unsigned a[NCH];
    const bool lds_kernel = MIX == M_LDS32 || MIX == M_LDS32_IADD3;
#pragma unroll
    for (int k = 0; k < NCH; ++k) {
        const bool lds_chain = MIX == M_LDS32 || (MIX == M_LDS32_IADD3 && (k & 1) == 0);
        a[k] = lds_chain ? sbase + 4u * ((threadIdx.x & 31) + 32u * (((threadIdx.x >> 5) * 7 + k * 13) % (SMEM_WORDS / 32)))
                         : seed + threadIdx.x * NCH + k;
    }
    (void)lds_kernel;
    const unsigned b = seed ^ 0x9e3779b9u ^ threadIdx.x, c = b * 5u + 3u;
    __syncthreads();
    const unsigned long long g0 = gtimer();
    const long long c0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < NCH; ++k) chain_op<MIX>(a[k], k, b, c, one, sbase);
    }
    const long long c1 = clock64();
    const unsigned long long g1 = gtimer();
    unsigned acc = 0;
#pragma unroll
    for (int k = 0; k < NCH; ++k) acc ^= a[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0) {
        stamps[2 * blockIdx.x] = (unsigned long long)(c1 - c0);
        stamps[2 * blockIdx.x + 1] = g1 - g0;
    }
}

struct Result { double ms, sm_mhz, inst_rate, add_rate; };

template <int MIX>
static Result run(int nsm, int iters, unsigned* d_out, unsigned long long* d_st) {
    const size_t smem = 120 * 1024;  // > half of the SM's shared memory: at most one block per SM
    CK(cudaFuncSetAttribute(ubench<MIX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ubench<MIX><<<nsm, THREADS, smem>>>(d_out, d_st, 64, 1u, 7u);  // warm-up
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    CK(cudaEventRecord(e0));
    ubench<MIX><<<nsm, THREADS, smem>>>(d_out, d_st, iters, 1u, 7u);
    CK(cudaEventRecord(e1));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    std::vector<unsigned long long> st(2 * nsm);
    CK(cudaMemcpy(st.data(), d_st, st.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    double cyc = 0.0, ns = 0.0;
    for (int i = 0; i < nsm; ++i) { cyc += (double)st[2 * i]; ns += (double)st[2 * i + 1]; }
    Result r;
    r.ms = ms;
    r.sm_mhz = cyc / ns * 1e3;  // SM cycles per nanosecond of the in-kernel timed region
    // per-SM rates from the in-kernel cycle count of the block that ran on each SM (mean over SMs)
    const double cycles_per_block = cyc / nsm;
    r.inst_rate = (double)(NCH + 3) * iters * THREADS / cycles_per_block;
    r.add_rate = (double)kAdds[MIX] * iters * THREADS / cycles_per_block;
    CK(cudaEventDestroy(e0));
    CK(cudaEventDestroy(e1));
    return r;
}

int main(int argc, char** argv) {
    const int iters = argc > 1 ? std::atoi(argv[1]) : 8192;
    const char* only = argc > 2 ? argv[2] : nullptr;  // run one kernel only (for ncu)
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    const int nsm = prop.multiProcessorCount;
    unsigned* d_out;
    unsigned long long* d_st;
    CK(cudaMalloc(&d_out, (size_t)nsm * THREADS * sizeof(unsigned)));
    CK(cudaMalloc(&d_st, (size_t)2 * nsm * sizeof(unsigned long long)));
    Result r[M_COUNT];
    bool ran[M_COUNT] = {false};
#define RUN(M)                                                        \
    if (!only || std::strcmp(only, kNames[M]) == 0) {                 \
        r[M] = run<M>(nsm, iters, d_out, d_st);                       \
        ran[M] = true;                                                \
    }
    RUN(M_IADD_2IN) RUN(M_IADD3_3IN) RUN(M_LOP3) RUN(M_PRMT) RUN(M_IMAD) RUN(M_IDP4A) RUN(M_IMAD_IMM) RUN(M_IADD3_IMAD)
    RUN(M_LOP3_IMAD) RUN(M_PRMT_IMAD) RUN(M_LOP3_IDP4A) RUN(M_PRMT_IDP4A) RUN(M_LOP3_PRMT) RUN(M_LDS32)
    RUN(M_LDS32_IADD3)
#undef RUN
    std::printf("{\"device\": \"%s\", \"sms\": %d, \"iters\": %d, \"threads_per_sm\": %d, \"chains\": %d, \"kernels\": {",
                prop.name, nsm, iters, THREADS, NCH);
    bool first = true;
    for (int m = 0; m < M_COUNT; ++m) {
        if (!ran[m]) continue;
        std::printf("%s\"%s\": {\"ms\": %.4f, \"sm_mhz\": %.1f, \"inst_per_clk_per_sm\": %.2f", first ? "" : ", ", kNames[m],
                    r[m].ms, r[m].sm_mhz, r[m].inst_rate);
        if (kAdds[m]) std::printf(", \"adds_per_clk_per_sm\": %.2f", r[m].add_rate);
        std::printf("}");
        first = false;
    }
    std::printf("}}\n");
    return 0;
}
