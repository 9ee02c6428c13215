// Ahead-of-time instantiations of the kernel templates for sm_100a (nvcc -> ddp_aot.cubin beside the
// library).  ddp_rt.cpp looks a configuration's kernel up here BY NAME before it falls back to NVRTC,
// so the default configurations and the shapes listed below need no run-time compiler.  The names
// are the ones ddp_rt.cpp::kernel_name() builds: <kind>_s<SPT>_d<DPT>_u<UNROLL>_g<STAGING>_v<VEC>_t<threads>.
#include "ddp_params.h"
#include "ddp_kernels.cuh"

#define DDP_AOT_U8(S, D, U, G, V, T, W) DDP_DEFINE_DEDISP(ddp_dedisp_u8_s##S##_d##D##_u##U##_g##G##_v##V##_t##T##_w##W, ddp_u8, S, D, U, G, V, T, W)
#define DDP_AOT_U32(S, D, U, G, V, T) DDP_DEFINE_DEDISP(ddp_dedisp_u32_s##S##_d##D##_u##U##_g##G##_v##V##_t##T##_w0, ddp_u32, S, D, U, G, V, T, 0)
#define DDP_AOT_U16(S, D, U, G, V, T, W) DDP_DEFINE_DEDISP(ddp_dedisp_u16_s##S##_d##D##_u##U##_g##G##_v##V##_t##T##_w##W, ddp_u16, S, D, U, G, V, T, W)
#define DDP_AOT_INTEG(S, D, U, G, V, T) DDP_DEFINE_INTEG(ddp_integ_s##S##_d##D##_u##U##_g##G##_v##V##_t##T, S, D, U, G, V, T)
#define DDP_AOT_SNR(S, D, U, G, V, T) DDP_DEFINE_SNR(ddp_snr_s##S##_d##D##_u##U##_g##G##_v##V##_t##T, S, D, U, G, V, T)

#define DDP_AOT_ISNR(S, D, T) DDP_DEFINE_ISNR(ddp_isnr_s##S##_d##D##_t##T, S, D, T)

// plan defaults (ddp_plan.cpp::default_kcfgs); W = code flags (bit 0 wide flush, bit 1 uint16 result,
// bits 2-3 log2 lane-sum group of the packed uint16 kernel, bit 4 single buffer, bit 6 diagonal time tiles of step 1)
DDP_AOT_U8(16, 4, 8, 1, 16, 256, 1)
DDP_AOT_U8(16, 2, 8, 1, 16, 256, 2)
DDP_AOT_U8(16, 2, 8, 1, 16, 256, 66)   // the same with diagonal time tiles (chosen per plan from its step-1 delays)
DDP_AOT_U16(4, 8, 8, 2, 16, 256, 8)
DDP_AOT_U32(4, 4, 4, 0, 16, 256)
DDP_AOT_INTEG(4, 1, 1, 0, 16, 256)
DDP_AOT_SNR(4, 1, 4, 0, 16, 256)
DDP_AOT_ISNR(16, 1, 256)
DDP_AOT_ISNR(16, 1, 512)   // cfg1 / cfg2 tuned [32,16,16,1,1,direct,16]: 128 blocks of 16 rows
// one instance of every staging mode per kernel (SASS evidence: LDS / UBLKCP paths)
DDP_AOT_U8(8, 4, 8, 0, 4, 256, 0)
DDP_AOT_U8(16, 4, 8, 1, 16, 256, 0)
DDP_AOT_U8(16, 4, 8, 2, 16, 256, 1)
DDP_AOT_U8(16, 4, 8, 2, 16, 256, 0)
DDP_AOT_U16(4, 4, 4, 0, 8, 256, 0)
DDP_AOT_U16(4, 8, 8, 1, 16, 256, 8)
DDP_AOT_U32(4, 4, 4, 1, 16, 256)
DDP_AOT_U32(4, 4, 4, 2, 16, 256)
DDP_AOT_INTEG(4, 1, 1, 1, 16, 256)
DDP_AOT_INTEG(4, 1, 1, 2, 16, 256)
DDP_AOT_SNR(4, 1, 1, 1, 16, 256)
DDP_AOT_SNR(4, 1, 1, 2, 16, 256)
// tuned shapes of tuned_b200.json (cfg1 / cfg2 / cfg3 on B200), so that the bench needs no run-time compiler
// cfg1 direct [64,8,16,8,8,MERGE4,16] is compiled at first use by NVRTC (its code measured 13 % faster on the B200
// than nvcc's for this kernel: 3.14 vs 3.62 ms; the cubin lands in kcache/)
DDP_AOT_U8(16, 4, 16, 2, 16, 512, 1)   // cfg1 direct, best packed shape [64,8,16,4,16,TMA,16]
DDP_AOT_U8(16, 8, 8, 2, 16, 512, 17)   // cfg3 direct   [128,4,16,8,8,TMA,16], wide flush, single-buffered copies
DDP_AOT_U8(16, 8, 4, 2, 16, 512, 1)    // cfg3 direct, best double-buffered shape [64,8,16,8,4,TMA,16]
DDP_AOT_U8(16, 8, 16, 2, 16, 512, 82)  // cfg2 sub1     [128,4,16,8,16,TMA,16], uint16 result, diagonal time tiles, single-buffered copies
DDP_AOT_U8(16, 8, 8, 2, 16, 512, 66)   // cfg2 sub1, best double-buffered shape with diagonal tiles [128,4,16,8,8,TMA,16]
DDP_AOT_U8(16, 8, 4, 2, 16, 512, 18)   // cfg2 sub1 without diagonal tiles (an ascending band) [128,4,16,8,4,TMA,16], single-buffered copies
DDP_AOT_U16(8, 4, 8, 2, 16, 256, 8)    // cfg2 sub2     [32,8,8,4,8,TMA,16], lane-sum group 4
DDP_AOT_INTEG(16, 2, 1, 0, 16, 256)    // integrate     [16|64,2,16,2,1,direct,16]
DDP_AOT_SNR(8, 1, 1, 0, 8, 256)        // snr cfg1/cfg2 [64,2,8,1,1,direct,8]
DDP_AOT_SNR(8, 1, 2, 0, 8, 256)        // snr cfg3      [32,8,8,1,2,direct,8]
DDP_AOT_INTEG(16, 1, 1, 0, 16, 256)    // integrate cfg2 [16,2,16,1,1,direct,16]
DDP_AOT_SNR(8, 1, 1, 0, 16, 256)       // snr cfg2      [64,4,8,1,1,direct,16]
