/* ddp_static.h -- ONE entry point of the library that allocates nothing (libddp_static.so).
 *
 * Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it.  The plan API of ddp.h never allocates either, but it needs a caller-provided workspace for the
 * subband intermediate; this call needs none: the intermediate S of the two-step subband dedispersion
 * (reading SB.1) lives in a file-scope `static __device__` array of
 * DDP_STATIC_SCRATCH_BYTES inside the library.  Every GPU that loads the library holds that array until the
 * process exits.
 *
 * What it computes (the same sums as ddp_dedisperse on a subband plan, bit-identical):
 *   S[a][s][t] = sum_{c in subband s} in[c][t + d1[a][c]]        0 <= t < nsamp_out + max_d2   (scratch, uint32)
 *   out[a*n_fine + b][t] = sum_s S[a][s][t + d2[b][s]]            0 <= t < nsamp_out
 * Coarse trials are processed in groups as large as the scratch holds, so only ONE coarse trial's intermediate
 * (n_subbands rows of round_up(nsamp_out + max_d2 + 32, 32) uint32) has to fit; a larger one is rejected with
 * DDP_STATIC_E_TOO_LARGE.  The kernels are the generic (direct-load) shapes of the library's dedispersion
 * template: correct for every geometry, not the tuned ones.
 *
 * Sharing: every call on a device uses the same array, which keeps the last call's contents.  Nothing in it has to
 * start at zero: step 1 writes every element step 2 uses in the same call.  Calls that overlap on one GPU (two
 * streams, two threads) RACE on the array: serialise them (one stream, or events between them).
 * The call launches kernels on `stream` and returns without synchronising; it calls no cudaMalloc, cudaFree or
 * any allocating routine (at the first call on a device it resolves the array's device address with
 * cudaGetSymbolAddress, once).
 */
#ifndef DDP_STATIC_H_
#define DDP_STATIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DDP_STATIC_SCRATCH_BYTES (16u << 20) /* 16 MiB per GPU */

enum {
    DDP_STATIC_OK = 0,
    DDP_STATIC_E_ARG = -1,       /* NULL pointer, non-positive size, n_subbands does not divide nchan         */
    DDP_STATIC_E_SHAPE = -2,     /* stride too small / not a multiple of 16 (in) or 4 (out), misaligned pointer */
    DDP_STATIC_E_TOO_LARGE = -3, /* one coarse trial's intermediate exceeds DDP_STATIC_SCRATCH_BYTES            */
    DDP_STATIC_E_CUDA = -4       /* a CUDA runtime call failed (no device, launch error)                       */
};

/* d_in   device, uint8 [nchan][in_stride], time fastest; in_stride >= round_up(nsamp_out + max_d1 + max_d2 + 32, 16),
 *        a multiple of 16, d_in 16-byte aligned (what ddp_plan_query reports as in_stride_min for the same plan).
 * d_d1   device, int32 [n_coarse][nchan]: step-1 delays (ddp_plan_get_delays(plan, 1, ...) uploaded by the caller);
 *        max_d1 >= every entry.  d_d2 device, int32 [n_fine][n_subbands]: step-2 delays; max_d2 >= every entry.
 *        Entries must be >= 0 and non-decreasing along the trial index (as the plan's tables are).
 * d_out  device, uint32 [n_coarse * n_fine][out_stride], out_stride >= round_up(nsamp_out, 4), a multiple of 4,
 *        16-byte aligned; columns >= nsamp_out are not written.
 * stream a CUstream / cudaStream_t (NULL = the default stream).
 * Returns DDP_STATIC_OK or a negative code; ddp_static_last_error() has the text (per thread). */
int ddp_static_subband_dedisperse(const uint8_t* d_in, size_t in_stride, int nchan, int n_subbands,
                                  const int32_t* d_d1, int n_coarse, int max_d1,
                                  const int32_t* d_d2, int n_fine, int max_d2,
                                  int nsamp_out, uint32_t* d_out, size_t out_stride, void* stream);

/* DDP_STATIC_SCRATCH_BYTES as the library was built. */
size_t ddp_static_scratch_bytes(void);

/* Text of the calling thread's last failure ("" if none). */
const char* ddp_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DDP_STATIC_H_ */
