/* ddp.h -- C ABI of the B200-native single-pulse-search hot path behind AMBER's auto-tuning
 * (arXiv:1811.04165): brute-force incoherent dedispersion (direct, and two-step subband), boxcar
 * integration over a set of pulse widths, per-(DM, width) S/N, and the three tuners (GA, brute
 * force, random) that time those kernels.
 *
 * Citations: P:n = PAPER.md line n; BJ = BASELINE.json (north_star / cfgN); DD.x SB.x INT.x SNR.x
 * GA.x = the readings listed in DESIGN.md.  The call list is the one BJ:north_star names
 * ("plan_create with the channel frequencies, t_samp, DM list and width set; dedisperse; integrate;
 * snr; tune_ga; tune_bruteforce; tune_random").
 *
 * General conventions
 *  - Every function returns a ddp_status (0 = OK, negative = error); no exceptions, no abort, no
 *    output on stdout/stderr.  ddp_last_error(plan) gives a plan-owned message for the last failure.
 *  - "host" pointers are ordinary CPU memory, "device" pointers are CUDA global memory of the
 *    plan's device.  ALL device memory (input, outputs, workspace) is allocated and owned by the
 *    caller; the plan owns only host tables and compiled kernels.  Compute calls never allocate,
 *    never synchronise and run asynchronously on `stream` (a cudaStream_t passed as void*; NULL =
 *    the legacy default stream).  tune_* calls synchronise on their own CUDA events.
 *  - A plan is used from one host thread at a time.
 *  - There is no CPU fallback: without a CUDA device every compute/tune call returns DDP_E_CUDA.
 *    Plan creation, geometry queries, configuration validity/repair/enumeration and the tuners
 *    driven by a caller-supplied fitness callback are pure host code and work without a GPU.
 */
#ifndef DDP_H_
#define DDP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    DDP_OK = 0,
    DDP_E_ARG = -1,       /* NULL / non-finite / out-of-range argument                          */
    DDP_E_SHAPE = -2,     /* stride or buffer too small or misaligned for the plan               */
    DDP_E_OVERFLOW = -3,  /* uint32 accumulation (255*nchan*max_w) or S/N moments could overflow */
    DDP_E_WORKSPACE = -4, /* workspace not bound or too small                                    */
    DDP_E_CONFIG = -5,    /* kernel configuration invalid for this plan (never silently repaired)*/
    DDP_E_COMPILE = -6,   /* NVRTC compilation / module load failed                              */
    DDP_E_CUDA = -7,      /* CUDA runtime/driver error or no device                              */
    DDP_E_BUDGET = -8     /* tuner: evaluation budget is zero or exhausted before any result     */
} ddp_status;

typedef struct ddp_plan ddp_plan; /* opaque; created by ddp_plan_create, freed by ddp_plan_destroy */

#define DDP_MAX_WIDTHS 16

/* The kernels of the pipeline (two-step de-dispersion, downsampling, S/N; one-step
 * de-dispersion P:237). */
typedef enum {
    DDP_K_DIRECT = 0,    /* one-step dedispersion, channels -> DM trials */
    DDP_K_SUB1 = 1,      /* step one: channels -> subbands at the coarse DMs     */
    DDP_K_SUB2 = 2,      /* step two: subbands -> fine DM trials per coarse DM     */
    DDP_K_INTEGRATE = 3, /* decimating boxcar sums per width   */
    DDP_K_SNR = 4,       /* (max-mean)/std per (DM, width)                        (BJ:cfg0)     */
    DDP_K_ISNR = 5,      /* integration and S/N in one pass over the dedispersed series; not a
                            slot of the tuners' joint configuration (BJ:cfg4 names four kernels)              */
    DDP_K_COUNT = 6
} ddp_kernel;

/* One "kernel chromosome" (gene set and value ranges from BJ:cfg4, cf. Table 3):
 *   threads_t   threads of a block along time     {16,32,...,1024}   (nrSamplesPerBlock, nrThreadsD0)
 *   threads_dm  threads of a block along DM       {1,2,...,32}       (nrDMsPerBlock)
 *   samples_per_thread {1,2,4,8,16}                                   (nrSamplesPerThread, nrItemsD0)
 *   dms_per_thread     {1,2,4,8,16}                                   (nrDMsPerThread)
 *   unroll      reduction-loop unroll / rows per staging chunk {1,2,4,8,16}   (unroll)
 *   staging     how the delayed input window reaches the threads: 0 direct global loads,
 *               1 cooperative copy to shared memory, 2 TMA bulk copy to shared memory  (localMem);
 *               uint8 dedispersion kernels only: 3 / 4 = TMA bulk copy, then 2 / 4 adjacent channels are
 *               pre-summed EXACTLY in shared memory for every distinct tuple of their relative delays in
 *               the tile, and the trials add those partial sums (same integers as the plain sum)
 *   vec_bytes   width in bytes of one input load instruction {1,4,8,16}
 * All genes are powers of two. */
typedef struct {
    int threads_t, threads_dm, samples_per_thread, dms_per_thread, unroll, staging, vec_bytes;
} ddp_kcfg;

enum { DDP_STAGE_DIRECT = 0, DDP_STAGE_SMEM = 1, DDP_STAGE_TMA = 2, DDP_STAGE_TMA_MERGE2 = 3, DDP_STAGE_TMA_MERGE4 = 4 };

/* Options of ddp_plan_create; zero-initialise for a direct plan with defaults. */
typedef struct {
    int n_subbands;        /* 0 = direct plan; >0 = two-step subband plan (must divide nchan; SB.3) */
    int n_coarse;          /* subband plan: number of coarse ("subbanding") DMs     */
    double coarse_dm_first;/*               first coarse DM     */
    double coarse_dm_step; /*               coarse DM step     */
    int n_fine;            /*               fine DMs per coarse DM     */
    double fine_dm_step;   /*               fine DM step; fine offsets are b*fine_dm_step  */
    int snr_ddof;          /* 0 = population std (default, SNR.2), 1 = sample std                     */
    int device;            /* CUDA device ordinal                                                      */
    const char* cache_dir; /* directory for compiled-kernel cubins; NULL = no disk cache               */
    int integration_mode;  /* DDP_INTEG_DECIMATE (0, default: block sums, stride w; INT.1) or DDP_INTEG_SLIDING (1:
                              stride-1 boxcar I^s_w[t] = sum_{k<w} Y[t+k], t <= nsamp_out - w).  In sliding
                              mode the sums are never materialised: only ddp_integrate_snr (d_integ = NULL) and the
                              search calls run; ddp_integrate, ddp_snr and the tuners return DDP_E_CONFIG         */
    const uint8_t* chan_mask; /* host, nchan bytes or NULL: channels whose byte is 0 are left out of every sum
                              (zapped channels); copied at plan creation                  */
    int subband_ref;       /* subband plan: frequency the step-2 delays of a subband are computed at (SB.2; the paper
                              does not say): DDP_SUBREF_TOP (0, default) = its highest channel frequency,
                              DDP_SUBREF_CENTRE (1) = (highest + lowest channel frequency of the subband) / 2
                              (SURVEY 8(c) SB.2 alternative, 8(f) f4).  Ignored by a direct plan                  */
    int input_bits;        /* bits per input sample (P:90 INPUT_BITS): 0 or 8 = unsigned 8-bit (default, DD.6), 16 =
                              unsigned 16-bit.  With 16 every `uint8_t* in` argument of this header
                              points at uint16 elements, strides stay in ELEMENTS, sums stay uint32 (plan creation
                              proves 65535 * nchan * max width < 2^32), the subband intermediate is uint32, and the
                              merged staging genes (3, 4) are not valid                                           */
} ddp_options;
enum { DDP_INTEG_DECIMATE = 0, DDP_INTEG_SLIDING = 1 };
enum { DDP_SUBREF_TOP = 0, DDP_SUBREF_CENTRE = 1 };

/* Geometry of a plan (all counts in elements unless named *_bytes). */
typedef struct {
    int subband;                 /* 0 direct, 1 two-step                                               */
    int nchan, ndm, nwidths, nsamp_out;
    int n_subbands, n_coarse, n_fine;
    int max_delay;               /* direct: max delay[i][c]; subband: max d1 + max d2   (DD.5, SB.5)   */
    int max_d1, max_d2;          /* subband tables' maxima (0 for a direct plan)                        */
    int64_t nsamp_in_required;   /* samples every channel row must hold = nsamp_out + max_delay         */
    int64_t in_stride_min;       /* smallest legal in_stride (a multiple of 16)                         */
    int64_t out_stride_min;      /* smallest legal out_stride (a multiple of 4)                         */
    int64_t nsamp_sub;           /* subband: samples per intermediate row = nsamp_out + max_d2 (SB.4)   */
    int64_t sub_stride;          /* subband: element stride of the intermediate rows                    */
    int widths[DDP_MAX_WIDTHS];
    int64_t plane_len[DDP_MAX_WIDTHS];    /* values per series: floor(nsamp_out / w) (INT.2); sliding mode: nsamp_out - w + 1 */
    int64_t plane_stride[DDP_MAX_WIDTHS]; /* row stride of plane w in d_integ; 0 for w == 1            */
    int64_t plane_offset[DDP_MAX_WIDTHS]; /* element offset of plane w in d_integ; -1 for w == 1       */
    int64_t integ_elems;         /* uint32 elements the caller allocates for d_integ                    */
    int64_t workspace_bytes;     /* bytes the caller allocates for ddp_plan_bind_workspace              */
    double adds_dedisp;          /* algorithmic integer adds of one dedisperse call                     */
    int sub_elem_bytes;          /* subband: bytes per element of the intermediate S: 2 (uint16) when
                                    255 * channels-per-subband <= 65535 makes that exact, else 4 (SB.4)  */
    int integration_mode;        /* DDP_INTEG_DECIMATE or DDP_INTEG_SLIDING                               */
    int nchan_masked;            /* channels left out by the plan's channel mask                          */
    int subband_ref;             /* DDP_SUBREF_TOP or DDP_SUBREF_CENTRE (0 for a direct plan)                */
    int input_bits;              /* 8 or 16: width of one input sample                                       */
} ddp_plan_info;

/* ---- plan -------------------------------------------------------------------------------------
 * chan_freq_mhz[nchan]  host, channel centre frequencies in MHz, any order, finite and > 0.
 * t_samp_s              sampling time in seconds (> 0).
 * dm_list[ndm]          host, trial DMs in pc cm^-3, non-negative and non-decreasing (direct plan).
 *                       For a subband plan pass NULL (ndm is then n_coarse*n_fine and trial
 *                       a*n_fine+b has DM coarse_first + a*coarse_step + b*fine_step), or the
 *                       identical grid (checked).
 * widths[nwidths]       host, strictly increasing boxcar widths, each a power of two (1, 2, 4, ...;
 *                       INT.3: BJ configs; the paper's own factor list is garbled),
 *                       nwidths <= DDP_MAX_WIDTHS.
 * nsamp_out             output samples per DM trial (> 0); floor(nsamp_out / max width) >= 2.
 * Delay tables (DD.1-DD.3): delay[i][c] = floor(((4.148808e3*DM[i]) * (f[c]^-2 - f_ref^-2)) / t_samp + 0.5)
 * in float64, f_ref = max_c f[c].  Errors: DDP_E_ARG, DDP_E_SHAPE (nchan % n_subbands),
 * DDP_E_OVERFLOW (255*nchan*max_w >= 2^32, or (255*nchan)^2*max_w*nsamp_out >= 2^64). */
ddp_status ddp_plan_create(ddp_plan** out, const double* chan_freq_mhz, int nchan, double t_samp_s,
                           const double* dm_list, int ndm, const int* widths, int nwidths,
                           int nsamp_out, const ddp_options* opt);
ddp_status ddp_plan_destroy(ddp_plan* plan);

/* Host-only geometry queries. */
ddp_status ddp_plan_query(const ddp_plan* plan, ddp_plan_info* out);
/* step 0: direct table [ndm][nchan]; 1: d1 [n_coarse][nchan]; 2: d2 [n_fine][n_subbands]. host_out is
 * caller-owned host memory of that many int32. */
ddp_status ddp_plan_get_delays(const ddp_plan* plan, int step, int32_t* host_out);

/* Hands the plan `bytes` (>= workspace_bytes, 256-byte aligned) of caller-owned DEVICE memory and
 * uploads the delay tables into it on `stream` (asynchronously; the host tables outlive the copy).
 * The workspace also holds the subband intermediate S.  Must be called before any compute or
 * (real-hardware) tune call; the memory must stay valid until plan destroy or re-bind. */
ddp_status ddp_plan_bind_workspace(ddp_plan* plan, void* d_workspace, size_t bytes, void* stream);

/* ---- compute (device pointers, asynchronous on stream) ------------------------------------------
 * ddp_dedisperse: d_in uint8 [nchan][in_stride] time-fastest, row c = channel c of chan_freq_mhz;
 *   in_stride >= in_stride_min and a multiple of 16, d_in 16-byte aligned (vector/TMA loads).
 *   d_out uint32 [ndm][out_stride], out_stride >= out_stride_min, multiple of 4, d_out 16-byte aligned.
 *   Direct plan (DD): out[i][t] = sum_c in[c][t + delay[i][c]], 0 <= t < nsamp_out.
 *   Subband plan (SB.1): S[a][s][t] = sum_{c in s} in[c][t + d1[a][c]] into the workspace, then
 *   out[a*n_fine+b][t] = sum_s S[a][s][t + d2[b][s]].  Columns t >= nsamp_out are not written. */
ddp_status ddp_dedisperse(ddp_plan* plan, const uint8_t* d_in, size_t in_stride, uint32_t* d_out,
                          size_t out_stride, void* stream);
/* ddp_integrate (INT.1, INT.2): for every width w > 1, plane w of d_integ (layout from ddp_plan_query)
 *   I_w[i][j] = sum_{k<w} dedisp[i][j*w + k], 0 <= j < floor(nsamp_out / w).  The w == 1 plane is
 *   d_dedisp itself and is not copied. */
ddp_status ddp_integrate(ddp_plan* plan, const uint32_t* d_dedisp, size_t stride, uint32_t* d_integ,
                         void* stream);
/* ddp_snr (SNR.1-SNR.4): d_snr float32 [ndm][nwidths], d_argmax uint32 [ndm][nwidths] (may be NULL):
 *   snr = (max - mean)/std over the n_w values of (DM, width), std with the plan's ddof, computed
 *   from exact integer moments, finished in float64, rounded once to float32; argmax = lowest index
 *   of the maximum; a constant series gives snr = 0, argmax = 0. */
ddp_status ddp_snr(ddp_plan* plan, const uint32_t* d_dedisp, size_t stride, const uint32_t* d_integ,
                   float* d_snr, uint32_t* d_argmax, void* stream);
/* ddp_integrate_snr (INT.1-2, SNR.1-4): integration and S/N in ONE kernel.  The dedispersed series
 *   is read once; the block sums of every width are formed in registers and fed straight into the exact integer
 *   moment / max accumulators of their width, so d_snr / d_argmax hold bit for bit what ddp_integrate followed by
 *   ddp_snr gives.  d_integ may be NULL: the planes are then never written (that is the point: at BJ:cfg1 they
 *   are 199 MB written and read again); when it is given, the planes are stored too, identical to ddp_integrate's.
 *   Kernel configuration DDP_K_ISNR: threads_t = 32 (one warp per series), threads_dm series per block,
 *   samples_per_thread in {4, 8, 16}, dms_per_thread series per warp one after the other; the other genes are pinned. */
ddp_status ddp_integrate_snr(ddp_plan* plan, const uint32_t* d_dedisp, size_t stride, uint32_t* d_integ, float* d_snr,
                             uint32_t* d_argmax, void* stream);
/* One whole search through HOST buffers (the end-to-end path): copies h_in (uint8 [nchan][in_stride],
 * pinned or pageable host memory) into the caller's device buffer d_in, runs dedisperse -> integrate
 * -> snr on `stream` (d_integ == NULL: dedisperse -> ddp_integrate_snr, no planes), copies the S/N table (and
 * argmax if h_argmax != NULL) back to the host and synchronises the stream before returning.  Device buffers as
 * for the calls above. */
ddp_status ddp_search_host(ddp_plan* plan, const uint8_t* h_in, size_t in_stride, uint8_t* d_in,
                           uint32_t* d_out, size_t out_stride, uint32_t* d_integ, float* d_snr,
                           uint32_t* d_argmax, float* h_snr, uint32_t* h_argmax, void* stream);
/* Consecutive batches of one observation: h_in is uint8 [nchan][h_stride] host memory
 * (pinned for the copies to overlap) holding at least nbatches*nsamp_out + max_delay samples per channel; batch b
 * searches samples [b*nsamp_out, (b+1)*nsamp_out + max_delay) -- exactly the columns b*nsamp_out.. of one long
 * dedispersion.  Only the nsamp_out NEW samples of a batch are uploaded: the max_delay samples shared with the
 * previous batch are carried over on the device between the two input buffers d_in0 / d_in1 (each uint8
 * [nchan][in_stride], as for ddp_dedisperse), and the upload of batch b+1 runs on a plan-owned copy stream while
 * batch b is searched on `stream` (dedisperse -> ddp_integrate_snr, no planes).  h_snr float32 [nbatches][ndm]
 * [nwidths]; h_argmax likewise or NULL.  Both streams are synchronised before returning. */
ddp_status ddp_search_host_batches(ddp_plan* plan, const uint8_t* h_in, size_t h_stride, int nbatches,
                                   uint8_t* d_in0, uint8_t* d_in1, size_t in_stride, uint32_t* d_out,
                                   size_t out_stride, float* d_snr, uint32_t* d_argmax, float* h_snr,
                                   uint32_t* h_argmax, void* stream);
/* Debug accessor: device pointer of the subband intermediate S[n_coarse][n_subbands][sub_stride]
 * (elements of sub_elem_bytes bytes: uint16 or uint32) inside the bound workspace (NULL for a direct
 * plan or before bind). */
ddp_status ddp_plan_subband_buffer(const ddp_plan* plan, void** d_sub);

/* ---- kernel configurations ----------------------------------------------------------------------
 * Validity rules V1-V7 are listed in DESIGN.md (from P:136-152 and the sm_100a limits). */
ddp_status ddp_get_kcfg(const ddp_plan* plan, ddp_kernel k, ddp_kcfg* out);
/* Validates, then (on a machine with a GPU) compiles/loads the kernel; DDP_E_CONFIG if invalid. */
ddp_status ddp_set_kcfg(ddp_plan* plan, ddp_kernel k, const ddp_kcfg* cfg);
/* DDP_OK if valid for this plan, DDP_E_CONFIG otherwise (pure host). */
ddp_status ddp_check_kcfg(const ddp_plan* plan, ddp_kernel k, const ddp_kcfg* cfg);
/* Moves *inout to the nearest valid configuration (BJ:cfg4 "repaired to the nearest valid one";
 * deterministic, idempotent, identity on valid input, total). */
ddp_status ddp_repair_kcfg(const ddp_plan* plan, ddp_kernel k, ddp_kcfg* inout);
/* Compiles the code shape of (k, cfg) for sm_100a with NVRTC (host only, no GPU needed; the cubin
 * goes to the plan's cache_dir when one is set).  DDP_E_CONFIG / DDP_E_COMPILE (log in ddp_last_error). */
ddp_status ddp_compile_kcfg(ddp_plan* plan, ddp_kernel k, const ddp_kcfg* cfg);
/* Brute-force space of kernel k: every valid configuration, canonical order.  Writes at most
 * `cap` entries to out (may be NULL) and the total count to *n. */
ddp_status ddp_enumerate_kcfgs(const ddp_plan* plan, ddp_kernel k, ddp_kcfg* out, size_t cap, size_t* n);

/* ---- tuning --------------------------------------------------------------------------------------
 * A joint configuration is 4 ddp_kcfg in pipeline order: [0] sub1 (or direct for a direct plan),
 * [1] sub2 (ignored for a direct plan), [2] integrate, [3] snr  ("all four kernels"). */
#define DDP_NSLOTS 4

/* Fitness callback for tests and external drivers: returns the cost (ms; lower is better, +inf =
 * failed) of a joint configuration.  NULL = the built-in CUDA-event harness (
 * BJ:cfg4 "summed CUDA-event time of the four kernels, median of 5 runs"). */
typedef double (*ddp_fitness_fn)(void* user, const ddp_kcfg cfg[DDP_NSLOTS]);

typedef struct {
    const uint8_t* d_in; size_t in_stride;       /* device buffers as for the compute calls          */
    uint32_t* d_out; size_t out_stride;
    uint32_t* d_integ;
    float* d_snr; uint32_t* d_argmax;
    void* stream;
    void* d_flush; size_t flush_bytes;            /* optional: written before each timed pass (L2)    */
    ddp_fitness_fn fitness; void* user;           /* non-NULL: use instead of the hardware harness    */
    int reps;                                     /* timed passes per evaluation (default 5)          */
    int warmup;                                   /* untimed passes per evaluation (default 1)        */
    double cutoff_factor;                         /* >0: abandon an evaluation whose first timed pass
                                                     exceeds cutoff_factor x best-so-far (0 = never)  */
} ddp_tune_io;

typedef struct {
    uint64_t seed;
    int population;      /* N_pop (BJ:cfg4 64; paper 20)                                        */
    int generations;     /* BJ:cfg4 50                                                                  */
    int tournament;      /* pool size (BJ:cfg4 3; paper 20% of N_pop)                            */
    double p_cross;      /* per-kernel crossover probability (0.8)                               */
    int crossover_kind;  /* 0 uniform "coin toss" (P:197b), 1 one-point (P:197a)                        */
    double p_mut;        /* mutation probability (BJ:cfg4 0.05 per gene; paper 0.1 per kernel)   */
    int mutation_kind;   /* 0 per gene (BJ:cfg4), 1 per kernel (paper)                                  */
    int elitism;         /* parents copied unchanged (BJ:cfg4 2)                                        */
    int replacement;     /* 0 elitism + offspring (BJ:cfg4), 1 best half of parents and of offspring */
    int64_t max_evals;   /* cap on fitness calls (0 = population + generations*(population-elitism))    */
} ddp_ga_params;

typedef struct {
    int64_t max_evals_per_kernel; /* 0 = every valid configuration; else an evenly strided subset     */
    int isolated;                 /* 0: candidate timed inside the whole pipeline (other kernels at the
                                     plan's current configuration); 1: the kernel under test alone     */
    unsigned slots;               /* bit s set: search pipeline slot s (0 = all slots); slots left out
                                     keep the plan's current configuration (resumable campaigns)        */
} ddp_bf_params;
typedef struct { uint64_t seed; int64_t max_evals; } ddp_rand_params;

typedef struct {
    ddp_kcfg best[DDP_NSLOTS];
    double best_ms;                 /* fitness of `best` (for brute force: the four winners timed together) */
    double kernel_ms[DDP_NSLOTS];   /* per-kernel medians of `best` (hardware harness only, else 0)    */
    int64_t n_fitness_calls;        /* evaluations of not-yet-seen candidates (GA/random: joint; BF: per kernel) */
    int64_t n_kernel_timings;       /* kernel launches timed                                            */
    int64_t n_compiles;             /* NVRTC compilations                                               */
    double wall_seconds;
    double* history; size_t history_cap; size_t history_len; /* caller array: best-so-far after each fitness call */
    double sum_isolated_min_ms;     /* brute force: sum of the per-kernel minima (GA.6)                 */
    /* optional, caller arrays ("configurations at the end of every algorithm run"): the GA's last population,
       best first -- random search: the last final_cap configurations it drew -- as final_len joint configurations
       of DDP_NSLOTS ddp_kcfg each, with their fitness values; final_pop == NULL: not recorded */
    ddp_kcfg* final_pop; double* final_fit; size_t final_cap; size_t final_len;
} ddp_tune_result;

ddp_status ddp_tune_ga(ddp_plan* plan, const ddp_tune_io* io, const ddp_ga_params* p, ddp_tune_result* res);
ddp_status ddp_tune_bruteforce(ddp_plan* plan, const ddp_tune_io* io, const ddp_bf_params* p, ddp_tune_result* res);
ddp_status ddp_tune_random(ddp_plan* plan, const ddp_tune_io* io, const ddp_rand_params* p, ddp_tune_result* res);
/* One fitness evaluation of a joint configuration with the hardware harness (or io->fitness):
 * *ms = median over io->reps passes of the summed kernel times; kernel_ms[4] per-kernel medians. */
ddp_status ddp_time_pipeline(ddp_plan* plan, const ddp_tune_io* io, const ddp_kcfg cfg[DDP_NSLOTS],
                             double* ms, double kernel_ms[DDP_NSLOTS]);

const char* ddp_status_str(ddp_status s);        /* static string                                     */
const char* ddp_last_error(const ddp_plan* plan);/* plan-owned, valid until the next call on the plan  */
const char* ddp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DDP_H_ */
