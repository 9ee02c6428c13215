// Internal declarations shared by the host translation units of libddp (not part of the ABI).
#ifndef DDP_INTERNAL_H_
#define DDP_INTERNAL_H_

#include <cstdint>
#include <functional>
#include <map>
#include <string>
#include <unordered_map>
#include <utility>
#include <vector>

#include "../../include/ddp.h"
#include "ddp_params.h"

// Gene candidate arrays (BJ:cfg4; powers of two).
static const int DDP_CAND_THREADS_T[] = {16, 32, 64, 128, 256, 512, 1024};
static const int DDP_CAND_THREADS_DM[] = {1, 2, 4, 8, 16, 32};
static const int DDP_CAND_SPT[] = {1, 2, 4, 8, 16};
static const int DDP_CAND_DPT[] = {1, 2, 4, 8, 16};
static const int DDP_CAND_UNROLL[] = {1, 2, 4, 8, 16};
static const int DDP_CAND_STAGING[] = {0, 1, 2, 3, 4};
static const int DDP_CAND_VEC[] = {1, 4, 8, 16};
#define DDP_NGENES 7
struct DdpGeneDomain { const int* v; int n; };
const DdpGeneDomain* ddp_gene_domains();        // [DDP_NGENES], struct order of ddp_kcfg
int* ddp_gene_ptr(ddp_kcfg* c, int gene);
int ddp_gene_get(const ddp_kcfg& c, int gene);
int ddp_gene_index(int gene, int value);        // -1 if not a candidate

#define DDP_SMEM_LIMIT 232448                   // 227 KB per CTA on sm_100a

// Geometry of one kernel as the validity rules see it.
struct DdpKGeom {
    int ns_k;      // time-axis length the kernel tiles
    int ndm_k;     // DM-axis length the kernel tiles
    int nred;      // reduction trip count (0 = no reduction loop rule)
    int in_bytes;  // bytes per input element (1, 2 or 4)
};

struct DdpCompiled;  // runtime kernel handle (ddp_rt.cpp)

// Merged staging (staging genes 3 / 4): per DM tile of TD trials and per group of G adjacent reduction rows,
// the distinct tuples of relative delays ("variants") and which variant every trial uses.  Depends on the
// delay table, TD and G only, so it is built once on the host and kept in the workspace, instead of being
// rediscovered by every block.  blob = one record of rw int32 words per (tile t < ntiles, global group
// gg < ngg = rows / G), tile-major:
//   [0] variants   [1] span = delta of the last live trial   [2..3] 0
//   [4 .. 4+G)        delay of the tile's first trial for the G rows      (window starts)
//   [4+G .. 4+2G)     delay of the tile's last live trial                 (window ends)
//   [4+2G .. +vcap)   per variant: tau[1..G) as signed bytes (tau[0] = 0)
//   [.. + TD)         per trial: variant << 24 | delta
// delta = d[j][r0] - d[first trial][r0]; tau[m] = (d[j][r0+m] - d[j][r0]) - (same for the tile's first trial).
struct DdpMergeTable {
    int vmax = 0, vcap = 0, rw = 0, ntiles = 0, ngg = 0;
    std::vector<int32_t> nvar;                 // [ntiles][ngg]
    mutable std::map<int, int> rows_max;       // chunk length U -> largest sum of variants over a chunk's groups
    mutable std::vector<unsigned char> blob;   // device image, built by ddp_merge_table_blob on first launch
};

struct ddp_plan {
    // problem
    int nchan = 0, ndm = 0, nwidths = 0, ns = 0;
    double tsamp = 0;
    std::vector<double> freq, dms;
    int widths[DDP_MAX_WIDTHS] = {0};
    bool subband = false;
    int nsub = 0, ncoarse = 0, nfine = 0, cps = 0;
    double coarse_first = 0, coarse_step = 0, fine_step = 0;
    int ddof = 0, device = 0;
    int subband_ref = 0;                   // DDP_SUBREF_TOP / DDP_SUBREF_CENTRE (SB.2)
    int in_bytes = 1;                      // bytes per input sample: 1 (uint8, DD.6) or 2 (uint16, INPUT_BITS = 16)
    int integ_mode = 0;                    // DDP_INTEG_DECIMATE / DDP_INTEG_SLIDING
    std::vector<unsigned char> chan_mask;  // empty = every channel used; else nchan bytes, 0 = left out
    std::vector<int32_t> rowmap_host;      // host copy of the row map (outlives the asynchronous upload)
    int32_t* d_rowmap = nullptr;           // device: input row of every reduction row, -1 = masked (null without a mask)
    unsigned char* d_zero_row = nullptr;   // device: in_stride_min zero bytes a masked row reads
    std::string cache_dir;
    // host tables
    std::vector<int32_t> delay, d1, d2;
    ddp_plan_info info;
    // configurations + validity caches
    ddp_kcfg kcfg[DDP_K_COUNT];
    mutable std::map<int, int> spread_cache[3];              // dedisp kernel -> (TD -> max window spread)
    mutable std::map<int, std::pair<int, int>> diag_cache;   // step 1, TD -> (max spread of the delays relative to a subband's first row, max shift D_last - D_first), (-1, -1) = not usable
    mutable std::map<std::pair<int, int>, DdpMergeTable> merge_tables[3];  // host copies, built on first use
    int64_t merge_capacity = 0;                               // bytes of the workspace region for the resident table
    unsigned char* d_merge = nullptr;                         // device: resident merge table (one (kernel, TD, G) at a time)
    int merge_resident[3] = {-1, 0, 0};                       // (which, TD, G) of the table at d_merge
    mutable std::vector<ddp_kcfg> valid[DDP_K_COUNT];
    mutable bool valid_built[DDP_K_COUNT] = {false, false, false, false, false};
    // device side (ddp_rt.cpp)
    void* ws = nullptr;
    size_t ws_bytes = 0;
    int32_t *d_delay = nullptr, *d_d1 = nullptr, *d_d2 = nullptr;
    uint32_t* d_sub = nullptr;
    DdpCompiled* active[DDP_K_COUNT] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    void* rt = nullptr;  // per-plan runtime state (events), owned by ddp_rt.cpp
    mutable std::string err;
};

// ---- ddp_plan.cpp (pure host)
DdpKGeom ddp_kgeom(const ddp_plan* p, ddp_kernel k);
bool ddp_kernel_in_plan(const ddp_plan* p, ddp_kernel k);
int ddp_spread_max(const ddp_plan* p, ddp_kernel k, int TD);           // dedisp kernels only
int ddp_slide_nb(const ddp_plan* p, const ddp_kcfg& c);                 // sliding boxcar kernel: prefix-sum ring length in chunks
int ddp_dedisp_win(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c);  // staged row window (elements)
size_t ddp_smem_bytes(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c);
bool ddp_u8_single_buffered(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c);  // packed uint8 kernel: one copy buffer
// Subband step 1, packed uint8 kernel: time tiles aligned to the input with a per-trial output shift (code flag
// bit 6, "DIAG").  *shift_max = largest D_last - D_first over the DM tiles and subbands (extra time tiles of the grid).
bool ddp_sub1_diag(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, int* rel_spread = nullptr, int* shift_max = nullptr);
// Merged staging (staging genes 3 / 4: G = 2 / 4 adjacent rows pre-summed exactly; uint8 dedispersion only).
inline int ddp_merge_group(const ddp_kcfg& c) { return c.staging == 3 ? 2 : (c.staging == 4 ? 4 : 0); }
// producer warps the merged kernel adds to its threads_t x threads_dm consumer threads (4 or 12 warps)
inline int ddp_merge_producer_threads(const ddp_kcfg& c) { return c.threads_t * c.threads_dm >= 512 ? 384 : 128; }
int ddp_merge_vmax(const ddp_plan* p, ddp_kernel k, int TD, int G);  // largest number of distinct relative-shift tuples
struct DdpMergeGeom { int vmax, vcap, rw, rows_max, lw, le; };
int64_t ddp_merge_table_bytes(const ddp_plan* p, ddp_kernel k, int TD, int G);
int ddp_merge_rows_max(const ddp_plan* p, ddp_kernel k, int TD, int G, int U);
const DdpMergeTable& ddp_merge_table(const ddp_plan* p, ddp_kernel k, int TD, int G);         // counts only
const std::vector<unsigned char>& ddp_merge_table_blob(const ddp_plan* p, ddp_kernel k, int TD, int G);
DdpMergeGeom ddp_merge_geom(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c);
#define DDP_MERGE_VMAX_LIMIT 32                 // variants per group the kernel's tables allow
bool ddp_kcfg_valid(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, std::string* why);
const std::vector<ddp_kcfg>& ddp_valid_set(const ddp_plan* p, ddp_kernel k);
bool ddp_kcfg_equal(const ddp_kcfg& a, const ddp_kcfg& b);
ddp_kernel ddp_slot_kernel(const ddp_plan* p, int slot);               // slot -> kernel, DDP_K_COUNT if unused
ddp_status ddp_fail(const ddp_plan* p, ddp_status s, const std::string& msg);

// ---- ddp_rt.cpp (CUDA)
void ddp_rt_release(ddp_plan* p);
ddp_status ddp_rt_activate(ddp_plan* p, ddp_kernel k, const ddp_kcfg& c);  // compile/load, make active
// Hardware fitness of a joint configuration (median of summed CUDA-event times); only the slots in
// slot_mask are launched (brute force may time one kernel alone on the buffers of an earlier pass).
ddp_status ddp_rt_time_pipeline_mask(ddp_plan* p, const ddp_tune_io* io, const ddp_kcfg cfg[DDP_NSLOTS], unsigned slot_mask,
                                     double best_so_far, double* ms, double kernel_ms[DDP_NSLOTS], int64_t* n_timings);
// NVRTC-compiles (on all host cores) every code shape of the list that is not known yet.
void ddp_rt_precompile(const ddp_plan* p, const std::vector<std::pair<ddp_kernel, ddp_kcfg>>& list);
int64_t ddp_rt_compile_count();

#endif  // DDP_INTERNAL_H_
