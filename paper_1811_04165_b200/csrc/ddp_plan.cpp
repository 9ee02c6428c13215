// Host-only part of libddp: plan creation (delay tables, geometry), kernel-configuration validity,
// nearest-valid repair and brute-force enumeration.  No CUDA calls here.
//
// P:n = PAPER.md line n; BJ = BASELINE.json; readings DD.x/SB.x/INT.x/SNR.x and rules V1-V7 are
// listed in DESIGN.md.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>

#include "ddp_internal.h"

// ------------------------------------------------------------------------------------ genes
static const DdpGeneDomain kDomains[DDP_NGENES] = {
    {DDP_CAND_THREADS_T, 7}, {DDP_CAND_THREADS_DM, 6}, {DDP_CAND_SPT, 5}, {DDP_CAND_DPT, 5},
    {DDP_CAND_UNROLL, 5},    {DDP_CAND_STAGING, 5},    {DDP_CAND_VEC, 4}};
const DdpGeneDomain* ddp_gene_domains() { return kDomains; }
int* ddp_gene_ptr(ddp_kcfg* c, int gene) {
    switch (gene) {
        case 0: return &c->threads_t;
        case 1: return &c->threads_dm;
        case 2: return &c->samples_per_thread;
        case 3: return &c->dms_per_thread;
        case 4: return &c->unroll;
        case 5: return &c->staging;
        default: return &c->vec_bytes;
    }
}
int ddp_gene_get(const ddp_kcfg& c, int gene) { return *ddp_gene_ptr(const_cast<ddp_kcfg*>(&c), gene); }
int ddp_gene_index(int gene, int value) {
    for (int i = 0; i < kDomains[gene].n; ++i)
        if (kDomains[gene].v[i] == value) return i;
    return -1;
}
bool ddp_kcfg_equal(const ddp_kcfg& a, const ddp_kcfg& b) { return std::memcmp(&a, &b, sizeof(ddp_kcfg)) == 0; }

ddp_status ddp_fail(const ddp_plan* p, ddp_status s, const std::string& msg) {
    if (p) p->err = msg;
    return s;
}

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
static inline int pow2ceil(int x) {
    int p = 1;
    while (p < x) p <<= 1;
    return p;
}

// ------------------------------------------------------------------------------------ delays
// DD.1/DD.2 (BJ:north_star): floor(((K*DM) * (f^-2 - f_ref^-2)) / t_samp + 0.5) in float64, this
// association; this file is compiled with -ffp-contract=off.
static bool fill_delays(const double* f, int nf, double f_ref, const double* dm, int ndm, double tsamp,
                        std::vector<int32_t>& out, int* maxv) {
    const double kdm = 4.148808e3;
    const double inv_ref2 = 1.0 / (f_ref * f_ref);
    out.resize((size_t)ndm * nf);
    int mx = 0;
    for (int i = 0; i < ndm; ++i)
        for (int c = 0; c < nf; ++c) {
            const double g = 1.0 / (f[c] * f[c]) - inv_ref2;
            const double x = ((kdm * dm[i]) * g) / tsamp;
            const double r = std::floor(x + 0.5);
            if (!(r >= 0.0 && r < 1.0e9)) return false;
            const int32_t d = (int32_t)r;
            out[(size_t)i * nf + c] = d;
            if (d > mx) mx = d;
        }
    *maxv = mx;
    return true;
}

// ------------------------------------------------------------------------------------ plan
static void default_kcfgs(ddp_plan* p);

extern "C" ddp_status ddp_plan_create(ddp_plan** out, const double* chan_freq_mhz, int nchan, double t_samp_s,
                                      const double* dm_list, int ndm, const int* widths, int nwidths, int nsamp_out,
                                      const ddp_options* opt) {
    if (!out) return DDP_E_ARG;
    *out = nullptr;
    if (!chan_freq_mhz || nchan <= 0 || !widths || nwidths <= 0 || nwidths > DDP_MAX_WIDTHS || nsamp_out <= 0)
        return DDP_E_ARG;
    if (!(t_samp_s > 0.0) || !std::isfinite(t_samp_s)) return DDP_E_ARG;
    for (int c = 0; c < nchan; ++c)
        if (!(chan_freq_mhz[c] > 0.0) || !std::isfinite(chan_freq_mhz[c])) return DDP_E_ARG;
    for (int k = 0; k < nwidths; ++k) {
        if (widths[k] < 1) return DDP_E_ARG;
        if ((widths[k] & (widths[k] - 1)) != 0 || widths[k] >= (1 << (DDP_MAXW - 1))) return DDP_E_ARG;  // INT.3
        if (k > 0 && widths[k] <= widths[k - 1]) return DDP_E_ARG;
    }
    if (nsamp_out / widths[nwidths - 1] < 2) return DDP_E_ARG;

    ddp_plan* p = new ddp_plan();
    p->nchan = nchan;
    p->ns = nsamp_out;
    p->tsamp = t_samp_s;
    p->nwidths = nwidths;
    p->freq.assign(chan_freq_mhz, chan_freq_mhz + nchan);
    for (int k = 0; k < nwidths; ++k) p->widths[k] = widths[k];
    if (opt) {
        p->ddof = opt->snr_ddof;
        p->device = opt->device;
        if (opt->cache_dir) p->cache_dir = opt->cache_dir;
        p->integ_mode = opt->integration_mode;
        if (opt->chan_mask) p->chan_mask.assign(opt->chan_mask, opt->chan_mask + nchan);
        p->subband_ref = opt->subband_ref;
        if (opt->input_bits != 0 && opt->input_bits != 8 && opt->input_bits != 16) {
            delete p;
            return DDP_E_ARG;
        }
        p->in_bytes = opt->input_bits == 16 ? 2 : 1;
    }
    auto bail = [&](ddp_status s) {
        delete p;
        return s;
    };
    if (p->ddof != 0 && p->ddof != 1) return bail(DDP_E_ARG);
    if (p->integ_mode != DDP_INTEG_DECIMATE && p->integ_mode != DDP_INTEG_SLIDING) return bail(DDP_E_ARG);
    if (nsamp_out / widths[nwidths - 1] - p->ddof < 1) return bail(DDP_E_ARG);
    const double f_ref = *std::max_element(p->freq.begin(), p->freq.end());  // DD.3

    int max_delay = 0, max_d1 = 0, max_d2 = 0;
    if (opt && opt->n_subbands > 0) {
        p->subband = true;
        p->nsub = opt->n_subbands;
        p->ncoarse = opt->n_coarse;
        p->nfine = opt->n_fine;
        p->coarse_first = opt->coarse_dm_first;
        p->coarse_step = opt->coarse_dm_step;
        p->fine_step = opt->fine_dm_step;
        if (p->ncoarse <= 0 || p->nfine <= 0) return bail(DDP_E_ARG);
        if (!(p->coarse_first >= 0.0) || !(p->coarse_step >= 0.0) || !(p->fine_step >= 0.0)) return bail(DDP_E_ARG);
        if (!std::isfinite(p->coarse_first) || !std::isfinite(p->coarse_step) || !std::isfinite(p->fine_step))
            return bail(DDP_E_ARG);
        if (nchan % p->nsub != 0) return bail(DDP_E_SHAPE);  // SB.3
        if ((int64_t)p->ncoarse * p->nfine > (int64_t)std::numeric_limits<int>::max()) return bail(DDP_E_ARG);
        p->cps = nchan / p->nsub;
        p->ndm = p->ncoarse * p->nfine;
        if (dm_list && ndm != p->ndm) return bail(DDP_E_ARG);
        std::vector<double> A(p->ncoarse), F(p->nfine), fsub(p->nsub);
        for (int a = 0; a < p->ncoarse; ++a) A[a] = p->coarse_first + a * p->coarse_step;
        for (int b = 0; b < p->nfine; ++b) F[b] = b * p->fine_step;
        p->dms.resize(p->ndm);
        for (int a = 0; a < p->ncoarse; ++a)
            for (int b = 0; b < p->nfine; ++b) p->dms[(size_t)a * p->nfine + b] = A[a] + F[b];
        if (dm_list)
            for (int i = 0; i < p->ndm; ++i)
                if (dm_list[i] != p->dms[i]) return bail(DDP_E_ARG);
        if (p->subband_ref != DDP_SUBREF_TOP && p->subband_ref != DDP_SUBREF_CENTRE) return bail(DDP_E_ARG);
        for (int s = 0; s < p->nsub; ++s) {  // SB.2: subband reference = its highest channel frequency, or its centre
            const auto b = p->freq.begin() + (size_t)s * p->cps, e = b + p->cps;
            const double hi = *std::max_element(b, e);
            fsub[s] = p->subband_ref == DDP_SUBREF_CENTRE ? 0.5 * (hi + *std::min_element(b, e)) : hi;
        }
        if (!fill_delays(p->freq.data(), nchan, f_ref, A.data(), p->ncoarse, t_samp_s, p->d1, &max_d1)) return bail(DDP_E_ARG);
        if (!fill_delays(fsub.data(), p->nsub, f_ref, F.data(), p->nfine, t_samp_s, p->d2, &max_d2)) return bail(DDP_E_ARG);
        max_delay = max_d1 + max_d2;
    } else {
        if (!dm_list || ndm <= 0) return bail(DDP_E_ARG);
        for (int i = 0; i < ndm; ++i) {
            if (!(dm_list[i] >= 0.0) || !std::isfinite(dm_list[i])) return bail(DDP_E_ARG);
            if (i > 0 && dm_list[i] < dm_list[i - 1]) return bail(DDP_E_ARG);
        }
        p->ndm = ndm;
        p->dms.assign(dm_list, dm_list + ndm);
        if (!fill_delays(p->freq.data(), nchan, f_ref, dm_list, ndm, t_samp_s, p->delay, &max_delay)) return bail(DDP_E_ARG);
    }
    if ((int64_t)nsamp_out + max_delay + 64 >= (int64_t)1 << 31) return bail(DDP_E_ARG);

    // Overflow proofs (INT.5): uint32 sums and uint64 second moments must be exact.
    const int wmax = widths[nwidths - 1];
    const long double vmax = p->in_bytes == 2 ? 65535.0L : 255.0L;  // largest input sample
    if (vmax * nchan * wmax >= 4294967296.0L) return bail(DDP_E_OVERFLOW);
    if (p->integ_mode == DDP_INTEG_SLIDING) {
        // ns - w + 1 window sums of at most vmax * nchan * w each: their sum fits 64 bits, their squares' sum the
        // sliding kernel's 96 bits (DdpSlideMom)
        if (vmax * nchan * wmax * nsamp_out >= 18446744073709551616.0L) return bail(DDP_E_OVERFLOW);
        if (vmax * nchan * vmax * nchan * wmax * wmax * nsamp_out >= 79228162514264337593543950336.0L) return bail(DDP_E_OVERFLOW);
    } else if (vmax * nchan * vmax * nchan * wmax * nsamp_out >= 18446744073709551616.0L) {
        return bail(DDP_E_OVERFLOW);  // floor(ns / w) block sums of at most vmax * nchan * w: squares in 64 bits
    }

    ddp_plan_info& I = p->info;
    std::memset(&I, 0, sizeof(I));
    I.subband = p->subband ? 1 : 0;
    I.nchan = nchan;
    I.ndm = p->ndm;
    I.nwidths = nwidths;
    I.nsamp_out = nsamp_out;
    I.n_subbands = p->nsub;
    I.n_coarse = p->ncoarse;
    I.n_fine = p->nfine;
    I.max_delay = max_delay;
    I.max_d1 = max_d1;
    I.max_d2 = max_d2;
    I.nsamp_in_required = (int64_t)nsamp_out + max_delay;
    I.in_stride_min = round_up(I.nsamp_in_required + 32, 16);
    I.out_stride_min = round_up(nsamp_out, 4);
    I.nsamp_sub = p->subband ? (int64_t)nsamp_out + max_d2 : 0;
    I.sub_stride = p->subband ? round_up(I.nsamp_sub + 32, 32) : 0;
    // SB.4: the intermediate is stored as uint16 whenever that is exact (255 * channels per subband
    // fits 16 bits), which halves its HBM and shared-memory traffic; uint32 otherwise.
    I.sub_elem_bytes = p->subband ? (p->in_bytes == 1 && 255 * (int64_t)p->cps <= 65535 ? 2 : 4) : 0;
    I.input_bits = 8 * p->in_bytes;
    I.integration_mode = p->integ_mode;
    I.subband_ref = p->nsub > 0 ? p->subband_ref : 0;
    I.nchan_masked = 0;
    for (unsigned char m : p->chan_mask) I.nchan_masked += m == 0;
    int64_t off = 0;
    for (int k = 0; k < nwidths; ++k) {
        I.widths[k] = widths[k];
        I.plane_len[k] = p->integ_mode == DDP_INTEG_SLIDING ? nsamp_out - widths[k] + 1 : nsamp_out / widths[k];
        if (widths[k] == 1 || p->integ_mode == DDP_INTEG_SLIDING) {  // sliding sums are never materialised
            I.plane_stride[k] = 0;
            I.plane_offset[k] = -1;
        } else {
            I.plane_stride[k] = round_up(I.plane_len[k], 32);
            I.plane_offset[k] = off;
            off += I.plane_stride[k] * p->ndm;
        }
    }
    I.integ_elems = off;
    int64_t tbytes = p->subband ? round_up((int64_t)p->d1.size() * 4, 256) + round_up((int64_t)p->d2.size() * 4, 256)
                                : round_up((int64_t)p->delay.size() * 4, 256);
    int64_t sbytes = p->subband ? round_up((int64_t)p->ncoarse * p->nsub * I.sub_stride * I.sub_elem_bytes, 256) : 0;
    // region for the resident merged-staging table (one (kernel, TD, G) at a time; DdpMergeTable)
    p->merge_capacity = round_up(2 * (int64_t)(p->subband ? p->d1.size() : p->delay.size()) * 4 + (1 << 20), 256);
    // channel mask: row map (one int per channel) and the row of zeros a masked channel reads
    const int64_t mbytes = p->chan_mask.empty() ? 0 : round_up((int64_t)nchan * 4, 256) + round_up(I.in_stride_min * p->in_bytes, 256);
    I.workspace_bytes = tbytes + sbytes + p->merge_capacity + mbytes + 256;
    const double nused = (double)(nchan - I.nchan_masked);  // masked channels are not part of the algorithmic work
    I.adds_dedisp = p->subband ? (double)p->ncoarse * nused * (double)I.nsamp_sub + (double)p->ndm * p->nsub * nsamp_out
                               : (double)p->ndm * nused * nsamp_out;
    default_kcfgs(p);
    *out = p;
    return DDP_OK;
}

extern "C" ddp_status ddp_plan_destroy(ddp_plan* plan) {
    if (!plan) return DDP_E_ARG;
    ddp_rt_release(plan);
    delete plan;
    return DDP_OK;
}

extern "C" ddp_status ddp_plan_query(const ddp_plan* plan, ddp_plan_info* out) {
    if (!plan || !out) return DDP_E_ARG;
    *out = plan->info;
    return DDP_OK;
}

extern "C" ddp_status ddp_plan_get_delays(const ddp_plan* plan, int step, int32_t* host_out) {
    if (!plan || !host_out) return DDP_E_ARG;
    const std::vector<int32_t>* t = nullptr;
    if (step == 0 && !plan->subband) t = &plan->delay;
    if (step == 1 && plan->subband) t = &plan->d1;
    if (step == 2 && plan->subband) t = &plan->d2;
    if (!t) return ddp_fail(plan, DDP_E_ARG, "delay table step does not exist for this plan");
    std::memcpy(host_out, t->data(), t->size() * sizeof(int32_t));
    return DDP_OK;
}

// ------------------------------------------------------------------------------------ kernel geometry
bool ddp_kernel_in_plan(const ddp_plan* p, ddp_kernel k) {
    switch (k) {
        case DDP_K_DIRECT: return !p->subband;
        case DDP_K_SUB1:
        case DDP_K_SUB2: return p->subband;
        case DDP_K_INTEGRATE:
        case DDP_K_SNR: return p->integ_mode == DDP_INTEG_DECIMATE;
        case DDP_K_ISNR: return true;
        default: return false;
    }
}
ddp_kernel ddp_slot_kernel(const ddp_plan* p, int slot) {
    switch (slot) {
        case 0: return p->subband ? DDP_K_SUB1 : DDP_K_DIRECT;
        case 1: return p->subband ? DDP_K_SUB2 : DDP_K_COUNT;
        case 2: return DDP_K_INTEGRATE;
        case 3: return DDP_K_SNR;
        default: return DDP_K_COUNT;
    }
}
DdpKGeom ddp_kgeom(const ddp_plan* p, ddp_kernel k) {
    DdpKGeom g{p->ns, p->ndm, 0, 4};
    switch (k) {
        case DDP_K_DIRECT: g = {p->ns, p->ndm, p->nchan, p->in_bytes}; break;
        case DDP_K_SUB1: g = {(int)p->info.nsamp_sub, p->ncoarse, p->cps, p->in_bytes}; break;
        case DDP_K_SUB2: g = {p->ns, p->nfine, p->nsub, p->info.sub_elem_bytes}; break;
        default: break;
    }
    return g;
}

// Sliding boxcar kernel: chunks of prefix sums a warp keeps = 1 + ceil(largest width / chunk).
int ddp_slide_nb(const ddp_plan* p, const ddp_kcfg& c) {
    int maxw = 1;
    for (int i = 0; i < p->nwidths; ++i) maxw = std::max(maxw, p->widths[i]);
    const int ch = 32 * c.samples_per_thread;
    return 1 + (maxw + ch - 1) / ch;
}
// Largest (dmax - dmin) of any reduction row over any DM tile of TD trials: bounds the staged window.
int ddp_spread_max(const ddp_plan* p, ddp_kernel k, int TD) {
    const int which = k == DDP_K_DIRECT ? 0 : (k == DDP_K_SUB1 ? 1 : 2);
    auto it = p->spread_cache[which].find(TD);
    if (it != p->spread_cache[which].end()) return it->second;
    const std::vector<int32_t>& t = which == 0 ? p->delay : (which == 1 ? p->d1 : p->d2);
    const int ni = which == 0 ? p->ndm : (which == 1 ? p->ncoarse : p->nfine);
    const int nc = which == 2 ? p->nsub : p->nchan;
    int mx = 0;
    for (int lo = 0; lo < ni; lo += TD) {
        const int hi = std::min(lo + TD, ni) - 1;
        const int32_t* a = &t[(size_t)lo * nc];
        const int32_t* b = &t[(size_t)hi * nc];
        for (int c = 0; c < nc; ++c) mx = std::max(mx, b[c] - a[c]);
    }
    p->spread_cache[which][TD] = mx;
    return mx;
}
// Step 1 with "diagonal" time tiles (ddp_kernels.cuh, DIAG): per DM tile and subband the delays relative to the
// subband's first channel, rel[a][c] = d1[a][c] - d1[a][first], spread over the tile by far less than the delays
// themselves (a coarse trial moves the whole subband).  Usable when no relative delay is negative (the first channel
// of every subband is its earliest: the staged window never starts in front of the row) and worth it when it shrinks
// the window by more than half.
bool ddp_sub1_diag(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, int* rel_spread, int* shift_max) {
    if (k != DDP_K_SUB1 || c.staging == 0 || ddp_merge_group(c) || p->in_bytes != 1) return false;
    const int TD = c.threads_dm * c.dms_per_thread;
    auto it = p->diag_cache.find(TD);
    if (it == p->diag_cache.end()) {
        int spread = 0, shift = 0;
        bool ok = true;
        const int nc = p->nchan, cps = p->cps;
        for (int lo = 0; lo < p->ncoarse && ok; lo += TD) {
            const int hi = std::min(lo + TD, p->ncoarse);
            for (int s = 0; s < p->nsub && ok; ++s) {
                const int c0 = s * cps;
                const int D0 = p->d1[(size_t)lo * nc + c0];
                shift = std::max(shift, p->d1[(size_t)(hi - 1) * nc + c0] - D0);
                for (int r = 0; r < cps; ++r) {
                    int mn = INT32_MAX, mx = INT32_MIN;
                    for (int a = lo; a < hi; ++a) {
                        const int Da = p->d1[(size_t)a * nc + c0];  // the kernel shifts trial a by Da rounded down to D0 + a multiple of 4
                        const int rel = p->d1[(size_t)a * nc + c0 + r] - (Da - ((Da - D0) & 3));
                        mn = std::min(mn, rel);
                        mx = std::max(mx, rel);
                    }
                    if (mn < 0) { ok = false; break; }
                    spread = std::max(spread, mx - mn);
                }
            }
        }
        it = p->diag_cache.emplace(TD, ok ? std::make_pair(spread, shift) : std::make_pair(-1, -1)).first;
    }
    if (it->second.first < 0) return false;
    if (2 * it->second.first + 64 >= ddp_spread_max(p, k, TD)) return false;
    if (rel_spread) *rel_spread = it->second.first;
    if (shift_max) *shift_max = it->second.second;
    return true;
}
// Merged staging.  One scan of the delay table per (kernel, TD, G): for every DM tile of TD trials and every
// group of G adjacent reduction rows, the distinct tuples tau[m] = (d[j][r0+m] - d[j][r0]) - (same for the tile's
// first trial) over the tile's trials ("variants"), which variant every trial uses, and its window offset
// delta = d[j][r0] - d[first][r0].  Record layout in DdpMergeTable (ddp_internal.h).
static void merge_dims(const ddp_plan* p, ddp_kernel k, int* ni, int* nc) {
    *ni = k == DDP_K_DIRECT ? p->ndm : p->ncoarse;
    *nc = p->nchan;
}
// Variants of one (tile, group): tau[v][0..4), vid[j] for j < TD; returns the count, or -1 when the group cannot
// be served (a shift outside +-15 words, more than DDP_MERGE_VMAX_LIMIT variants, a delay that decreases with
// the trial index).  Trials past the end of a ragged tile repeat the last live one.
static int merge_scan_group(const int32_t* t, int nc, int lo, int nd, int TD, int r0, int G, int32_t* tau,
                            unsigned char* vid) {
    const int32_t* d0 = &t[(size_t)lo * nc + r0];
    int nv = 0;
    for (int j = 0; j < TD; ++j) {
        const int32_t* d = &t[(size_t)(lo + std::min(j, nd - 1)) * nc + r0];
        int32_t tj[4] = {0, 0, 0, 0};
        for (int m = 1; m < G; ++m) tj[m] = (d[m] - d[0]) - (d0[m] - d0[0]);
        int v = 0;
        for (; v < nv; ++v) {
            bool same = true;
            for (int m = 1; m < G; ++m) same = same && tau[v * 4 + m] == tj[m];
            if (same) break;
        }
        if (v == nv) {
            if (nv == DDP_MERGE_VMAX_LIMIT) return -1;
            for (int m = 1; m < G; ++m)
                if (tj[m] < -15 || tj[m] > 15) return -1;  // E rows carry 16 words in front
            for (int m = 0; m < 4; ++m) tau[nv * 4 + m] = tj[m];
            ++nv;
        }
        vid[j] = (unsigned char)v;
        if (d[0] - d0[0] < 0 || d[0] - d0[0] >= (1 << 24)) return -1;
        for (int m = 0; m < G; ++m)
            if (d[m] < d0[m]) return -1;  // window starts are the first trial's delays
    }
    return nv;
}
// Light part (variant counts): what the validity rules and the shared-memory size need.
const DdpMergeTable& ddp_merge_table(const ddp_plan* p, ddp_kernel k, int TD, int G) {
    const int which = k == DDP_K_DIRECT ? 0 : 1;
    auto key = std::make_pair(TD, G);
    auto it = p->merge_tables[which].find(key);
    if (it != p->merge_tables[which].end()) return it->second;
    DdpMergeTable& T = p->merge_tables[which][key];
    const std::vector<int32_t>& t = which == 0 ? p->delay : p->d1;
    int ni, nc;
    merge_dims(p, k, &ni, &nc);
    T.ntiles = (ni + TD - 1) / TD;
    T.ngg = nc / G;
    T.vmax = DDP_MERGE_VMAX_LIMIT + 1;
    const int nred = ddp_kgeom(p, k).nred;
    if (nred % G != 0 || nc % G != 0 || TD > 4096) return T;  // groups never straddle a subband
    std::vector<int32_t> nvar((size_t)T.ntiles * T.ngg);
    std::vector<int32_t> tau((size_t)4 * DDP_MERGE_VMAX_LIMIT);
    std::vector<unsigned char> vid(TD);
    int vmax = 0;
    for (int ti = 0; ti < T.ntiles; ++ti) {
        const int lo = ti * TD, nd = std::min(TD, ni - lo);
        for (int gg = 0; gg < T.ngg; ++gg) {
            const int nv = merge_scan_group(t.data(), nc, lo, nd, TD, gg * G, G, tau.data(), vid.data());
            if (nv < 0) return T;
            nvar[(size_t)ti * T.ngg + gg] = nv;
            vmax = std::max(vmax, nv);
        }
    }
    T.nvar.swap(nvar);
    T.vmax = vmax;
    T.vcap = (vmax + 3) & ~3;
    T.rw = (4 + 2 * G + T.vcap + TD + 3) & ~3;
    return T;
}
// The device image (record layout in ddp_internal.h), built when a launch needs it.
const std::vector<unsigned char>& ddp_merge_table_blob(const ddp_plan* p, ddp_kernel k, int TD, int G) {
    const DdpMergeTable& T = ddp_merge_table(p, k, TD, G);
    if (!T.blob.empty() || T.vmax > DDP_MERGE_VMAX_LIMIT) return T.blob;
    const std::vector<int32_t>& t = k == DDP_K_DIRECT ? p->delay : p->d1;
    int ni, nc;
    merge_dims(p, k, &ni, &nc);
    T.blob.assign((size_t)T.ntiles * T.ngg * T.rw * 4, 0);
    int32_t* rec = (int32_t*)T.blob.data();
    std::vector<int32_t> tau((size_t)4 * DDP_MERGE_VMAX_LIMIT);
    std::vector<unsigned char> vid(TD);
    for (int ti = 0; ti < T.ntiles; ++ti) {
        const int lo = ti * TD, nd = std::min(TD, ni - lo);
        for (int gg = 0; gg < T.ngg; ++gg, rec += T.rw) {
            const int r0 = gg * G;
            const int nv = merge_scan_group(t.data(), nc, lo, nd, TD, r0, G, tau.data(), vid.data());
            const int32_t* d0 = &t[(size_t)lo * nc + r0];
            const int32_t* dl = &t[(size_t)(lo + nd - 1) * nc + r0];
            rec[0] = nv;
            rec[1] = dl[0] - d0[0];  // span: largest window offset of the group
            for (int m = 0; m < G; ++m) {
                rec[4 + m] = d0[m];
                rec[4 + G + m] = dl[m];
            }
            for (int v = 0; v < nv; ++v) {
                uint32_t code = 0;
                for (int m = 1; m < G; ++m) code |= (uint32_t)(tau[(size_t)v * 4 + m] & 0xff) << (8 * (m - 1));
                rec[4 + 2 * G + v] = (int32_t)code;
            }
            for (int j = 0; j < TD; ++j) {
                const int32_t* d = &t[(size_t)(lo + std::min(j, nd - 1)) * nc + r0];
                rec[4 + 2 * G + T.vcap + j] = (int32_t)(((uint32_t)vid[j] << 24) | (uint32_t)(d[0] - d0[0]));
            }
        }
    }
    return T.blob;
}
int ddp_merge_vmax(const ddp_plan* p, ddp_kernel k, int TD, int G) { return ddp_merge_table(p, k, TD, G).vmax; }
int64_t ddp_merge_table_bytes(const ddp_plan* p, ddp_kernel k, int TD, int G) {
    const DdpMergeTable& T = ddp_merge_table(p, k, TD, G);
    return (int64_t)T.ntiles * T.ngg * T.rw * 4;
}
// Variant rows a chunk of U reduction rows needs at most: chunks start at multiples of U inside a kernel group.
int ddp_merge_rows_max(const ddp_plan* p, ddp_kernel k, int TD, int G, int U) {
    const DdpMergeTable& T = ddp_merge_table(p, k, TD, G);
    if (T.vmax > DDP_MERGE_VMAX_LIMIT) return 0;
    auto it = T.rows_max.find(U);
    if (it != T.rows_max.end()) return it->second;
    const int NG = U / G;
    int best = 0;
    for (int ti = 0; ti < T.ntiles; ++ti)
        for (int gg = 0; gg + NG <= T.ngg; gg += NG) {
            int sum = 0;
            for (int q = 0; q < NG; ++q) sum += T.nvar[(size_t)ti * T.ngg + gg + q];
            best = std::max(best, sum);
        }
    T.rows_max[U] = best;
    return best;
}
DdpMergeGeom ddp_merge_geom(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    const int G = ddp_merge_group(c);
    const int64_t TT = (int64_t)c.threads_t * c.samples_per_thread;
    const int TD = c.threads_dm * c.dms_per_thread;
    const int spread = ddp_spread_max(p, k, TD);
    const DdpMergeTable& T = ddp_merge_table(p, k, TD, G);
    DdpMergeGeom g;
    g.vmax = T.vmax;
    g.vcap = T.vcap;
    g.rw = T.rw;
    g.rows_max = T.vmax > DDP_MERGE_VMAX_LIMIT ? 0 : ddp_merge_rows_max(p, k, TD, G, c.unroll);
    g.lw = (int)round_up(TT / 2 + spread + 4, 4);        // variant row: y <= TT/2 + spread
    g.le = (int)round_up(16 + TT / 2 + spread + 48, 4);  // expanded row: 16 words in front, 16-byte carry, shifts within +-15
    return g;
}

int ddp_dedisp_win(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    const DdpKGeom g = ddp_kgeom(p, k);
    const int AL = 16 / g.in_bytes;
    const int64_t TT = (int64_t)c.threads_t * c.samples_per_thread;
    const int64_t TD = (int64_t)c.threads_dm * c.dms_per_thread;
    if (g.in_bytes == 1) {  // packed kernel: 16-byte carry + shifted-copy tail, in bytes, multiple of 16
        int rel = 0;
        if (ddp_sub1_diag(p, k, c, &rel)) return (int)round_up(TT + rel + 32, 16);
        return (int)round_up(TT + ddp_spread_max(p, k, (int)TD) + 32, 16);
    }
    if (g.in_bytes == 2 && c.staging != 0)  // packed uint16 kernel: 8-element carry + 4 spare words, multiple of 8
        return (int)round_up(TT + ddp_spread_max(p, k, (int)TD) + 16, 8);
    return (int)round_up(TT + ddp_spread_max(p, k, (int)TD) + 2 * AL, AL);
}
// ddp_dedisp_packed_body with nb buffers of shifted copies: copies [nb][U][4 or 3][win], offs [2][TD][U],
// dls [2][TD][64], TMA: raw [2][U][win + 16] + mbarriers, DIAG: dmm [2][2][64] + dsh [TD]
static size_t packed_u8_layout(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, size_t nb) {
    const size_t row = (size_t)ddp_dedisp_win(p, k, c);
    const size_t TD = (size_t)c.threads_dm * c.dms_per_thread;
    const size_t ncp = nb == 1 && c.staging == 2 ? 3 : 4;  // single-buffered with TMA: the unshifted copy is the raw slot (RAW0)
    size_t b = nb * ncp * row * c.unroll + ((2 * TD * c.unroll + 3) & ~(size_t)3) * 4 + 2 * TD * 64 * 4;
    if (c.staging == 2) b += 2 * (size_t)c.unroll * (row + 16) + 16;
    if (ddp_sub1_diag(p, k, c)) b += (4 * 64 + TD) * 4;
    return b;
}
size_t ddp_smem_bytes(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    const int64_t TT = (int64_t)c.threads_t * c.samples_per_thread;
    switch (k) {
        case DDP_K_DIRECT:
        case DDP_K_SUB1:
        case DDP_K_SUB2: {
            if (c.staging == 0) return 0;
            const DdpKGeom g = ddp_kgeom(p, k);
            const size_t row = (size_t)ddp_dedisp_win(p, k, c) * g.in_bytes;
            if (g.in_bytes == 1 && ddp_merge_group(c)) {  // ddp_dedisp_merge_body (same carve-up, same order)
                const size_t G = (size_t)ddp_merge_group(c), U = (size_t)c.unroll, NG = U / G;
                const size_t TD = (size_t)c.threads_dm * c.dms_per_thread;
                const DdpMergeGeom mg = ddp_merge_geom(p, k, c);
                if (mg.vmax > DDP_MERGE_VMAX_LIMIT) return (size_t)DDP_SMEM_LIMIT + 1;
                size_t b = 2 * (size_t)mg.rows_max * mg.lw * 4;       // pw
                b += 2 * U * (size_t)mg.le * 4;                       // ebuf
                b += 2 * U * (row + 16);                              // raw
                b += 2 * NG * (size_t)mg.rw * 4;                      // record staging
                b += 16 * (((16 + 4 * U + 8 * (size_t)mg.rows_max + TD * NG) + 3) & ~(size_t)3) * 4;  // descriptor ring
                b += (4 + 2 * 16 + 2) * 8 + 128;                      // mbarriers, scheduler state
                return b;
            }
            if (g.in_bytes == 1) {  // ddp_dedisp_packed_body
                // two buffers of shifted copies when they fit, else one (ddp_u8_single_buffered)
                const size_t two = packed_u8_layout(p, k, c, 2);
                return two <= DDP_SMEM_LIMIT ? two : packed_u8_layout(p, k, c, 1);
            }
            if (g.in_bytes == 2) {  // ddp_dedisp_packed16_body: copies [NB][U][2][win/2] words, offs [TD][nred4], mbar [NB]
                const size_t TD = (size_t)c.threads_dm * c.dms_per_thread;
                const size_t nb = c.staging == 2 ? 3 : 2;
                return nb * c.unroll * 2 * row + TD * (size_t)((g.nred + 3) & ~3) * 4 + nb * 8;
            }
            return c.staging == 1 ? row * c.unroll : 2 * row * c.unroll + 16;
        }
        case DDP_K_INTEGRATE: {
            size_t b = (size_t)c.threads_dm * 32 * 4;  // warp totals [threads_dm][32]
            if (c.staging != 0) b += (size_t)c.threads_dm * TT * 4 + 16;
            return b;
        }
        case DDP_K_ISNR: {
            if (p->integ_mode == DDP_INTEG_SLIDING) {  // prefix-sum ring per warp: (1 + ceil(wmax / chunk)) chunks, skewed
                const int64_t ring = (int64_t)ddp_slide_nb(p, c) * 32 * c.samples_per_thread;
                return (size_t)c.threads_dm * (size_t)(ring + (ring >> 5)) * 4;
            }
            return (size_t)c.threads_dm * 8 * 8 * 4;  // wide-level accumulators [threads_dm][8][8]
        }
        case DDP_K_SNR: {
            size_t b = (size_t)c.threads_dm * 32 * 24;
            if (c.staging != 0) b += (size_t)c.threads_dm * (c.staging == 2 ? 2 : 1) * TT * 4 + (size_t)c.threads_dm * 16;
            return b;
        }
        default: return 0;
    }
}

// The packed uint8 kernel keeps two buffers of shifted copies (chunk c+1 converted while chunk c is
// summed); a configuration whose two buffers exceed 227 KB runs with one, if that fits.
bool ddp_u8_single_buffered(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c) {
    if (c.staging == 0 || ddp_merge_group(c) || ddp_kgeom(p, k).in_bytes != 1) return false;
    return packed_u8_layout(p, k, c, 2) > DDP_SMEM_LIMIT;
}

// Validity rules (from Table 3 P:136-152 + sm_100a limits).
bool ddp_kcfg_valid(const ddp_plan* p, ddp_kernel k, const ddp_kcfg& c, std::string* why) {
    auto no = [&](const char* m) {
        if (why) *why = m;
        return false;
    };
    if (!ddp_kernel_in_plan(p, k)) return no("kernel not part of this plan");
    for (int g = 0; g < DDP_NGENES; ++g)
        if (ddp_gene_index(g, ddp_gene_get(c, g)) < 0) return no("gene value outside its candidate array");
    const DdpKGeom geo = ddp_kgeom(p, k);
    const int64_t threads = (int64_t)c.threads_t * c.threads_dm;
    const int64_t TT = (int64_t)c.threads_t * c.samples_per_thread;
    const int64_t TD = (int64_t)c.threads_dm * c.dms_per_thread;
    if (k == DDP_K_ISNR) {  // fused integration + S/N: one warp per series, everything else pinned (V7)
        if (c.threads_t != 32) return no("V1: the fused kernel gives one warp to a series: threads_t must be 32");
        if (c.samples_per_thread < 4) return no("V5: the fused kernel loads 16-byte vectors: samples_per_thread >= 4");
        if (c.unroll != 1 || c.staging != 0 || c.vec_bytes != 16) return no("V7: the fused kernel pins unroll = 1, staging = 0, vec_bytes = 16");
        if ((int64_t)c.threads_dm * c.dms_per_thread > pow2ceil(p->ndm)) return no("V3: DM tile larger than the problem");
        int maxw = 1;
        for (int i = 0; i < p->nwidths; ++i) maxw = std::max(maxw, p->widths[i]);
        if (maxw > 32 * c.samples_per_thread * 256) return no("V3: a width is longer than 256 chunks of the fused kernel");
        if (ddp_smem_bytes(p, k, c) > DDP_SMEM_LIMIT) return no("V6: shared memory over 227 KB");
        return true;
    }
    // V7: a gene the kernel does not read is pinned (snr reads `unroll` only with direct loads)
    if (k == DDP_K_SNR && c.staging != 0 && c.unroll != 1) return no("V7: snr ignores unroll when staged; must be 1");
    // merged staging (genes 3, 4) exists for the uint8 dedispersion kernels only; its groups are whole
    // multiples of the chunk, its window words hold two samples, the vector-width gene is unused (V7)
    const int MG = ddp_merge_group(c);
    if (MG) {
        if (geo.in_bytes != 1 || geo.nred == 0) return no("V6: merged staging is for uint8 dedispersion only");
        if (c.unroll % MG != 0) return no("V4: unroll is not a multiple of the merge group");
        if (c.vec_bytes != 16) return no("V7: merged staging ignores vec_bytes; must be 16");
        if (c.samples_per_thread < 2) return no("V5: merged staging needs samples_per_thread >= 2");
        if (c.threads_t < 32) return no("V1: merged staging needs threads_t >= 32");
        if (threads > 512) return no("V1: merged staging adds its producer warps to the block: at most 512 consumer threads");
        if ((c.threads_dm * c.dms_per_thread) % 4 != 0) return no("V3: merged staging needs a DM tile of a multiple of 4 trials");
    }
    // V5: vector width vs. what a thread loads contiguously
    if (MG) {
    } else if (geo.in_bytes == 1) {
        if (c.vec_bytes > 1 && c.vec_bytes > c.samples_per_thread) return no("V5: vec_bytes > samples_per_thread bytes");
        if (c.staging != 0) {  // the packed kernel works on whole 4-sample words, one warp per 32 of them
            if (c.samples_per_thread < 4) return no("V5: staged uint8 input needs samples_per_thread >= 4");
            if (c.vec_bytes < 4) return no("V5: staged uint8 input needs vec_bytes >= 4");
            if (c.threads_t < 32) return no("V1: staged uint8 input needs threads_t >= 32");
        }
    } else if (geo.in_bytes == 2) {
        if (c.vec_bytes < 4) return no("V5: uint16 input needs vec_bytes >= 4");
        if (c.vec_bytes > 2 * c.samples_per_thread) return no("V5: vec_bytes > samples_per_thread*2");
        if (c.staging != 0 && c.threads_t < 32)  // the packed kernel gives each warp 32 consecutive 2-sample words
            return no("V1: staged uint16 input needs threads_t >= 32");
    } else {
        if (c.vec_bytes < 4) return no("V5: uint32 input needs vec_bytes >= 4");
        if (c.vec_bytes > 4 * c.samples_per_thread) return no("V5: vec_bytes > samples_per_thread*4");
    }
    // V4: unroll divides the reduction trip count
    if (geo.nred > 0 && geo.nred % c.unroll != 0) return no("V4: unroll does not divide the reduction length");
    // V1: block size
    if (threads < 32 || threads > 1024) return no("V1: threads per block outside 32..1024");
    // V2: register budget
    if (c.samples_per_thread * c.dms_per_thread > 128) return no("V2: samples_per_thread*dms_per_thread > 128");
    // V3: tile not larger than the (power-of-two rounded) problem
    if (TT > pow2ceil(geo.ns_k)) return no("V3: time tile larger than the problem");
    if (TD > pow2ceil(geo.ndm_k)) return no("V3: DM tile larger than the problem");
    if (k == DDP_K_INTEGRATE) {
        for (int i = 0; i < p->nwidths; ++i)
            if (p->widths[i] > 1 && TT % p->widths[i] != 0) return no("V3: a width does not divide the time tile");
    }
    // V6: staged window fits shared memory; merged staging: the variant rows of a group fit the kernel's table
    if (MG) {
        const int vm = ddp_merge_vmax(p, k, (int)TD, MG);
        if (vm > DDP_MERGE_VMAX_LIMIT) return no("V6: too many relative-shift variants per group for merged staging");
        if (ddp_merge_table_bytes(p, k, (int)TD, MG) > p->merge_capacity)
            return no("V6: merged-staging table larger than its workspace region");
    }
    if (ddp_smem_bytes(p, k, c) > DDP_SMEM_LIMIT) return no("V6: shared memory over 227 KB");
    return true;
}

const std::vector<ddp_kcfg>& ddp_valid_set(const ddp_plan* p, ddp_kernel k) {
    if (!p->valid_built[k]) {
        std::vector<ddp_kcfg>& v = p->valid[k];
        v.clear();
        const DdpGeneDomain* D = kDomains;
        ddp_kcfg c;
        for (int a = 0; a < D[0].n; ++a)
            for (int b = 0; b < D[1].n; ++b)
                for (int s = 0; s < D[2].n; ++s)
                    for (int d = 0; d < D[3].n; ++d)
                        for (int u = 0; u < D[4].n; ++u)
                            for (int g = 0; g < D[5].n; ++g)
                                for (int w = 0; w < D[6].n; ++w) {
                                    c = {D[0].v[a], D[1].v[b], D[2].v[s], D[3].v[d], D[4].v[u], D[5].v[g], D[6].v[w]};
                                    if (ddp_kcfg_valid(p, k, c, nullptr)) v.push_back(c);
                                }
        p->valid_built[k] = true;
    }
    return p->valid[k];
}

extern "C" ddp_status ddp_check_kcfg(const ddp_plan* plan, ddp_kernel k, const ddp_kcfg* cfg) {
    if (!plan || !cfg || k < 0 || k >= DDP_K_COUNT) return DDP_E_ARG;
    std::string why;
    if (!ddp_kcfg_valid(plan, k, *cfg, &why)) return ddp_fail(plan, DDP_E_CONFIG, why);
    return DDP_OK;
}

// Nearest valid configuration (BJ:cfg4): minimise sum over genes of |index distance| in the
// candidate arrays (= |delta log2| for the power-of-two genes); ties -> first in canonical order.
// A gene value outside its array is first snapped to the nearest candidate (ties -> smaller).
extern "C" ddp_status ddp_repair_kcfg(const ddp_plan* plan, ddp_kernel k, ddp_kcfg* inout) {
    if (!plan || !inout || k < 0 || k >= DDP_K_COUNT) return DDP_E_ARG;
    if (!ddp_kernel_in_plan(plan, k)) return ddp_fail(plan, DDP_E_CONFIG, "kernel not part of this plan");
    int idx[DDP_NGENES];
    for (int g = 0; g < DDP_NGENES; ++g) {
        const int v = ddp_gene_get(*inout, g);
        int best = 0;
        long bestd = -1;
        for (int i = 0; i < kDomains[g].n; ++i) {
            const long d = std::labs((long)kDomains[g].v[i] - v);
            if (bestd < 0 || d < bestd) { bestd = d; best = i; }
        }
        idx[g] = best;
        *ddp_gene_ptr(inout, g) = kDomains[g].v[best];
    }
    if (ddp_kcfg_valid(plan, k, *inout, nullptr)) return DDP_OK;
    const std::vector<ddp_kcfg>& V = ddp_valid_set(plan, k);
    if (V.empty()) return ddp_fail(plan, DDP_E_CONFIG, "no valid configuration exists for this kernel");
    int bestdist = 1 << 30;
    const ddp_kcfg* best = nullptr;
    for (const ddp_kcfg& c : V) {
        int d = 0;
        for (int g = 0; g < DDP_NGENES; ++g) d += std::abs(ddp_gene_index(g, ddp_gene_get(c, g)) - idx[g]);
        if (d < bestdist) { bestdist = d; best = &c; }
    }
    *inout = *best;
    return DDP_OK;
}

extern "C" ddp_status ddp_enumerate_kcfgs(const ddp_plan* plan, ddp_kernel k, ddp_kcfg* out, size_t cap, size_t* n) {
    if (!plan || !n || k < 0 || k >= DDP_K_COUNT) return DDP_E_ARG;
    if (!ddp_kernel_in_plan(plan, k)) { *n = 0; return DDP_OK; }
    const std::vector<ddp_kcfg>& V = ddp_valid_set(plan, k);
    *n = V.size();
    if (out)
        for (size_t i = 0; i < V.size() && i < cap; ++i) out[i] = V[i];
    return DDP_OK;
}

extern "C" ddp_status ddp_get_kcfg(const ddp_plan* plan, ddp_kernel k, ddp_kcfg* out) {
    if (!plan || !out || k < 0 || k >= DDP_K_COUNT) return DDP_E_ARG;
    if (!ddp_kernel_in_plan(plan, k)) return ddp_fail(plan, DDP_E_CONFIG, "kernel not part of this plan");
    *out = plan->kcfg[k];
    return DDP_OK;
}

extern "C" ddp_status ddp_set_kcfg(ddp_plan* plan, ddp_kernel k, const ddp_kcfg* cfg) {
    if (!plan || !cfg || k < 0 || k >= DDP_K_COUNT) return DDP_E_ARG;
    std::string why;
    if (!ddp_kcfg_valid(plan, k, *cfg, &why)) return ddp_fail(plan, DDP_E_CONFIG, why);
    ddp_status s = ddp_rt_activate(plan, k, *cfg);  // DDP_OK without a device: compiled lazily at first launch
    if (s != DDP_OK) return s;
    plan->kcfg[k] = *cfg;
    return DDP_OK;
}

// Default configurations: preferred shapes repaired into the plan's valid space.
static void default_kcfgs(ddp_plan* p) {
    const ddp_kcfg pref[DDP_K_COUNT] = {
        /* direct    */ {64, 4, 16, 4, 8, 1, 16},
        /* sub1      */ {64, 4, 16, 2, 8, 1, 16},
        /* sub2      */ {128, 2, 4, 8, 8, 2, 16},
        /* integrate */ {256, 1, 4, 1, 1, 0, 16},
        /* snr       */ {256, 1, 4, 1, 4, 0, 16},
        /* isnr      */ {32, 8, 16, 1, 1, 0, 16},
    };
    for (int k = 0; k < DDP_K_COUNT; ++k) {
        p->kcfg[k] = pref[k];
        if (ddp_kernel_in_plan(p, (ddp_kernel)k)) ddp_repair_kcfg(p, (ddp_kernel)k, &p->kcfg[k]);
    }
}

extern "C" const char* ddp_status_str(ddp_status s) {
    switch (s) {
        case DDP_OK: return "ok";
        case DDP_E_ARG: return "bad argument";
        case DDP_E_SHAPE: return "bad shape/stride/alignment";
        case DDP_E_OVERFLOW: return "accumulation could overflow";
        case DDP_E_WORKSPACE: return "workspace missing or too small";
        case DDP_E_CONFIG: return "invalid kernel configuration";
        case DDP_E_COMPILE: return "kernel compilation failed";
        case DDP_E_CUDA: return "CUDA error or no device";
        case DDP_E_BUDGET: return "evaluation budget exhausted";
        default: return "unknown status";
    }
}
extern "C" const char* ddp_last_error(const ddp_plan* plan) { return plan ? plan->err.c_str() : ""; }
extern "C" const char* ddp_version(void) { return "ddp 0.1 (sm_100a)"; }
