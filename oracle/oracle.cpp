// ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded CPU statement of what the
// single-pulse-search hot path computes.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, link or call this file.  It shares no code,
// header, table or constant generator with paper_1811_04165_b200/ (the CUDA product path).
//
// Citations: P:n = /root/reference/PAPER.md line n; BJ = /root/repo/BASELINE.json;
// DD.x / SB.x / INT.x / SNR.x = readings listed in DESIGN.md.
//
// What is defined where:
//   * the pipeline = two-step de-dispersion, downsampling ("smoothing"), S/N
//   * de-dispersion = "appropriate shift and integration of frequency channels"
//   * subband structure (SUBBANDS, SUBBANDING_DMS x DMS, fine grid starts at 0.0) P:71 fn.4
//   * downsampled length NRSAMPLES = SAMPLES / DOWNSAMPLING
//   * 8-bit input
//   * delay formula 4.148808e3*DM*(f^-2 - f_ref^-2)/t_samp rounded to nearest,
//     uint32 accumulation, SNR = (max - mean)/std in float32                      BJ north_star, BJ cfg0
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): DM=0 row == plain channel sum; hand-derived
// 4-channel worked example (tests/golden/worked_example.txt); single-impulse response (sign and
// every delay); constant input; linearity; brute force in pure Python on tiny inputs; subband
// rows with zero fine offset == direct rows; nSub=1 identity; integration invariants
// I_2w[j]=I_w[2j]+I_w[2j+1]; S/N affine + permutation invariance and numpy float64 closed form;
// injected pulse recovered at its DM and width on BJ cfg0; sliding boxcar: constant / impulse closed forms,
// numpy cumulative-sum difference, block sums are its samples at multiples of w, a misaligned pulse is
// recovered at its true width; channel mask: pure-Python brute force over the kept channels, complement
// identity; consecutive batches with carried samples == one long dedispersion; 16-bit input (the _u16
// functions): worked example scaled by 257, linearity over the two bytes against the pinned uint8 functions,
// numpy brute force, saturated input.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC oracle.cpp -o liboracle.so
#include <cmath>
#include <cstddef>
#include <cstdint>

extern "C" {

// DD (BJ north_star).  delay[i][c] = floor(x + 0.5),
//   x = ((K * DM[i]) * (1/f[c]^2 - 1/f_ref^2)) / t_samp      in IEEE float64, this association (DD.2).
// f in MHz, t_samp in s, DM in pc cm^-3, K = 4.148808e3 (DD.1).  f_ref is passed explicitly: the
// highest channel frequency for direct and step-1 tables (DD.3), and also for the step-2 table,
// whose "channels" are the subband reference frequencies (SB.1, SB.2).
// Returns 0, or -1 on a non-finite / negative-overflowing entry.
int oracle_delay_table(const double* f_mhz, int nchan, double f_ref_mhz,
                       const double* dm, int ndm, double t_samp_s, int32_t* delay) {
    const double K = 4.148808e3;
    const double inv_ref = 1.0 / (f_ref_mhz * f_ref_mhz);
    for (int i = 0; i < ndm; ++i) {
        for (int c = 0; c < nchan; ++c) {
            const double g = 1.0 / (f_mhz[c] * f_mhz[c]) - inv_ref;
            const double x = ((K * dm[i]) * g) / t_samp_s;
            const double r = std::floor(x + 0.5);
            if (!(r >= -2147483648.0 && r <= 2147483647.0)) return -1;
            delay[(size_t)i * nchan + c] = (int32_t)r;
        }
    }
    return 0;
}

// DD: Y[i][t] = sum_c X[c][t + delay[i][c]],  0 <= t < ns.  uint8 in, uint32 sums, no scaling (DD.6);
// the caller supplies ns + max delay samples per channel (DD.5).  `delay` holds the nrows rows
// to compute (any subset of the DM grid), so sampled rows of a large search cost only those rows.
int oracle_dedisperse(const uint8_t* X, int nchan, size_t in_stride,
                      const int32_t* delay, int nrows, int ns,
                      uint32_t* Y, size_t out_stride) {
    for (int i = 0; i < nrows; ++i) {
        uint32_t* y = Y + (size_t)i * out_stride;
        for (int t = 0; t < ns; ++t) y[t] = 0u;
        for (int c = 0; c < nchan; ++c) {
            const int32_t d = delay[(size_t)i * nchan + c];
            if (d < 0 || (size_t)d + (size_t)ns > in_stride) return -2;
            const uint8_t* x = X + (size_t)c * in_stride + d;
            for (int t = 0; t < ns; ++t) y[t] += (uint32_t)x[t];
        }
    }
    return 0;
}

// SB step one (P:63, P:71 fn.4; reading SB.1 "B"):
//   S[a][s][t] = sum_{c in subband s} X[c][t + d1[a][c]],  0 <= t < ns1 (= ns + max d2),
// subband s = channels s*cps .. s*cps+cps-1 in array order (SB.3).  `d1` holds ncoarse rows.
int oracle_subband_step1(const uint8_t* X, int nchan, size_t in_stride, int nsub,
                         const int32_t* d1, int ncoarse, int ns1,
                         uint32_t* S, size_t s_stride) {
    if (nsub <= 0 || nchan % nsub != 0) return -1;
    const int cps = nchan / nsub;
    for (int a = 0; a < ncoarse; ++a) {
        for (int s = 0; s < nsub; ++s) {
            uint32_t* out = S + ((size_t)a * nsub + s) * s_stride;
            for (int t = 0; t < ns1; ++t) out[t] = 0u;
            for (int k = 0; k < cps; ++k) {
                const int c = s * cps + k;
                const int32_t d = d1[(size_t)a * nchan + c];
                if (d < 0 || (size_t)d + (size_t)ns1 > in_stride) return -2;
                const uint8_t* x = X + (size_t)c * in_stride + d;
                for (int t = 0; t < ns1; ++t) out[t] += (uint32_t)x[t];
            }
        }
    }
    return 0;
}

// SB step two (reading SB.1 "B"):
//   Y[a*nfine + b][t] = sum_s S[a][s][t + d2[b][s]],  0 <= t < ns;  trial DM = A[a] + F[b].
int oracle_subband_step2(const uint32_t* S, int nsub, size_t s_stride, int ns1,
                         const int32_t* d2, int nfine, int ncoarse, int ns,
                         uint32_t* Y, size_t out_stride) {
    for (int a = 0; a < ncoarse; ++a) {
        for (int b = 0; b < nfine; ++b) {
            uint32_t* y = Y + ((size_t)a * nfine + b) * out_stride;
            for (int t = 0; t < ns; ++t) y[t] = 0u;
            for (int s = 0; s < nsub; ++s) {
                const int32_t d = d2[(size_t)b * nsub + s];
                if (d < 0 || d + ns > ns1) return -2;
                const uint32_t* in = S + ((size_t)a * nsub + s) * s_stride + d;
                for (int t = 0; t < ns; ++t) y[t] += in[t];
            }
        }
    }
    return 0;
}

// INT ("downsampling (smoothing)"; readings INT.1 decimating, INT.2 drop the tail):
//   n_w = floor(ns / w);  I_w[i][j] = sum_{k<w} Y[i][j*w + k],  0 <= j < n_w.
int oracle_integrate(const uint32_t* Y, size_t stride, int nrows, int ns, int w,
                     uint32_t* I, size_t i_stride) {
    if (w <= 0) return -1;
    const int nw = ns / w;
    for (int i = 0; i < nrows; ++i) {
        const uint32_t* y = Y + (size_t)i * stride;
        uint32_t* o = I + (size_t)i * i_stride;
        for (int j = 0; j < nw; ++j) {
            uint32_t acc = 0u;
            for (int k = 0; k < w; ++k) acc += y[(size_t)j * w + k];
            o[j] = acc;
        }
    }
    return 0;
}

// INT, sliding reading (SURVEY 8(c) INT.1 alternative, 8(f) f1; BJ "boxcar integration over a set of pulse
// widths"; reading INT.1s): the stride-1 boxcar
//   n = ns - w + 1;  I^s_w[i][t] = sum_{k<w} Y[i][t + k],  0 <= t < n.
// Every output is a full-width sum (no partial windows at the edges); w = 1 is Y itself.
int oracle_integrate_sliding(const uint32_t* Y, size_t stride, int nrows, int ns, int w,
                             uint32_t* I, size_t i_stride) {
    if (w <= 0 || w > ns) return -1;
    const int n = ns - w + 1;
    for (int i = 0; i < nrows; ++i) {
        const uint32_t* y = Y + (size_t)i * stride;
        uint32_t* o = I + (size_t)i * i_stride;
        for (int t = 0; t < n; ++t) {
            uint32_t acc = 0u;
            for (int k = 0; k < w; ++k) acc += y[(size_t)t + k];
            o[t] = acc;
        }
    }
    return 0;
}

// DD with a channel mask ("zapped channels"; reading DD.7m): channels whose mask byte is 0
// are left out of the sum, every other channel contributes exactly as in oracle_dedisperse.
int oracle_dedisperse_masked(const uint8_t* X, int nchan, size_t in_stride, const uint8_t* mask,
                             const int32_t* delay, int nrows, int ns, uint32_t* Y, size_t out_stride) {
    for (int i = 0; i < nrows; ++i) {
        uint32_t* y = Y + (size_t)i * out_stride;
        for (int t = 0; t < ns; ++t) y[t] = 0u;
        for (int c = 0; c < nchan; ++c) {
            if (mask[c] == 0) continue;
            const int32_t d = delay[(size_t)i * nchan + c];
            if (d < 0 || (size_t)d + (size_t)ns > in_stride) return -2;
            const uint8_t* x = X + (size_t)c * in_stride + d;
            for (int t = 0; t < ns; ++t) y[t] += (uint32_t)x[t];
        }
    }
    return 0;
}

// INPUT_BITS = 16 (P:90 lists the sample width as a parameter of the setup): the same two sums over
// unsigned 16-bit samples.  Nothing else changes: uint32 totals, same delays, same ranges.
int oracle_dedisperse_u16(const uint16_t* X, int nchan, size_t in_stride, const int32_t* delay, int nrows, int ns,
                          uint32_t* Y, size_t out_stride) {
    for (int i = 0; i < nrows; ++i) {
        uint32_t* y = Y + (size_t)i * out_stride;
        for (int t = 0; t < ns; ++t) y[t] = 0u;
        for (int c = 0; c < nchan; ++c) {
            const int32_t d = delay[(size_t)i * nchan + c];
            if (d < 0 || (size_t)d + (size_t)ns > in_stride) return -2;
            const uint16_t* x = X + (size_t)c * in_stride + d;
            for (int t = 0; t < ns; ++t) y[t] += (uint32_t)x[t];
        }
    }
    return 0;
}
int oracle_subband_step1_u16(const uint16_t* X, int nchan, size_t in_stride, int nsub, const int32_t* d1, int ncoarse,
                             int ns1, uint32_t* S, size_t s_stride) {
    if (nsub <= 0 || nchan % nsub != 0) return -1;
    const int cps = nchan / nsub;
    for (int a = 0; a < ncoarse; ++a) {
        for (int s = 0; s < nsub; ++s) {
            uint32_t* out = S + ((size_t)a * nsub + s) * s_stride;
            for (int t = 0; t < ns1; ++t) out[t] = 0u;
            for (int k = 0; k < cps; ++k) {
                const int c = s * cps + k;
                const int32_t d = d1[(size_t)a * nchan + c];
                if (d < 0 || (size_t)d + (size_t)ns1 > in_stride) return -2;
                const uint16_t* x = X + (size_t)c * in_stride + d;
                for (int t = 0; t < ns1; ++t) out[t] += (uint32_t)x[t];
            }
        }
    }
    return 0;
}

// SNR ("signal-to-noise (S/N) computation"; definition BJ cfg0; readings SNR.1-SNR.4):
//   over the n values v_j of one (DM, width) series:
//   mean = (sum v_j)/n;  var = sum (v_j - mean)^2 / (n - ddof);  snr = (max - mean)/sqrt(var)
//   argmax = smallest j attaining the maximum;  var == 0 -> snr = 0, argmax = 0.
// Exact integer sum, two-pass float64 variance, one rounding to float32.
int oracle_snr(const uint32_t* V, size_t stride, int nrows, int n, int ddof,
               float* snr, uint32_t* argmax) {
    if (n - ddof <= 0) return -1;
    for (int i = 0; i < nrows; ++i) {
        const uint32_t* v = V + (size_t)i * stride;
        uint64_t sum = 0;
        uint32_t vmax = v[0];
        uint32_t imax = 0;
        for (int j = 0; j < n; ++j) {
            sum += v[j];
            if (v[j] > vmax) { vmax = v[j]; imax = (uint32_t)j; }
        }
        const double mean = (double)sum / (double)n;
        double ss = 0.0;
        for (int j = 0; j < n; ++j) {
            const double d = (double)v[j] - mean;
            ss += d * d;
        }
        const double var = ss / (double)(n - ddof);
        if (var > 0.0) {
            snr[i] = (float)(((double)vmax - mean) / std::sqrt(var));
            argmax[i] = imax;
        } else {
            snr[i] = 0.0f;
            argmax[i] = 0u;
        }
    }
    return 0;
}

}  // extern "C"
