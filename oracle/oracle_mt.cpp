// ORACLE, multi-core leg -- TEST INFRASTRUCTURE ONLY (same rules as oracle.cpp: only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build or call it).
//
// SURVEY.md 8(d) / BASELINE.md section 3: "the same loops with the DM axis split over all host cores
// (OpenMP `parallel for` on independent DM rows -- no other change)".  Every function here is an
// `omp parallel for` over independent rows whose body calls the single-thread oracle function of
// oracle.cpp on ONE row (direct: one DM trial; subband: one coarse DM with all its fine DMs), so the
// arithmetic is oracle.cpp's, untouched.  It exists so that the parity tests can afford EVERY row of
// the full-size configs and so that bench.py can quote a second, all-cores CPU figure.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fopenmp -shared -fPIC oracle.cpp oracle_mt.cpp -o liboracle_mt.so
#include <omp.h>

#include <cstddef>
#include <cstdint>

extern "C" {
int oracle_dedisperse(const uint8_t* X, int nchan, size_t in_stride, const int32_t* delay, int nrows, int ns,
                      uint32_t* Y, size_t out_stride);
int oracle_subband_step1(const uint8_t* X, int nchan, size_t in_stride, int nsub, const int32_t* d1, int ncoarse,
                         int ns1, uint32_t* S, size_t s_stride);
int oracle_subband_step2(const uint32_t* S, int nsub, size_t s_stride, int ns1, const int32_t* d2, int nfine,
                         int ncoarse, int ns, uint32_t* Y, size_t out_stride);
int oracle_integrate(const uint32_t* Y, size_t stride, int nrows, int ns, int w, uint32_t* I, size_t i_stride);
int oracle_snr(const uint32_t* V, size_t stride, int nrows, int n, int ddof, float* snr, uint32_t* argmax);

int oracle_mt_threads(void) { return omp_get_max_threads(); }

// DD: rows are DM trials.
int oracle_mt_dedisperse(const uint8_t* X, int nchan, size_t in_stride, const int32_t* delay, int nrows, int ns,
                         uint32_t* Y, size_t out_stride) {
    int rc = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < nrows; ++i) {
        const int r = oracle_dedisperse(X, nchan, in_stride, delay + (size_t)i * nchan, 1, ns, Y + (size_t)i * out_stride,
                                        out_stride);
        if (r != 0) {
#pragma omp critical
            rc = r;
        }
    }
    return rc;
}

// SB: rows are coarse DMs; step 1 then step 2 of one coarse DM (all its subbands / fine DMs).
int oracle_mt_subband(const uint8_t* X, int nchan, size_t in_stride, int nsub, const int32_t* d1, int ncoarse, int ns1,
                      uint32_t* S, size_t s_stride, const int32_t* d2, int nfine, int ns, uint32_t* Y,
                      size_t out_stride) {
    int rc = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int a = 0; a < ncoarse; ++a) {
        uint32_t* Sa = S + (size_t)a * nsub * s_stride;
        int r = oracle_subband_step1(X, nchan, in_stride, nsub, d1 + (size_t)a * nchan, 1, ns1, Sa, s_stride);
        if (r == 0)
            r = oracle_subband_step2(Sa, nsub, s_stride, ns1, d2, nfine, 1, ns, Y + (size_t)a * nfine * out_stride,
                                     out_stride);
        if (r != 0) {
#pragma omp critical
            rc = r;
        }
    }
    return rc;
}

// INT / SNR: rows are series.
int oracle_mt_integrate(const uint32_t* Y, size_t stride, int nrows, int ns, int w, uint32_t* I, size_t i_stride) {
    int rc = 0;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < nrows; ++i) {
        const int r = oracle_integrate(Y + (size_t)i * stride, stride, 1, ns, w, I + (size_t)i * i_stride, i_stride);
        if (r != 0) {
#pragma omp critical
            rc = r;
        }
    }
    return rc;
}

int oracle_mt_snr(const uint32_t* V, size_t stride, int nrows, int n, int ddof, float* snr, uint32_t* argmax) {
    int rc = 0;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < nrows; ++i) {
        const int r = oracle_snr(V + (size_t)i * stride, stride, 1, n, ddof, snr + i, argmax + i);
        if (r != 0) {
#pragma omp critical
            rc = r;
        }
    }
    return rc;
}

}  // extern "C"
