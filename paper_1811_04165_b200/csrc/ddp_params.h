// Kernel parameter records (plain data, passed by value at launch).  Included by the host launch
// code and by the device templates, both ahead-of-time (nvcc) and at tune time (NVRTC, where this
// text is concatenated in front of ddp_kernels.cuh) -- so no standard headers here.
#ifndef DDP_PARAMS_H_
#define DDP_PARAMS_H_

#define DDP_MAXW 16

// One dedispersion-type launch: out[g][i][t] = sum_{r<nred} in[g][r][t + delay[g][i][r]].
//   direct:        g = 0,           i = DM trial,   r = channel
//   subband step 1: g = subband s,   i = coarse DM a, r = channel within the subband
//   subband step 2: g = coarse DM a, i = fine DM b,   r = subband
struct DdpDedispParams {
    const void* in;              // rows of the input element type
    unsigned int* out;           // uint32 sums
    const int* delay;            // int32 delay table (device)
    long long in_row_stride;     // elements between consecutive reduction rows r
    long long in_group_stride;   // elements between the first rows of consecutive groups g
    long long in_row_len;        // readable elements per input row (loads are clipped to it)
    long long out_dm_stride;     // elements between consecutive i of one group
    long long out_group_stride;  // elements between the i = 0 rows of consecutive groups
    int delay_dm_stride;         // ints between consecutive i in the delay table
    int delay_group_off;         // ints between consecutive g in the delay table
    int nred;                    // reduction length
    int ndm;                     // length of the i axis
    int ns;                      // output samples per row
    int win;                     // staged modes: elements of one staged row window in shared memory
    const int* rowmap;           // channel mask: input row of reduction row g*nred + r, -1 = masked; null = no mask
    const unsigned char* zero_row;  //   the row of zeros a masked reduction row reads (in_row_len bytes)
    int one;                     // the value 1, unknown to the compiler (packed kernel: adds issued as IMAD)
    int vmax;                    // merged staging: variant slots per table record (largest variant count of the plan, padded to 4)
    int lw;                      // merged staging: words per variant row  (TT/2 + largest window spread, padded)
    int le;                      // merged staging: words per expanded channel row
    int rows_max;                // merged staging: variant rows per buffer = largest sum of variant counts over a chunk's groups
    const unsigned char* meta;   // merged staging: resident DdpMergeTable blob (device), one record per (DM tile, group)
    int meta_rw;                 //   int32 words per record
    int meta_ngg;                //   groups per DM tile in the table (all subbands)
    int meta_gg0_stride;         //   table groups between consecutive kernel groups g (subband step 1: cps / G; direct: 0)
    int threads_t, threads_dm;   // merged staging: consumer threads along time / DM (the block adds 4 or 8 producer warps)
    int n_ttiles, n_dtiles;      // merged staging (persistent kernel): time tiles, DM tiles,
    int nseg;                    //   segments of <= 256 reduction rows per tile,
    int nunits;                  //   work units = groups * n_dtiles * n_ttiles * nseg
};

// Integration: plane k holds I_w[i][j] = sum_{m<w} in[i][j*w+m] for w = width[k] > 1.
struct DdpIntegParams {
    const unsigned int* in;      // dedispersed series uint32 [ndm][in_stride]
    unsigned int* out;           // base of the planes
    long long in_stride;
    long long plane_off[DDP_MAXW];
    long long plane_stride[DDP_MAXW];
    int plane_len[DDP_MAXW];     // n_w
    int width[DDP_MAXW];
    int nplanes;                 // widths > 1 only
    int ndm;
    int ns;
    int tiles_per_block;         // consecutive time tiles one block walks (gene "unroll")
    int max_lvl;                 // log2 of the largest width
    int lvl_plane[DDP_MAXW];     // plane index of width 2^m, -1 if that width is not requested
};

// S/N (BJ:cfg0): series k of row i = n[k] values at base[k] + i*stride[k].
struct DdpSnrParams {
    const unsigned int* base[DDP_MAXW];
    long long stride[DDP_MAXW];
    int n[DDP_MAXW];
    float* snr;                  // [ndm][nwidths]
    unsigned int* argmax;        // [ndm][nwidths] or null
    int nwidths;
    int ndm;
    int ddof;
};

// Fused integration + S/N: level m = width 2^m; k = index of that width in the plan's width list.
struct DdpIsnrParams {
    const unsigned int* in;      // dedispersed series uint32 [ndm][in_stride]
    unsigned int* planes;        // base of the integration planes, or null: planes are not written
    long long in_stride;
    long long plane_off[DDP_MAXW];     // by width index k (w > 1)
    long long plane_stride[DDP_MAXW];
    int n[DDP_MAXW];             // values of series k: floor(ns / w)
    int lvl_k[DDP_MAXW];         // level m -> width index k, -1 if width 2^m is not requested
    float* snr;                  // [ndm][nwidths]
    unsigned int* argmax;        // [ndm][nwidths] or null
    int nwidths;
    int ndm;
    int ns;
    int ddof;
    int max_lvl;                 // log2 of the largest width
    int width[DDP_MAXW];         // sliding mode: the widths themselves
    int slide_nb;                // sliding mode: prefix-sum ring length in chunks = 1 + ceil(largest width / chunk)
};

#endif  // DDP_PARAMS_H_
