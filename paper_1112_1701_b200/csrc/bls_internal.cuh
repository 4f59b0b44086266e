// Internal declarations shared by the translation units of libbls_b200.so (sm_100a only).
// Nothing here is visible through the C ABI (include/bls.h) and nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bls.h"

namespace bls {

// One prepared point, 16 bytes so that one LDS.128 broadcast feeds a whole warp (DESIGN.md
// "Data layout").  t is widened to fp64 once here instead of once per point-fold.
struct __align__(16) PointRec {
    double t;      // days relative to the curve's origin (exactly the caller's fp32 value)
    uint32_t qw;   // rint(w_i * SW)            fixed-point weight
    int32_t qy;    // rint(w_i * x_i * SY)      fixed-point weighted residual
};

// Per-curve constants written by the prep kernel.  The bins hold exact integer sums of qw / qy;
// with SWT = sum_i qw_i (exact) a box of integer sums (R, S) has r = R/SWT, 1-r = (SWT-R)/SWT and
//   SR = S^2/(R (SWT-R)) * sr_scale ,  depth = S/(R (SWT-R)) * dp_scale
struct CurveMeta {
    float ncw;         // -1/SWT : the box search accumulates n = -r (one FFMA2 per box pair)
    float cy;          // 1/SY : bin integer -> weighted residual s (0 for a constant curve)
    int32_t status;    // BLS_CURVE_*
    int32_t force_canonical;  // 1: |f t| may reach 2^18 cycles, the fast phase is not valid
    uint32_t swt;      // sum_i qw_i (exact; < 2^32)
    uint32_t w0;       // sum of qw over the zero-time points (t == 0), which are not in the record list
    int32_t y0;        // sum of qy over them
    int32_t pad_;
    double sr_scale;   // SWT^2 / SY^2   (0 for a constant curve)
    double dp_scale;   // SWT^2 / SY
    double wx2;        // sum_i w_i x_i^2  (upper bound of SR)
};

// Peak candidate kept in the plan between bls_run and bls_topk.
struct PeakCand {
    int32_t freq_index;   // -1 = none
    float sr;
    float depth;
    uint32_t ak;          // start | width << 16
};

constexpr int kTileFreqs = 32;        // frequencies per tile = lanes of a warp
constexpr int kMaxSearchWarps = 10;   // kernel 1 upper bound (BLS_FLAG_WARPS override); 2 CTAs x 10 warps x 96 registers fill an SM
constexpr int kWsMaxWarps = 20;       // warp-specialised kernel: search warps + fold warps
constexpr int kWsSearchWarps = 8;     // launch shape 0 (equal registers): 8 search (two per SM sub-partition) + 12 fold; 20 warps = 5 per sub-partition leave 96 registers per thread
constexpr int kSmax = 8;              // starts per start tile a search thread holds at 96 registers
constexpr int kSmaxWide = 13;         // ... and with the registers the fold warps hand over (kernel 2, shapes 1 and 2)
constexpr int kWsShapes = 3;          // kernel 2 launch shapes (WsShape<0..2> in bls_search.cu)
constexpr int kMergeWarps = 8;        // upper bound of the warps that share the exact merge of a tile (BLS_FLAG_MERGE_WARPS)
constexpr int kSmallWarps = 2;        // small shapes: kernel 1 with CTAs of this many warps ...
constexpr int kSmallCtasMin = 8;      // ... when at least this many fit an SM
constexpr int kWtWarps = 5;           // warp-per-tile kernel: warps per CTA (two CTAs per SM)
constexpr int kFieldStars = 3;        // field kernel (kernel 4): stars of a field per CTA that share each epoch's bin index
constexpr int kFieldWarps = 2 * kFieldStars;   // ... and its CTA: all warps fold, then one pair of warps per star searches and merges
constexpr int kPrepThreads = 256;
constexpr int kPeakThreads = 256;

struct SearchArgs {
    const PointRec *pts;        // [n_points] prepared points of the whole batch
    const int64_t *offsets;     // device copy of the CSR offsets
    const int64_t *poffsets;    // [n_curves+1] offsets of the prepared records (each curve padded to a multiple of 4)
    const CurveMeta *meta;      // [n_curves]
    const double *freqs;        // [nf] the plan's grid (search mode)
    const double *f_lo;         // refine mode (n_fine > 0): [n_curves][refine_k] first fine frequency of each peak
    const double *f_step;       //                           and its fine step
    int refine_k, n_fine, n_shift;
    int nf, nb, kmin, kmax;
    int tiles_per_item, items_per_curve;
    int64_t curve_base;         // first curve of this chunk
    int threads;                // CTA size of the search kernel (multiple of 32, <= 32*kMaxSearchWarps)
    int pts_in_smem;            // 1: stage the curve in shared memory, 0: read it through L1
    int fold_depth;             // kernel 2: groups of 4 points a fold warp keeps in flight (1 or 2)
    int nrows;                  // bin rows per buffer: nb + cyclic extension (search_rows_for)
    int search_warps;           // kernel 2: this many search warps (then the fold warps)
    int ws_shape;               // kernel 2: 0 = equal registers, run-time split; 1, 2 = three roles, registers moved with setmaxnreg (WsShape)
    int merge_warps;            // warps that share the exact merge of a tile (1..kMergeWarps; they split the widths)
    int kernel;                 // 1 single buffer, 2 warp-specialised double buffer, 3 one warp per tile, 4 field (kFieldStars stars per CTA)
    int64_t field_curves;       // kernel 4: stars in this launch (the last group may hold fewer than kFieldStars)
    int force_canonical;        // BLS_FLAG_CANONICAL_PHASE
    float *sr;                  // chunk scratch, [chunk_curves][nf]
    uint32_t *ak;
    float *depth;
    float *u_sr;                // optional user outputs, [n_curves][nf] (whole batch), or NULL
    uint16_t *u_start;
    uint16_t *u_width;
    float *u_depth;
    unsigned long long *canon_count;
};

constexpr double kPhaseMagic = 1572864.0;   // 1.5 * 2^20: ulp = 2^-32, valid for |f t| < 2^19

#ifdef __CUDACC__
// Reading R8, the canonical rule: three individually rounded fp64 operations, no FMA.
__device__ __noinline__ int canonical_bin(double f, double t, int nb, double shift);

// Fast phase.  y = RN(f t + 1.5*2^20) has ulp 2^-32, so its low
// mantissa word is frac(f t) in units of 2^-32 cycle (error <= 2^-33 cycle, one rounding).
// ph * nb as a 64-bit product = (bin, position inside the bin in units of 2^-32 bin).  If the
// position is within G = nb + 8 units of a bin edge the canonical rule decides instead; outside
// the guard band both rules provably give floor(nb frac(f t)) (needs |f t| < 2^18).
__device__ __forceinline__ int fast_bin(double f, double t, int nb, uint32_t G, uint32_t &lo, double magic)
{
    const double y = fma(f, t, magic);
    const uint32_t ph = (uint32_t)__double2loint(y);
    const unsigned long long pr = (unsigned long long)ph * (uint32_t)nb + (unsigned long long)G;
    lo = (uint32_t)pr;                                 // position * 2^32 + G
    return (int)(pr >> 32);
}

// Same, returning the whole product: high word = bin, low word = position * 2^32 + G.
__device__ __forceinline__ unsigned long long fast_bin_pos(double f, double t, int nb, uint32_t G, double magic)
{
    const double y = fma(f, t, magic);
    const uint32_t ph = (uint32_t)__double2loint(y);
    return (unsigned long long)ph * (uint32_t)nb + (unsigned long long)G;
}

__device__ __forceinline__ int fold_bin(double f, double t, int nb, uint32_t G, bool force_canon,
                                        unsigned int &n_canon, double magic, double shift)
{
    uint32_t lo;
    int bin = fast_bin(f, t, nb, G, lo, magic);
    if (force_canon || lo < 2u * G) {
        bin = canonical_bin(f, t, nb, shift);
        ++n_canon;
    }
    return bin;
}
#endif

#ifdef __CUDACC__
// Fixed-shape block reductions over kPrepThreads threads (fixed strided accumulation + fixed tree:
// bitwise reproducible).  `sh` holds kPrepThreads / 32 doubles.
__device__ __forceinline__ double block_sum(double v, double *sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double tot = 0.0;
#pragma unroll
    for (int w = 0; w < kPrepThreads / 32; ++w) tot += sh[w];
    return tot;
}

__device__ __forceinline__ double block_max_d(double v, double *sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double tot = 0.0;
#pragma unroll
    for (int w = 0; w < kPrepThreads / 32; ++w) tot = fmax(tot, sh[w]);
    return tot;
}

#endif

// Bin rows a search buffer holds when the start bins are dealt to `slots` half-warps: the nb bins
// plus the cyclic extension the widest box of the last start reaches (bls_search.cu).
int search_rows_for(int nb, int kmax, int slots);
int ws_shape_warps(int shape, int *search_warps);   // kernel 2 launch shape -> warps per CTA, search warps (0 = run-time)
size_t search_smem_bytes(int nb, int kmax, int warps, int buffers, int64_t n_points_in_smem);
size_t field_smem_bytes(int nb, int kmax, int warps, int64_t n_pad);   // kernel 4: kFieldStars bin buffers + field records
cudaError_t launch_debug_bins(const double *f, const double *t, int64_t n, int nb, int force_canon,
                              int32_t *bins, unsigned long long *n_canon, int sm_count, cudaStream_t st);
cudaError_t launch_debug_bins_shift(const double *f, const double *t, int64_t n, int nb, int h, int n_shift, int force_canon,
                                    int32_t *bins, unsigned long long *n_canon, int sm_count, cudaStream_t st);
cudaError_t search_configure(int max_smem_optin);
cudaError_t launch_prep(const float *t, const float *mag, const float *sigma, const int64_t *offsets,
                        const int64_t *poffsets, int64_t n_curves, int64_t field_epochs, double fmax, PointRec *pts,
                        CurveMeta *meta, int32_t *u_status, cudaStream_t st);
cudaError_t launch_variability(const float *t, const float *mag, const float *sigma, const int64_t *d_offsets,
                               const int32_t *group, int64_t n, const bls_variability_config &cfg, int32_t *status,
                               double *mean_mag, double *rms, int32_t *cell, int32_t *count, int32_t *offset,
                               int32_t *cursor, int32_t *members, unsigned char *keep, double *expected,
                               double *scatter, int32_t *kept, int32_t *flag, cudaStream_t st);
cudaError_t launch_window(const float *t, const int64_t *d_offsets, int64_t n_curves, int nf, const double *d_freqs,
                          double duration, int n_phase, int min_events, int32_t *count, double *eff, cudaStream_t st);
cudaError_t launch_search(const SearchArgs &a, int64_t chunk_curves, size_t smem, cudaStream_t st);
cudaError_t launch_peaks(const float *sr, const uint32_t *ak, const float *depth, const CurveMeta *meta,
                         int64_t curve_base, int64_t chunk_curves, int nf, int max_k, int min_sep, PeakCand *cand,
                         double2 *sr_stats, cudaStream_t st);
cudaError_t launch_refine_grid(const PeakCand *cand, int max_k, int k, int64_t n_curves, int nf, int n_fine,
                               const double *freqs, double *f_lo, double *f_step, cudaStream_t st);
cudaError_t launch_refine_reduce(const float *sr, const uint32_t *ak, const float *depth, const PeakCand *cand, int max_k,
                                 int k, int64_t curve_base, int64_t chunk_curves, int n_fine, int n_shift, int nb,
                                 const double *f_lo, const double *f_step, const double2 *sr_stats, const double *t_origin,
                                 bls_refined_peak *out, cudaStream_t st);
cudaError_t launch_format_peaks(const PeakCand *cand, int max_k, int k, int64_t n_curves, int nb,
                                const double *freqs, const double *t_origin, bls_peak *out, cudaStream_t st);

}  // namespace bls
