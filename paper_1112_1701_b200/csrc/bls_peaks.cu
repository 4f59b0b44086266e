// a5 Output (reading R14): per-curve top-k peaks of the SR spectrum.
// A sample q is a peak iff SR[q] > 0 and (q == 0 or SR[q] > SR[q-1]) and (q == nf-1 or
// SR[q] >= SR[q+1]); peaks are ranked by SR descending, then index ascending.  One CTA per curve
// selects max_k peaks in max_k rounds; each round is a block-wide argmax over the candidates that
// rank strictly after the previous pick.  The spectrum row is nf*4 bytes (<= 2 MB) and stays in
// L1/L2 across rounds, so HBM sees it once.
// With a minimum separation (bls_plan_set_peak_min_sep; SURVEY 8(c) reading 14) a candidate must also lie MORE than
// min_sep grid steps from every peak picked in the earlier rounds: the round's argmax over the peaks that are still
// allowed is exactly the greedy walk in rank order (a peak passed over because it was too close stays too close,
// the accepted set only grows, and it suppresses nothing itself).
#include "bls_internal.cuh"

namespace bls {

// rank key: larger = better.  SR > 0, so its bit pattern orders like its value.
__device__ __forceinline__ unsigned long long rank_key(float sr, int q)
{
    return ((unsigned long long)__float_as_uint(sr) << 32) | (unsigned long long)(0xffffffffu - (uint32_t)q);
}

__global__ void __launch_bounds__(kPeakThreads)
peaks_kernel(const float *__restrict__ sr, const uint32_t *__restrict__ ak, const float *__restrict__ depth,
             const CurveMeta *__restrict__ meta, int64_t curve_base, int nf, int max_k, int min_sep,
             PeakCand *__restrict__ cand, double2 *__restrict__ sr_stats)
{
    __shared__ int s_acc[32];                  // indices picked so far (max_top_k <= 32)
    __shared__ unsigned long long sh[kPeakThreads / 32];
    __shared__ double shd[kPeakThreads / 32];
    __shared__ unsigned long long s_prev;
    const int64_t cl = blockIdx.x;
    const int64_t c = curve_base + cl;
    const float *row = sr + cl * (int64_t)nf;
    PeakCand *out = cand + c * (int64_t)max_k;
    const bool ok = meta[c].status == BLS_CURVE_OK;

    // reading S1: mean and population standard deviation of the curve's spectrum (for bls_refine's SDE);
    // fixed strided order + fixed tree, two passes like the oracle's
    {
        double a = 0.0;
        for (int q = threadIdx.x; q < nf; q += kPeakThreads) a += (double)row[q];
        const double mean = block_sum(a, shd) / (double)nf;
        a = 0.0;
        for (int q = threadIdx.x; q < nf; q += kPeakThreads) { const double d = (double)row[q] - mean; a += d * d; }
        const double sd = sqrt(block_sum(a, shd) / (double)nf);
        if (threadIdx.x == 0) sr_stats[c] = make_double2(mean, sd);
        __syncthreads();
    }

    unsigned long long prev = ~0ull;           // everything ranks after "infinity"
    for (int round = 0; round < max_k; ++round) {
        unsigned long long best = 0ull;        // 0 = no candidate (SR > 0 makes every real key > 0)
        if (ok) {
            for (int q = threadIdx.x; q < nf; q += kPeakThreads) {
                const float v = row[q];
                if (!(v > 0.f)) continue;
                if (q > 0 && !(v > row[q - 1])) continue;
                if (q < nf - 1 && !(v >= row[q + 1])) continue;
                const unsigned long long key = rank_key(v, q);
                if (key < prev && key > best) {
                    bool far = true;
                    if (min_sep > 0)
                        for (int j = 0; j < round; ++j) far = far && abs(q - s_acc[j]) > min_sep;
                    if (far) best = key;
                }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
            best = other > best ? other : best;
        }
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = best;
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long b = 0ull;
#pragma unroll
            for (int w = 0; w < kPeakThreads / 32; ++w) b = sh[w] > b ? sh[w] : b;
            s_prev = b;
            PeakCand pc;
            if (b == 0ull) { pc.freq_index = -1; pc.sr = 0.f; pc.depth = 0.f; pc.ak = 0u; }
            else {
                const int q = (int)(0xffffffffu - (uint32_t)(b & 0xffffffffull));
                pc.freq_index = q;
                s_acc[round] = q;
                pc.sr = row[q];
                pc.depth = depth[cl * (int64_t)nf + q];
                pc.ak = ak[cl * (int64_t)nf + q];
            }
            out[round] = pc;
        }
        __syncthreads();
        prev = s_prev;
        if (prev == 0ull) {                    // list exhausted: pad the rest
            for (int r2 = round + 1 + threadIdx.x; r2 < max_k; r2 += kPeakThreads) {
                PeakCand pc; pc.freq_index = -1; pc.sr = 0.f; pc.depth = 0.f; pc.ak = 0u;
                out[r2] = pc;
            }
            break;
        }
    }
}

__global__ void format_peaks_kernel(const PeakCand *__restrict__ cand, int max_k, int k, int64_t n_curves,
                                    int nb, const double *__restrict__ freqs,
                                    const double *__restrict__ t_origin, bls_peak *__restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_curves * (int64_t)k) return;
    const int64_t c = i / k;
    const int j = (int)(i % k);
    const PeakCand pc = cand[c * (int64_t)max_k + j];
    bls_peak p;
    p.freq_index = pc.freq_index;
    p.sr = pc.sr;
    p.depth = pc.depth;
    p.start_bin = (uint16_t)(pc.ak & 0xffffu);
    p.width_bins = (uint16_t)(pc.ak >> 16);
    if (pc.freq_index >= 0) {
        p.freq = freqs[pc.freq_index];
        const double mid = ((double)p.start_bin + 0.5 * (double)p.width_bins) / (double)nb;
        p.epoch = (t_origin ? t_origin[c] : 0.0) + mid / p.freq;
    } else {
        p.freq = 0.0;
        p.epoch = 0.0;
    }
    out[i] = p;
}

// ---- f1: refinement around the peaks (readings S2-S4) -------------------
// refine_grid_kernel: (f_lo, step) of the fine grid of every (curve, peak): the peak's two neighbours on
// the coarse grid, step = (f_hi - f_lo)/(n_fine - 1) by IEEE division (as the oracle).  Padded peaks get
// the first coarse frequency and step 0 (their results are discarded).
__global__ void refine_grid_kernel(const PeakCand *__restrict__ cand, int max_k, int k, int64_t n_curves, int nf,
                                   int n_fine, const double *__restrict__ freqs, double *__restrict__ f_lo,
                                   double *__restrict__ f_step)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_curves * (int64_t)k) return;
    const int64_t c = i / k;
    const int q = cand[c * (int64_t)max_k + (int)(i % k)].freq_index;
    double lo = freqs[0], st = 0.0;
    if (q >= 0) {
        lo = freqs[max(q - 1, 0)];
        const double hi = freqs[min(q + 1, nf - 1)];
        st = n_fine > 1 ? __ddiv_rn(__dsub_rn(hi, lo), (double)(n_fine - 1)) : 0.0;
    }
    f_lo[i] = lo;
    f_step[i] = st;
}

// refine_reduce_kernel: one warp per (curve, peak) picks the best of its n_fine * n_shift fine entries
// (largest SR, ties to the smallest index: reading S4) and writes the refined record.
__global__ void refine_reduce_kernel(const float *__restrict__ sr, const uint32_t *__restrict__ ak,
                                     const float *__restrict__ depth, const PeakCand *__restrict__ cand, int max_k, int k,
                                     int64_t curve_base, int64_t chunk_curves, int n_fine, int n_shift, int nb,
                                     const double *__restrict__ f_lo, const double *__restrict__ f_step,
                                     const double2 *__restrict__ sr_stats, const double *__restrict__ t_origin,
                                     bls_refined_peak *__restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const int64_t wi = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (wi >= chunk_curves * (int64_t)k) return;
    const int64_t cl = wi / k;
    const int peak = (int)(wi % k);
    const int64_t c = curve_base + cl;
    const int m = n_fine * n_shift;
    const int64_t row = (cl * k + peak) * (int64_t)m;
    unsigned long long best = 0ull;               // (SR bits << 32) | ~index : SR > 0 orders like its bits
    for (int q = lane; q < m; q += 32) {
        const float v = sr[row + q];
        if (v > 0.f) {
            const unsigned long long key = ((unsigned long long)__float_as_uint(v) << 32) | (0xffffffffu - (uint32_t)q);
            best = key > best ? key : best;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
        best = other > best ? other : best;
    }
    if (lane != 0) return;
    const PeakCand pc = cand[c * (int64_t)max_k + peak];
    bls_refined_peak r;
    r.freq_index = pc.freq_index;
    r.fine_index = -1; r.shift_index = -1;
    r.start_bin = 0; r.width_bins = 0;
    r.sr = 0.f; r.depth = 0.f; r.sde = 0.f; r.coarse_sr = pc.freq_index >= 0 ? pc.sr : 0.f;
    r.freq = 0.0; r.period = 0.0; r.epoch = 0.0; r.duration = 0.0;
    if (pc.freq_index >= 0) {
        const double2 ms = sr_stats[c];
        r.sde = ms.y > 0.0 ? (float)(((double)pc.sr - ms.x) / ms.y) : 0.f;
        if (best != 0ull) {
            const int q = (int)(0xffffffffu - (uint32_t)(best & 0xffffffffull));
            const int j = q / n_shift, h = q - j * n_shift;
            const int64_t pi = c * (int64_t)k + peak;
            const uint32_t akv = ak[row + q];
            r.fine_index = j; r.shift_index = h;
            r.start_bin = (uint16_t)(akv & 0xffffu); r.width_bins = (uint16_t)(akv >> 16);
            r.sr = sr[row + q]; r.depth = depth[row + q];
            r.freq = __dadd_rn(f_lo[pi], __dmul_rn((double)j, f_step[pi]));
            r.period = 1.0 / r.freq;
            const double shift = (double)h / (double)(n_shift * nb);
            const double mid = ((double)r.start_bin + 0.5 * (double)r.width_bins) / (double)nb + shift;
            r.epoch = (t_origin ? t_origin[c] : 0.0) + mid / r.freq;
            r.duration = ((double)r.width_bins / (double)nb) / r.freq;
        }
    }
    out[c * (int64_t)k + peak] = r;
}

cudaError_t launch_refine_grid(const PeakCand *cand, int max_k, int k, int64_t n_curves, int nf, int n_fine,
                               const double *freqs, double *f_lo, double *f_step, cudaStream_t st)
{
    const int64_t total = n_curves * (int64_t)k;
    if (total <= 0) return cudaSuccess;
    refine_grid_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(cand, max_k, k, n_curves, nf, n_fine, freqs, f_lo, f_step);
    return cudaGetLastError();
}

cudaError_t launch_refine_reduce(const float *sr, const uint32_t *ak, const float *depth, const PeakCand *cand, int max_k,
                                 int k, int64_t curve_base, int64_t chunk_curves, int n_fine, int n_shift, int nb,
                                 const double *f_lo, const double *f_step, const double2 *sr_stats, const double *t_origin,
                                 bls_refined_peak *out, cudaStream_t st)
{
    const int64_t warps = chunk_curves * (int64_t)k;
    if (warps <= 0) return cudaSuccess;
    refine_reduce_kernel<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, st>>>(sr, ak, depth, cand, max_k, k, curve_base,
                                                                              chunk_curves, n_fine, n_shift, nb, f_lo, f_step,
                                                                              sr_stats, t_origin, out);
    return cudaGetLastError();
}

cudaError_t launch_peaks(const float *sr, const uint32_t *ak, const float *depth, const CurveMeta *meta,
                         int64_t curve_base, int64_t chunk_curves, int nf, int max_k, int min_sep, PeakCand *cand,
                         double2 *sr_stats, cudaStream_t st)
{
    static_assert(kPeakThreads == kPrepThreads, "block_sum's shape");
    if (chunk_curves <= 0) return cudaSuccess;
    peaks_kernel<<<(unsigned)chunk_curves, kPeakThreads, 0, st>>>(sr, ak, depth, meta, curve_base, nf, max_k, min_sep, cand, sr_stats);
    return cudaGetLastError();
}

cudaError_t launch_format_peaks(const PeakCand *cand, int max_k, int k, int64_t n_curves, int nb,
                                const double *freqs, const double *t_origin, bls_peak *out, cudaStream_t st)
{
    const int64_t total = n_curves * (int64_t)k;
    if (total <= 0) return cudaSuccess;
    const int threads = 256;
    const int64_t blocks = (total + threads - 1) / threads;
    format_peaks_kernel<<<(unsigned)blocks, threads, 0, st>>>(cand, max_k, k, n_curves, nb, freqs, t_origin, out);
    return cudaGetLastError();
}

}  // namespace bls
