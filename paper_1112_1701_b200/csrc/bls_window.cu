// f4: eclipse detection efficiency of a cadence (Fig. 13): "the
// probability that at least two eclipses will be observed from an eclipsing target with a specified period,
// after observing window and weather effects have been taken into account", "based on simulations including
// the actual observing cadences of the survey".  Readings W1-W4: the cadence is a
// curve's sorted epoch list; targets of frequency f and eclipse duration d at the n_phase mid-eclipse phases
// phi_k = (k + 1/2)/n_phase; epoch t is in eclipse iff |x - rint(x)| <= h with x = RN(RN(f t) - phi_k),
// h = RN(RN(d/2) f), its eclipse is cycle rint(x); detected iff >= min_events distinct cycles are observed.
//
// One CTA per (cadence, tile of 8 frequencies): the cadence is staged in shared memory once (fp64) and every
// thread walks it for one frequency and kPhasesPerThread phases held in registers, so one LDS and one DMUL
// serve kPhasesPerThread phase tests.  Every decision is an fp64 compare on individually rounded operations
// (the oracle's sequence), so counts are identical, not close.
#include "bls_internal.cuh"

namespace bls {

constexpr int kWinThreads = 256;
constexpr int kWinFreqs = 8;            // frequencies per CTA
constexpr int kPhasesPerThread = 4;
constexpr int kWinChunk = 4096;         // epochs staged at a time

__global__ void __launch_bounds__(kWinThreads)
window_kernel(const float *__restrict__ t, const int64_t *__restrict__ offsets, int nf, const double *__restrict__ freqs,
              double duration, int n_phase, int min_events, int32_t *__restrict__ count, double *__restrict__ eff)
{
    __shared__ double ts[kWinChunk];
    __shared__ int s_det[kWinFreqs];
    const int64_t c = blockIdx.y;
    const int q0 = blockIdx.x * kWinFreqs;
    const int64_t beg = offsets[c], n = offsets[c + 1] - beg;
    const int tpf = kWinThreads / kWinFreqs;                    // threads per frequency
    const int fi = threadIdx.x / tpf, lt = threadIdx.x % tpf;
    const int q = q0 + fi;
    const bool live = q < nf;
    const double f = live ? freqs[q] : 1.0;
    const double h = __dmul_rn(__dmul_rn(0.5, duration), f);
    if (threadIdx.x < kWinFreqs) s_det[threadIdx.x] = 0;
    int det = 0;
    // phases k = lt + tpf * (j + kPhasesPerThread * pass), j < kPhasesPerThread; the pass count is the same for
    // every thread (CTA barriers inside): phases past n_phase are walked and ignored
    const int npass = (n_phase + tpf * kPhasesPerThread - 1) / (tpf * kPhasesPerThread);
    for (int pass = 0; pass < npass; ++pass) {
        const int k0 = lt + pass * tpf * kPhasesPerThread;
        double phi[kPhasesPerThread], last[kPhasesPerThread];
        int ev[kPhasesPerThread];
#pragma unroll
        for (int j = 0; j < kPhasesPerThread; ++j) {
            const int k = k0 + j * tpf;
            phi[j] = __ddiv_rn(__dadd_rn((double)k, 0.5), (double)n_phase);
            ev[j] = 0; last[j] = 0.0;
        }
        for (int64_t base = 0; base < n; base += kWinChunk) {
            const int m = (int)min((int64_t)kWinChunk, n - base);
            __syncthreads();
            for (int i = threadIdx.x; i < m; i += kWinThreads) ts[i] = (double)t[beg + base + i];
            __syncthreads();
            for (int i = 0; i < m; ++i) {
                const double u = __dmul_rn(f, ts[i]);
#pragma unroll
                for (int j = 0; j < kPhasesPerThread; ++j) {
                    const double x = __dsub_rn(u, phi[j]);
                    const double mm = rint(x);
                    if (fabs(__dsub_rn(x, mm)) <= h && (ev[j] == 0 || mm != last[j])) { ++ev[j]; last[j] = mm; }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < kPhasesPerThread; ++j)
            if (live && k0 + j * tpf < n_phase && ev[j] >= min_events) ++det;
    }
    if (det) atomicAdd(&s_det[fi], det);
    __syncthreads();
    if (threadIdx.x < kWinFreqs && q0 + threadIdx.x < nf) {
        const int d = s_det[threadIdx.x];
        count[c * (int64_t)nf + q0 + threadIdx.x] = d;
        eff[c * (int64_t)nf + q0 + threadIdx.x] = (double)d / (double)n_phase;
    }
}

cudaError_t launch_window(const float *t, const int64_t *d_offsets, int64_t n_curves, int nf, const double *d_freqs,
                          double duration, int n_phase, int min_events, int32_t *count, double *eff, cudaStream_t st)
{
    if (n_curves <= 0 || nf <= 0) return cudaSuccess;
    if (n_curves > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)((nf + kWinFreqs - 1) / kWinFreqs), (unsigned)n_curves);
    window_kernel<<<grid, kWinThreads, 0, st>>>(t, d_offsets, nf, d_freqs, duration, n_phase, min_events, count, eff);
    return cudaGetLastError();
}

}  // namespace bls
