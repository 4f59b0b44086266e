// a1 Load, a2 Fold, a3/a4 box search, per-frequency argmax (DESIGN.md
// "Kernels / search").  PAPER.md L145: "the light curve data is read into fast shared memory by each
// thread block (with memory accesses coalesced for speed), then each thread picks an untested
// period, phases the light curve at that period and then tests a range of durations and phases."
//
// What is kept from that design: the curve is resident in shared memory across a block of trial
// frequencies, and a LANE owns a trial frequency.  What differs (Fermi -> sm_100a):
//   * a CTA owns one curve and a tile of 32 consecutive frequencies at a time; ALL its warps fold
//     the curve into the tile's bins (each warp takes every NW-th point, every lane its own
//     frequency), so the bins of a frequency are private to a lane column: bins[bin][lane] puts
//     lane l in bank l -> the native 32-bit ATOMS.ADD is conflict-free by construction;
//   * bins accumulate int32 fixed point (exact, order independent, bitwise reproducible);
//   * the phase is one DFMA with a magic constant whose low mantissa word is frac(f t) * 2^32;
//     one IMAD.WIDE gives (bin, position inside the bin); positions inside a guard band of a bin
//     edge fall back to the canonical 3-rounding fp64 rule, so bin indices equal the oracle's
//     bit for bit (DESIGN.md "Fold / fast phase" has the error bound);
//   * the box search is register tiled: a thread owns 4 consecutive start bins of its lane's
//     frequency and slides a 7-bin window, so one shared load feeds 4 boxes; sums are direct
//     running sums in bin order (no prefix differences), so boxes holding the same point set tie
//     bitwise and the canonical tie-break (smallest width, then smallest start) applies.
#include "bls_internal.cuh"

namespace bls {

constexpr int NW = kSearchThreads / 32;
constexpr int A = kStartsPerThread;

size_t search_smem_bytes(int nb, int64_t n_points_in_smem)
{
    size_t bins = (size_t)2 * nb * kTileFreqs * 4;
    size_t red = (size_t)2 * NW * kTileFreqs * 4;
    return bins + red + (size_t)n_points_in_smem * sizeof(PointRec);
}

__device__ __noinline__ int canonical_bin(double f, double t, int nb)
{
    double p = __dmul_rn(f, t);
    double phi = __dsub_rn(p, floor(p));
    double xb = __dmul_rn(phi, (double)nb);
    int b = (int)xb;
    return b >= nb ? nb - 1 : b;
}

__device__ __forceinline__ float fast_rcp(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Scalar, guarded re-search of one frequency column; only used when the fast search produced a
// non-finite or impossible value (a box holding the entire weight, r == 1.0f).
__device__ __noinline__ void careful_search(const float *Wf, const float *Yf, int lane, int nb, int kmin,
                                            int kmax, float &bv, uint32_t &bkey)
{
    bv = 0.f; bkey = ((uint32_t)kmin << 16);
    for (int a = 0; a < nb; ++a) {
        float r = 0.f, s = 0.f;
        for (int k = 1; k <= kmax; ++k) {
            int j = a + k - 1; if (j >= nb) j -= nb;
            r += Wf[j * 32 + lane]; s += Yf[j * 32 + lane];
            if (k < kmin) continue;
            float den = fmaf(-r, r, r);
            if (!(den > 0.f) || !(r < 1.f)) continue;
            float v = s * s / den;
            uint32_t key = ((uint32_t)k << 16) | (uint32_t)a;
            if (v > bv || (v == bv && v > 0.f && key < bkey)) { bv = v; bkey = key; }
        }
    }
}

template <bool PTS_SMEM>
__global__ void __launch_bounds__(kSearchThreads)
search_kernel(const SearchArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nb = a.nb;
    uint32_t *Wb = reinterpret_cast<uint32_t *>(smem_raw);              // [nb][32]
    int32_t *Yb = reinterpret_cast<int32_t *>(Wb + nb * 32);            // [nb][32]
    float *red_v = reinterpret_cast<float *>(Yb + nb * 32);             // [NW][32]
    uint32_t *red_key = reinterpret_cast<uint32_t *>(red_v + NW * 32);  // [NW][32]
    PointRec *pts_s = reinterpret_cast<PointRec *>(red_key + NW * 32);  // [n] if PTS_SMEM
    float *Wf = reinterpret_cast<float *>(Wb);
    float *Yf = reinterpret_cast<float *>(Yb);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t curve_local = blockIdx.x / a.items_per_curve;
    const int item = blockIdx.x % a.items_per_curve;
    const int64_t c = a.curve_base + curve_local;
    const int64_t beg = a.offsets[c];
    const int n = (int)(a.offsets[c + 1] - beg);
    const CurveMeta meta = a.meta[c];
    const int ntiles = (a.nf + kTileFreqs - 1) / kTileFreqs;
    const int tile0 = item * a.tiles_per_item;
    const int tile1 = min(tile0 + a.tiles_per_item, ntiles);
    const int kmin = a.kmin, kmax = a.kmax;

    if (meta.status != BLS_CURVE_OK) {   // data fault: zero-filled spectrum (include/bls.h)
        for (int q = tile0 * kTileFreqs + tid; q < min(tile1 * kTileFreqs, a.nf); q += kSearchThreads) {
            a.sr[curve_local * a.nf + q] = 0.f;
            a.ak[curve_local * a.nf + q] = (uint32_t)kmin << 16;
            a.depth[curve_local * a.nf + q] = 0.f;
            if (a.u_sr) a.u_sr[c * a.nf + q] = 0.f;
            if (a.u_start) a.u_start[c * a.nf + q] = 0;
            if (a.u_width) a.u_width[c * a.nf + q] = (uint16_t)kmin;
            if (a.u_depth) a.u_depth[c * a.nf + q] = 0.f;
        }
        return;
    }

    // ---- a1 Load: the curve becomes resident for every tile of this work item -------------------
    const PointRec *pts_g = a.pts + beg;
    if (PTS_SMEM) {
        const uint4 *src = reinterpret_cast<const uint4 *>(pts_g);
        uint4 *dst = reinterpret_cast<uint4 *>(pts_s);
        for (int i = tid; i < n; i += kSearchThreads) dst[i] = __ldg(src + i);
    }
    const PointRec *P = PTS_SMEM ? pts_s : pts_g;
    const bool force_canon = (a.force_canonical != 0) || (meta.force_canonical != 0);
    const float cw = meta.cw, cy = meta.cy;
    const uint32_t G = (uint32_t)nb + 8u;         // guard band, units of 2^-32 bin
    unsigned int n_canon = 0;

    for (int tile = tile0; tile < tile1; ++tile) {
        const int q0 = tile * kTileFreqs;
        const int q = min(q0 + lane, a.nf - 1);    // ragged last tile: surplus lanes repeat the last f
        const double f = a.freqs[q];

        // ---- zero the tile's bins -------------------------------------------------------------
        {
            uint4 *z = reinterpret_cast<uint4 *>(Wb);
            const int nvec = nb * 16;              // 2 * nb * 32 words / 4
            for (int i = tid; i < nvec; i += kSearchThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
        }
        __syncthreads();

        // ---- a2 Fold: warp w takes points w, w+NW, ...; lane l folds them at its frequency ------
#pragma unroll 4
        for (int i = warp; i < n; i += NW) {
            PointRec p;
            if (PTS_SMEM) p = P[i];
            else {
                uint4 raw = __ldg(reinterpret_cast<const uint4 *>(P + i));
                p.t = __hiloint2double((int)raw.y, (int)raw.x); p.qw = raw.z; p.qy = (int32_t)raw.w;
            }
            const int bin = fold_bin(f, p.t, nb, G, force_canon, n_canon);
            atomicAdd(&Wb[bin * 32 + lane], p.qw);
            atomicAdd(&Yb[bin * 32 + lane], p.qy);
        }
        __syncthreads();

        // ---- fixed point -> fp32 weight fraction / weighted residual, in place -------------------
        for (int i = tid; i < nb * 32; i += kSearchThreads) {
            Wf[i] = (float)Wb[i] * cw;
            Yf[i] = (float)Yb[i] * cy;
        }
        __syncthreads();

        // ---- a3/a4 box search: this thread owns start tiles warp, warp+NW, ... of column `lane` --
        float tb_v = 0.f;
        uint32_t tb_key = (uint32_t)kmin << 16;
        const int nst = (nb + A - 1) / A;
        for (int tl = warp; tl < nst; tl += NW) {
            const int a0 = tl * A;
            float r[A], s[A], ww[2 * A - 1], wy[2 * A - 1];
#pragma unroll
            for (int u = 0; u < A; ++u) { r[u] = 0.f; s[u] = 0.f; }
#pragma unroll
            for (int i = 0; i < A - 1; ++i) {
                int j = a0 + i; while (j >= nb) j -= nb;
                ww[i] = Wf[j * 32 + lane]; wy[i] = Yf[j * 32 + lane];
            }
            float lb_v = 0.f;
            int lb_code = 0;                       // (k << 8) | u of the tile-local best
            for (int k0 = 0; k0 < kmax; k0 += A) {
#pragma unroll
                for (int i = A - 1; i < 2 * A - 1; ++i) {
                    int j = a0 + k0 + i; while (j >= nb) j -= nb;
                    ww[i] = Wf[j * 32 + lane]; wy[i] = Yf[j * 32 + lane];
                }
#pragma unroll
                for (int jstep = 0; jstep < A; ++jstep) {
                    const int k = k0 + jstep + 1;
#pragma unroll
                    for (int u = 0; u < A; ++u) { r[u] += ww[u + jstep]; s[u] += wy[u + jstep]; }
                    if (k >= kmin && k <= kmax) {
#pragma unroll
                        for (int u = 0; u < A; ++u) {
                            const float den = fmaf(-r[u], r[u], r[u]);      // r (1 - r)
                            const float v = (s[u] * s[u]) * fast_rcp(den);  // NaN (0 * inf) never wins
                            if (v > lb_v) { lb_v = v; lb_code = (k << 8) | u; }
                        }
                    }
                }
#pragma unroll
                for (int i = 0; i < A - 1; ++i) { ww[i] = ww[i + A]; wy[i] = wy[i + A]; }
            }
            if (lb_v > 0.f) {
                int sa = a0 + (lb_code & 0xff); if (sa >= nb) sa -= nb;
                const uint32_t key = ((uint32_t)(lb_code >> 8) << 16) | (uint32_t)sa;
                if (lb_v > tb_v || (lb_v == tb_v && key < tb_key)) { tb_v = lb_v; tb_key = key; }
            }
        }
        red_v[warp * 32 + lane] = tb_v;
        red_key[warp * 32 + lane] = tb_key;
        __syncthreads();

        // ---- merge the NW partial results of each column, recompute (r, s) of the winner ---------
        if (warp == 0) {
            float bv = red_v[lane];
            uint32_t bkey = red_key[lane];
#pragma unroll
            for (int w = 1; w < NW; ++w) {
                const float v = red_v[w * 32 + lane];
                const uint32_t key = red_key[w * 32 + lane];
                if (v > bv || (v == bv && v > 0.f && key < bkey)) { bv = v; bkey = key; }
            }
            if (!(bv <= 1.001f * (float)meta.wx2 + 1e-30f))   // inf / impossible: r == 1.0f box
                careful_search(Wf, Yf, lane, nb, kmin, kmax, bv, bkey);
            const int bk = (int)(bkey >> 16), ba = (int)(bkey & 0xffffu);
            float r = 0.f, s = 0.f;
            for (int j = 0; j < bk; ++j) {
                int b = ba + j; if (b >= nb) b -= nb;
                r += Wf[b * 32 + lane]; s += Yf[b * 32 + lane];
            }
            const float den = fmaf(-r, r, r);
            float sr = 0.f, dp = 0.f;
            if (bv > 0.f && den > 0.f) { sr = (s * s) / den; dp = s / den; }
            if (q0 + lane < a.nf) {
                const int64_t o = curve_local * a.nf + q0 + lane;
                a.sr[o] = sr; a.ak[o] = bkey; a.depth[o] = dp;
                const int64_t uo = c * a.nf + q0 + lane;
                if (a.u_sr) a.u_sr[uo] = sr;
                if (a.u_start) a.u_start[uo] = (uint16_t)ba;
                if (a.u_width) a.u_width[uo] = (uint16_t)bk;
                if (a.u_depth) a.u_depth[uo] = dp;
            }
        }
        __syncthreads();
    }

    if (a.canon_count) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) n_canon += __shfl_xor_sync(0xffffffffu, n_canon, o);
        if (lane == 0 && n_canon) atomicAdd(a.canon_count, (unsigned long long)n_canon);
    }
}

// Diagnostic: the bin index the fold assigns to each (f, t) pair -- the same fold_bin() the search
// kernel inlines.  Lets tests compare bin indices with the oracle on very many pairs.
__global__ void debug_bins_kernel(const double *__restrict__ f, const double *__restrict__ t, int64_t n,
                                  int nb, int force_canon, int32_t *__restrict__ bins,
                                  unsigned long long *__restrict__ n_canon_out)
{
    const uint32_t G = (uint32_t)nb + 8u;
    unsigned int n_canon = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        bins[i] = fold_bin(f[i], t[i], nb, G, force_canon != 0, n_canon);
    if (n_canon && n_canon_out) atomicAdd(n_canon_out, (unsigned long long)n_canon);
}

cudaError_t launch_debug_bins(const double *f, const double *t, int64_t n, int nb, int force_canon,
                              int32_t *bins, unsigned long long *n_canon, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    int64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    debug_bins_kernel<<<(unsigned)blocks, 256, 0, st>>>(f, t, n, nb, force_canon, bins, n_canon);
    return cudaGetLastError();
}

cudaError_t search_configure(int max_smem_optin)
{
    cudaError_t e = cudaFuncSetAttribute(search_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         max_smem_optin);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(search_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                max_smem_optin);
}

cudaError_t launch_search(const SearchArgs &a, int64_t chunk_curves, size_t smem, cudaStream_t st)
{
    const int64_t grid = chunk_curves * (int64_t)a.items_per_curve;
    if (grid <= 0) return cudaSuccess;
    if (grid > 2147483647LL) return cudaErrorInvalidConfiguration;
    if (a.pts_in_smem)
        search_kernel<true><<<(unsigned)grid, kSearchThreads, smem, st>>>(a);
    else
        search_kernel<false><<<(unsigned)grid, kSearchThreads, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace bls
