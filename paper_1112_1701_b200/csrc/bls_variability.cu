// f3: the high-variability pre-filter (section 2.2.1): "We
// estimate the value and scatter of the locally expected photometric stability as a function of stellar
// magnitude in 0.1-mag bins, using a sigma-clipped average of the stars detected on each chip.  Objects
// that show a more than 2 sigma increased variability compared to the ensemble expectation are flagged".
// Readings V1-V5: per star the weighted mean magnitude and weighted RMS (fp64),
// cell = (group, 0.1-mag bin), per cell an iterated sigma clip of the members' RMS, flag = RMS above
// expected + nsig * scatter.  Five small kernels, all on the caller's stream:
//   var_stats_kernel     one CTA per star: status, mean magnitude, RMS, cell          (like a0 prep)
//   var_count_kernel     members per cell (integer atomics: exact in any order)
//   var_scan_kernel      exclusive scan of the counts -> cell offsets
//   var_scatter_kernel   STABLE counting-sort scatter by one CTA: members of a cell in star order, so
//                        every later sum runs in a fixed order (bitwise reproducible)
//   var_clip_kernel      one CTA per cell: iterated sigma clip (fixed-shape block reductions), then the
//                        per-star expected value, scatter, kept count and flag
#include "bls_internal.cuh"

namespace bls {

constexpr int kVarThreads = kPrepThreads;     // block_sum's shape
constexpr int kScatterThreads = 1024;

__global__ void __launch_bounds__(kVarThreads)
var_stats_kernel(const float *__restrict__ t, const float *__restrict__ mag, const float *__restrict__ sigma,
                 const int64_t *__restrict__ offsets, const int32_t *__restrict__ group, int n_groups, double mag_lo,
                 double mag_bin, int n_mag_bins, int32_t *__restrict__ status, double *__restrict__ mean_mag,
                 double *__restrict__ rms, int32_t *__restrict__ cell)
{
    __shared__ double sh[kVarThreads / 32];
    __shared__ int s_flags;
    const int64_t c = blockIdx.x;
    const int64_t beg = offsets[c], end = offsets[c + 1];
    if (threadIdx.x == 0) s_flags = 0;
    __syncthreads();
    double acc = 0.0;
    int flags = 0;
    for (int64_t i = beg + threadIdx.x; i < end; i += kVarThreads) {
        const float ti = t[i], mi = mag[i], si = sigma[i];
        if (!isfinite(ti) || !isfinite(mi) || !isfinite(si)) flags |= 1;
        else if (!(si > 0.0f)) flags |= 2;
        else { const double s = (double)si; acc += 1.0 / (s * s); }
    }
    if (flags) atomicOr(&s_flags, flags);
    const double sw = block_sum(acc, sh);
    __syncthreads();
    int st = BLS_CURVE_OK;
    if (end - beg < 2) st = BLS_CURVE_TOO_FEW;
    else if (s_flags & 1) st = BLS_CURVE_NONFINITE;
    else if (s_flags & 2) st = BLS_CURVE_BAD_SIGMA;
    else if (!isfinite(sw) || !(sw > 0.0)) st = BLS_CURVE_NONFINITE;
    double mu = 0.0, r = 0.0;
    int ce = -1;
    if (st == BLS_CURVE_OK) {
        acc = 0.0;
        for (int64_t i = beg + threadIdx.x; i < end; i += kVarThreads) {
            const double s = (double)sigma[i];
            acc += ((1.0 / (s * s)) / sw) * (double)mag[i];
        }
        mu = block_sum(acc, sh);
        acc = 0.0;
        for (int64_t i = beg + threadIdx.x; i < end; i += kVarThreads) {
            const double s = (double)sigma[i];
            const double x = (double)mag[i] - mu;
            acc += ((1.0 / (s * s)) / sw) * x * x;
        }
        r = sqrt(block_sum(acc, sh));
        const double b = floor((mu - mag_lo) / mag_bin);                 // reading V2
        const int g = group ? group[c] : 0;
        if (b >= 0.0 && b < (double)n_mag_bins && g >= 0 && g < n_groups) ce = g * n_mag_bins + (int)b;
    }
    if (threadIdx.x == 0) {
        status[c] = st; mean_mag[c] = mu; rms[c] = r; cell[c] = ce;
    }
}

__global__ void var_count_kernel(const int32_t *__restrict__ cell, int64_t n, int32_t *__restrict__ count)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < n && cell[c] >= 0) atomicAdd(&count[cell[c]], 1);
}

__global__ void var_scan_kernel(const int32_t *__restrict__ count, int n_cells, int32_t *__restrict__ offset,
                                int32_t *__restrict__ cursor)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        int32_t run = 0;
        for (int i = 0; i < n_cells; ++i) { offset[i] = run; cursor[i] = run; run += count[i]; }
        offset[n_cells] = run;
    }
}

// One CTA walks the stars in index order, 1024 at a time, one warp after the other; inside a warp the
// rank among lanes of the same cell comes from __match_any_sync.  members[] ends up sorted by
// (cell, star index): a stable counting sort.
__global__ void __launch_bounds__(kScatterThreads)
var_scatter_kernel(const int32_t *__restrict__ cell, int64_t n, int32_t *__restrict__ cursor, int32_t *__restrict__ members)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int64_t base = 0; base < n; base += kScatterThreads) {
        const int64_t c = base + threadIdx.x;
        const int ce = c < n ? cell[c] : -1;
        for (int w = 0; w < kScatterThreads / 32; ++w) {
            if (warp == w) {
                const unsigned active = __ballot_sync(0xffffffffu, ce >= 0);
                if (ce >= 0) {
                    const unsigned same = __match_any_sync(active, ce);
                    const int leader = __ffs(same) - 1;
                    int start = 0;
                    if (lane == leader) { start = cursor[ce]; cursor[ce] = start + __popc(same); }
                    start = __shfl_sync(same, start, leader);
                    members[start + __popc(same & ((1u << lane) - 1u))] = (int32_t)c;
                }
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(kVarThreads)
var_clip_kernel(const int32_t *__restrict__ offset, const int32_t *__restrict__ members, const double *__restrict__ rms,
                double clip, double nsig, int max_iter, int min_members, unsigned char *__restrict__ keep,
                double *__restrict__ expected, double *__restrict__ scatter, int32_t *__restrict__ kept,
                int32_t *__restrict__ flag)
{
    __shared__ double sh[kVarThreads / 32];
    __shared__ int s_dropped;
    const int ce = blockIdx.x;
    const int beg = offset[ce], end = offset[ce + 1];
    if (beg == end) return;
    for (int i = beg + threadIdx.x; i < end; i += kVarThreads) keep[i] = 1;
    __syncthreads();
    double E = 0.0, S = 0.0, nk = 0.0;
    for (int it = 0; it <= max_iter; ++it) {                   // reading V4
        double a = 0.0, cnt = 0.0;
        for (int i = beg + threadIdx.x; i < end; i += kVarThreads)
            if (keep[i]) { a += rms[members[i]]; cnt += 1.0; }
        const double tot = block_sum(a, sh);
        nk = block_sum(cnt, sh);
        if (nk == 0.0) { E = 0.0; S = 0.0; break; }
        E = tot / nk;
        a = 0.0;
        for (int i = beg + threadIdx.x; i < end; i += kVarThreads)
            if (keep[i]) { const double d = rms[members[i]] - E; a += d * d; }
        S = sqrt(block_sum(a, sh) / nk);
        if (it == max_iter) break;
        if (threadIdx.x == 0) s_dropped = 0;
        __syncthreads();
        int dropped = 0;
        for (int i = beg + threadIdx.x; i < end; i += kVarThreads)
            if (keep[i] && fabs(rms[members[i]] - E) > clip * S) { keep[i] = 0; dropped = 1; }
        if (dropped) s_dropped = 1;
        __syncthreads();
        if (!s_dropped) break;
        __syncthreads();
    }
    const int nkept = (int)nk;
    for (int i = beg + threadIdx.x; i < end; i += kVarThreads) {   // reading V5
        const int c = members[i];
        if (expected) expected[c] = E;
        if (scatter) scatter[c] = S;
        if (kept) kept[c] = nkept;
        if (flag) flag[c] = (nkept >= min_members && rms[c] > E + nsig * S) ? 1 : 0;
    }
}

__global__ void var_fill_kernel(int64_t n, double *expected, double *scatter, int32_t *kept, int32_t *flag)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    if (expected) expected[c] = 0.0;
    if (scatter) scatter[c] = 0.0;
    if (kept) kept[c] = 0;
    if (flag) flag[c] = 0;
}

cudaError_t launch_variability(const float *t, const float *mag, const float *sigma, const int64_t *d_offsets,
                               const int32_t *group, int64_t n, const bls_variability_config &cfg, int32_t *status,
                               double *mean_mag, double *rms, int32_t *cell, int32_t *count, int32_t *offset,
                               int32_t *cursor, int32_t *members, unsigned char *keep, double *expected,
                               double *scatter, int32_t *kept, int32_t *flag, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    const int n_cells = cfg.n_groups * cfg.n_mag_bins;
    const unsigned nb256 = (unsigned)((n + 255) / 256);
    var_stats_kernel<<<(unsigned)n, kVarThreads, 0, st>>>(t, mag, sigma, d_offsets, group, cfg.n_groups, cfg.mag_lo,
                                                         cfg.mag_bin, cfg.n_mag_bins, status, mean_mag, rms, cell);
    cudaError_t e = cudaMemsetAsync(count, 0, sizeof(int32_t) * (size_t)n_cells, st);
    if (e != cudaSuccess) return e;
    var_fill_kernel<<<nb256, 256, 0, st>>>(n, expected, scatter, kept, flag);
    var_count_kernel<<<nb256, 256, 0, st>>>(cell, n, count);
    var_scan_kernel<<<1, 32, 0, st>>>(count, n_cells, offset, cursor);
    var_scatter_kernel<<<1, kScatterThreads, 0, st>>>(cell, n, cursor, members);
    var_clip_kernel<<<(unsigned)n_cells, kVarThreads, 0, st>>>(offset, members, rms, cfg.clip, cfg.nsig, cfg.max_iter,
                                                             cfg.min_members, keep, expected, scatter, kept, flag);
    return cudaGetLastError();
}

}  // namespace bls

// ---- bls_variability_noalloc: the same filter for callers that must not allocate (include/bls.h) ------------
// Everything bls_variability takes from cudaMallocAsync lives here instead, in one array that is part of the
// library image: each GPU that loads the library carries its own copy (BLS_NOALLOC_SCRATCH_BYTES) until the
// process ends.  The slots are those of bls_variability's scratch block at the fixed maximum sizes.
#include <math.h>

#include <mutex>

namespace {

constexpr size_t na_pad(size_t bytes) { return (bytes + 255) & ~(size_t)255; }
constexpr size_t kNaStars = BLS_NOALLOC_MAX_STARS, kNaCells = BLS_NOALLOC_MAX_CELLS;
constexpr size_t kNaOffsets = 0;                                          // int64 [stars + 1]  device copy of batch->offsets
constexpr size_t kNaStatus = kNaOffsets + na_pad((kNaStars + 1) * 8);     // int32 [stars]      used when out->status is NULL
constexpr size_t kNaCell = kNaStatus + na_pad(kNaStars * 4);              // int32 [stars]      ... out->cell
constexpr size_t kNaMembers = kNaCell + na_pad(kNaStars * 4);             // int32 [stars]      stars sorted by (cell, index)
constexpr size_t kNaCount = kNaMembers + na_pad(kNaStars * 4);            // int32 [cells]      members per cell: MUST START AT ZERO
constexpr size_t kNaOffset = kNaCount + na_pad(kNaCells * 4);             // int32 [cells + 1]  exclusive scan of the counts
constexpr size_t kNaCursor = kNaOffset + na_pad((kNaCells + 1) * 4);      // int32 [cells]      write positions of the scatter
constexpr size_t kNaMean = kNaCursor + na_pad(kNaCells * 4);              // double [stars]     ... out->mean_mag
constexpr size_t kNaRms = kNaMean + na_pad(kNaStars * 8);                 // double [stars]     ... out->rms
constexpr size_t kNaKeep = kNaRms + na_pad(kNaStars * 8);                 // uint8 [stars]      clip marks, by member position
constexpr size_t kNaBytes = kNaKeep + na_pad(kNaStars);
static_assert(kNaBytes == BLS_NOALLOC_SCRATCH_BYTES, "bls.h states the size of the built-in scratch");

constexpr int kNaMaxDevices = 64;
std::mutex g_na_mutex;
unsigned char *g_na_address[kNaMaxDevices];   // g_na_address[d]: where the array lives on GPU d (nullptr = not looked up yet)

}  // namespace

// In HOST code this name is only a handle for the runtime: it is NOT a device address and must never be handed
// to a kernel or to cudaMemcpyAsync as a pointer.  The address on the current GPU comes from cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNaBytes];

// Where the built-in array lives on `device`, which must be the current device.  The first call per GPU asks the
// runtime (no allocation; the array came with the library image) and every later call reuses the answer.
static cudaError_t noalloc_scratch_on(int device, unsigned char **address)
{
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_address[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_na_address[device] = (unsigned char *)p;
    }
    *address = g_na_address[device];
    return cudaSuccess;
}

extern "C" {
#pragma GCC visibility push(default)

int bls_variability_noalloc(int32_t device, const bls_variability_config *cfg, const bls_batch *b, const int32_t *group,
                            const bls_variability_outputs *out, void *cuda_stream)
{
    // the checks of bls_variability, in its order
    if (!cfg || !b || !out) return BLS_ERR_NULL;
    if (cfg->struct_size != (int32_t)sizeof(bls_variability_config)) return BLS_ERR_CONFIG;
    if (cfg->n_groups < 1 || cfg->n_mag_bins < 1 || (int64_t)cfg->n_groups * cfg->n_mag_bins > (1 << 24)) return BLS_ERR_CONFIG;
    if (!(cfg->mag_bin > 0.0) || !isfinite(cfg->mag_lo) || !(cfg->clip > 0.0) || !isfinite(cfg->nsig)) return BLS_ERR_CONFIG;
    if (cfg->max_iter < 0 || cfg->max_iter > 100 || cfg->min_members < 0) return BLS_ERR_CONFIG;
    if (b->n_curves < 0) return BLS_ERR_BATCH;
    if (!b->offsets) return BLS_ERR_NULL;
    if (device < 0 || device >= kNaMaxDevices) return BLS_ERR_ARG;
    const int64_t nc = b->n_curves;
    const int64_t n_cells = (int64_t)cfg->n_groups * cfg->n_mag_bins;
    // the fixed capacity, before the offsets are walked and before any CUDA call
    if (nc > (int64_t)kNaStars || n_cells > (int64_t)kNaCells) return BLS_ERR_CAPACITY;
    if (b->offsets[0] != 0) return BLS_ERR_BATCH;
    for (int64_t c = 0; c < nc; ++c)
        if (b->offsets[c + 1] < b->offsets[c]) return BLS_ERR_BATCH;
    if (b->offsets[nc] > 0 && (!b->t || !b->mag || !b->sigma)) return BLS_ERR_NULL;
    if (nc == 0) return BLS_OK;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned char *scr = nullptr;
    if (noalloc_scratch_on(device, &scr) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaError_t e = cudaMemcpyAsync(scr + kNaOffsets, b->offsets, (size_t)(nc + 1) * 8, cudaMemcpyHostToDevice, st);
    int32_t *status = out->status ? out->status : (int32_t *)(scr + kNaStatus);
    int32_t *cell = out->cell ? out->cell : (int32_t *)(scr + kNaCell);
    double *mean_mag = out->mean_mag ? out->mean_mag : (double *)(scr + kNaMean);
    double *rms = out->rms ? out->rms : (double *)(scr + kNaRms);
    // launch_variability zeroes the member counts on `st` (cudaMemsetAsync) before the count kernel: the one slot
    // that must not carry the previous call's contents.  Every other slot is written before it is read: status,
    // cell, mean, rms by the per-star kernel; offset and cursor for all cells by the scan; members by the scatter;
    // keep, over exactly the member positions in use, at the top of the clip kernel.
    if (e == cudaSuccess)
        e = bls::launch_variability(b->t, b->mag, b->sigma, (const int64_t *)(scr + kNaOffsets), group, nc, *cfg, status,
                                    mean_mag, rms, cell, (int32_t *)(scr + kNaCount), (int32_t *)(scr + kNaOffset),
                                    (int32_t *)(scr + kNaCursor), (int32_t *)(scr + kNaMembers), scr + kNaKeep,
                                    out->expected, out->scatter, out->kept, out->flag, st);
    if (e != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    return BLS_OK;
}

#pragma GCC visibility pop
}  // extern "C"
