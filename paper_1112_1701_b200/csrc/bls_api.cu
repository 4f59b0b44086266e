// C ABI of libbls_b200.so (include/bls.h): plan lifetime, validation, scratch ownership, launch
// geometry and chunking.  Every arithmetic step of the path runs in the kernels of bls_prep.cu,
// bls_search.cu and bls_peaks.cu; this file only validates, allocates and enqueues.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "bls_internal.cuh"

using namespace bls;

struct bls_plan {
    int device = 0;
    int sm_count = 0;
    int max_smem_optin = 0;
    int max_smem_sm = 0;
    int64_t nf = 0;
    int nb = 0, kmin = 0, kmax = 0, max_top_k = 0;
    int peak_min_sep = 0;           // grid steps between reported peaks (bls_plan_set_peak_min_sep; 0 = plain R14)
    uint32_t flags = 0;
    double fmax = 0.0;
    int64_t scratch_budget = 0;

    double *d_freqs = nullptr;

    // grow-on-demand buffers
    PointRec *d_pts = nullptr;      int64_t cap_pts = 0;
    CurveMeta *d_meta = nullptr;    int64_t cap_curves = 0;
    int64_t *d_offsets = nullptr;
    int64_t *d_poffsets = nullptr;  // offsets of the prepared records (each curve padded to a multiple of 4)
    int64_t *h_poffsets = nullptr;  int64_t cap_hpoff = 0;   // host staging of those
    double *d_origin = nullptr;
    PeakCand *d_cand = nullptr;
    float *d_sr = nullptr;          int64_t cap_entries = 0; // (sr, ak, depth) entries the spectrum scratch holds
    uint32_t *d_ak = nullptr;
    float *d_depth = nullptr;
    unsigned long long *d_canon = nullptr;
    // staging for bls_search_host
    float *d_ht = nullptr, *d_hmag = nullptr, *d_hsig = nullptr;  int64_t cap_host_pts = 0;
    bls_peak *d_hpeaks = nullptr;   int64_t cap_host_peaks = 0;
    int32_t *d_hstatus = nullptr;   int64_t cap_host_status = 0;

    double2 *d_sr_stats = nullptr;  // [cap_curves] mean and sd of each curve's spectrum (reading S1)
    double *d_flo = nullptr, *d_fstep = nullptr;  int64_t cap_refine = 0;   // [n_curves * k] fine grids of bls_refine
    int64_t last_max_n = 0;
    int64_t last_n_curves = -1;
    bool last_has_origin = false;
    int64_t last_launches = 0;
    int64_t last_search_ctas = 0;
    int last_tiles_per_item = 0;
    int last_kernel = 0;
    int last_ws_shape = 0;
    cudaStream_t last_stream = nullptr;
    std::vector<cudaEvent_t> ev;    // event pairs bracketing each search launch of the last run
    size_t ev_used = 0;
    int64_t bytes_owned = 0;
    char cuda_err[256] = {0};
};

namespace {

int fail_cuda(bls_plan *p, cudaError_t e, const char *where)
{
    if (p) snprintf(p->cuda_err, sizeof(p->cuda_err), "%s: %s", where, cudaGetErrorString(e));
    cudaGetLastError();  // clear the sticky-less error state
    return BLS_ERR_CUDA;
}

#define BLS_CUDA(p, call)                                         \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return fail_cuda((p), e__, #call); \
    } while (0)

template <typename T>
int grow(bls_plan *p, T *&ptr, int64_t &cap, int64_t need, bool sync_first, cudaStream_t st)
{
    if (need <= cap && ptr) return BLS_OK;
    if (need < 1) need = 1;
    if (ptr) {
        if (sync_first) BLS_CUDA(p, cudaStreamSynchronize(st));
        BLS_CUDA(p, cudaFree(ptr));
        p->bytes_owned -= cap * (int64_t)sizeof(T);
        ptr = nullptr; cap = 0;
    }
    BLS_CUDA(p, cudaMalloc(&ptr, (size_t)need * sizeof(T)));
    cap = need;
    p->bytes_owned += need * (int64_t)sizeof(T);
    return BLS_OK;
}

template <typename T>
void release(T *&ptr)
{
    if (ptr) cudaFree(ptr);
    ptr = nullptr;
}


// Launch geometry of the search kernels for `nf` frequencies per curve, curves of at most max_n points,
// `chunk` curves per launch: which kernel, its CTA shape, shared memory and work items.  Fills every
// field of `a` that does not depend on the caller's output buffers.
struct SearchLaunch {
    SearchArgs a;
    size_t smem;
    int64_t items;
    int tiles_per_item, kernel, ws_shape;   // launch facts: bls_run stores them for BLS_QUERY_*, bls_refine does not
};

int search_launch_setup(bls_plan *p, int64_t nf, int64_t max_n, int64_t chunk, SearchLaunch &L)
{
    SearchArgs &a = L.a;
    size_t &smem_out = L.smem;
    const int ntiles = (int)((nf + kTileFreqs - 1) / kTileFreqs);
    const size_t optin = (size_t)p->max_smem_optin;
    const size_t sm_smem = (size_t)p->max_smem_sm;
    const int warps_flag = (int)((p->flags >> 8) & 0xffu);
    const int fold_flag = (int)((p->flags >> 16) & 0xffu);
    const int merge_flag = (int)((p->flags >> 24) & 7u);
    const int shape_flag = (int)((p->flags >> 4) & 7u);
    // Kernel 2 (warp-specialised, two bin buffers) whenever its buffers fit shared memory, with the
    // curve staged in shared memory if that fits too; otherwise kernel 1 (one buffer, two CTAs per SM).
    // Kernel 2 launch shape (WsShape in bls_search.cu): 0 = 20 warps at equal registers with a run-time split (what
    // the WARPS / FOLD_WARPS tuning flags address), the fold warps also merge; 1 = 8 search + 4 merge + 16 fold warps,
    // 2 = 12 search + 4 merge + 12 fold, registers moved to the search warps with setmaxnreg.  Measured (clocks per
    // pair, shapes 0 / 1 / 2): C1 651 / 597 / 568, C2 725 / 652 / 640, C3 1762 / 1620 / does not fit.  So shape 2
    // wherever its candidate arrays fit shared memory beside the bins, else shape 1, else shape 0.
    int ws_shape = 2;
    if (shape_flag >= 1 && shape_flag <= kWsShapes) ws_shape = shape_flag - 1;
    if (warps_flag || fold_flag) ws_shape = 0;
    int ws_search = kWsSearchWarps, ws_fold = 0;
    auto shape_warps = [&](int shape) {
        ws_search = kWsSearchWarps;
        if (warps_flag >= 1 && warps_flag <= kWsMaxWarps - 1) ws_search = warps_flag;
        ws_fold = kWsMaxWarps - ws_search;
        if (fold_flag >= 1 && fold_flag < ws_fold) ws_fold = fold_flag;
        if (shape > 0) {
            const int total = ws_shape_warps(shape, &ws_search);
            ws_fold = total - ws_search;
        }
    };
    {   // first the shapes that still leave room for the staged curve, then those that fit without it
        const int first = ws_shape;
        int pick = -1;
        for (int with_pts = 1; with_pts >= 0 && pick < 0; --with_pts)
            for (int sh = first; sh >= 0 && pick < 0; --sh) {
                shape_warps(sh);
                if (search_smem_bytes(p->nb, p->kmax, ws_search, 2, with_pts ? max_n : 0) <= optin) pick = sh;
            }
        ws_shape = pick < 0 ? 0 : pick;
        shape_warps(ws_shape);
    }
    const bool ws = !(p->flags & BLS_FLAG_SINGLE_BUFFER) &&
                    search_smem_bytes(p->nb, p->kmax, ws_search, 2, 0) <= optin;
    int k1_warps = kMaxSearchWarps;
    if (warps_flag >= 1 && warps_flag <= kMaxSearchWarps) k1_warps = warps_flag;
    const int warps = ws ? ws_search : k1_warps;            // warps that walk the boxes
    const int buffers = ws ? 2 : 1;
    int pts_in_smem = 1;
    size_t smem = search_smem_bytes(p->nb, p->kmax, warps, buffers, max_n);
    if (smem > optin) {                            // curve too long to stage: read it through L1/L2
        pts_in_smem = 0;
        smem = search_smem_bytes(p->nb, p->kmax, warps, buffers, 0);
    }
    if (smem > optin) return BLS_ERR_UNSUPPORTED;
    int threads = (ws ? ws_search + ws_fold : k1_warps) * 32;
    int kernel = ws ? 2 : 1;
    int nrows = search_rows_for(p->nb, p->kmax, 2 * warps);
    // Small shapes (C4: 200 epochs, 64 bins): a tile is too little work to pay for the hand-offs of kernel 2
    // and one CTA of 20 warps cannot hide its phases' latencies.  When CTAs of kSmallWarps warps (bins, candidates
    // and the staged curve) fit kSmallCtasMin times on an SM, run kernel 1 with that CTA shape: many small
    // CTAs in different phases overlap the LSU-bound fold of one with the XU-bound search of another.
    // (Kernel 3, one warp per tile with warp-private bins, measured slower: BLS_FLAG_WARP_PER_TILE selects it.)
    const size_t small_smem = search_smem_bytes(p->nb, p->kmax, kSmallWarps, 1, max_n);
    const bool small = !(p->flags & (BLS_FLAG_SINGLE_BUFFER | BLS_FLAG_NO_SMALL_CTAS)) && warps_flag == 0 &&
                       (size_t)kSmallCtasMin * (small_smem + 1024) <= sm_smem;
    if (small) {
        kernel = 1; smem = small_smem; pts_in_smem = 1; threads = kSmallWarps * 32;
        nrows = search_rows_for(p->nb, p->kmax, 2 * kSmallWarps);
    }
    const int wt_rows = search_rows_for(p->nb, p->kmax, 2);
    const size_t wt_smem = (size_t)kWtWarps * ((size_t)wt_rows * kTileFreqs * 8 + 256) + (size_t)max_n * sizeof(PointRec);
    if ((p->flags & BLS_FLAG_WARP_PER_TILE) && 2 * (wt_smem + 1024) <= sm_smem) {
        kernel = 3; smem = wt_smem; pts_in_smem = 1; threads = kWtWarps * 32; nrows = wt_rows;
    }
    int ctas_per_sm = (int)(sm_smem / (smem + 1024));
    if (ctas_per_sm < 1) ctas_per_sm = 1;
    // register-limited residency: kernels 1 and 3 are compiled for 96 registers, kernel 2 for one CTA per SM
    int max_ctas = kernel == 2 ? 1 : (int)(65536 / (96 * threads));
    if (kernel == 3) max_ctas = 2;
    if (max_ctas > 32) max_ctas = 32;
    if (ctas_per_sm > max_ctas) ctas_per_sm = max_ctas;
    const int waves = (kernel == 1 && !small) ? 12 : 24;            // enough waves to hide the tail
    const int64_t target_ctas = (int64_t)p->sm_count * ctas_per_sm * waves;
    int64_t items = (target_ctas + chunk - 1) / chunk;
    if (items < 1) items = 1;
    if (items > ntiles) items = ntiles;
    {   // where the last wave of CTAs would be mostly empty (equal curves: C3 at 24.1 waves lost 3.5 % to a 25th),
        // take a few more items per curve: the first count that loses less than 1 %, else the fullest
        const double per_wave = (double)p->sm_count * ctas_per_sm;
        auto tail_loss = [&](int64_t it) {
            const double w = (double)chunk * (double)it / per_wave, full = ceil(w - 1e-9);
            return full > 0.0 ? (full - w) / full : 0.0;
        };
        if (tail_loss(items) > 0.015) {
            double best_loss = tail_loss(items);
            int64_t best = items;
            for (int64_t it = items + 1; it < items + 8 && it <= ntiles; ++it) {
                const double loss = tail_loss(it);
                if (loss < best_loss) { best_loss = loss; best = it; }
                if (loss < 0.01) break;
            }
            items = best;
        }
    }
    int tiles_per_item = (int)((ntiles + items - 1) / items);
    items = (ntiles + tiles_per_item - 1) / tiles_per_item;
    L.tiles_per_item = tiles_per_item;
    L.kernel = kernel;
    L.ws_shape = kernel == 2 ? ws_shape : -1;

    a.pts = p->d_pts; a.offsets = p->d_offsets; a.poffsets = p->d_poffsets; a.meta = p->d_meta; a.freqs = p->d_freqs;
    a.nf = (int)nf; a.nb = p->nb; a.kmin = p->kmin; a.kmax = p->kmax;
    a.tiles_per_item = tiles_per_item; a.items_per_curve = (int)items;
    a.pts_in_smem = pts_in_smem;
    a.nrows = nrows;
    // long curves (and curves read through L1) want more loads in flight per fold warp; short ones fewer,
    // so the bursts of LDS/ATOMS do not delay the search warps (clocks per pair with 4 / 8 points in flight:
    // C1 643 / 649, C2 759 / 730, C3 2100 / 1778; 16 in flight is slower everywhere)
    a.fold_depth = (!pts_in_smem || max_n >= 2048) ? 2 : 1;
    if (p->flags & BLS_FLAG_FOLD_DEPTH(3)) a.fold_depth = (p->flags & BLS_FLAG_FOLD_DEPTH(2)) ? 2 : 1;
    a.search_warps = kernel == 2 ? ws_search : 0;
    // the exact merge re-walks ONE start per column (kmax rows): its widths are split over a few warps
    a.merge_warps = kernel == 2 ? 4 : (small ? kSmallWarps : 4);      // (kernel 2 shapes 1, 2: the four merge-role warps)
    if (merge_flag >= 1 && merge_flag <= kMergeWarps) a.merge_warps = merge_flag;
    a.kernel = kernel;
    a.ws_shape = kernel == 2 ? ws_shape : 0;
    a.threads = threads;
    a.force_canonical = (p->flags & BLS_FLAG_CANONICAL_PHASE) ? 1 : 0;
    a.sr = p->d_sr; a.ak = p->d_ak; a.depth = p->d_depth;
    a.u_sr = nullptr; a.u_start = nullptr; a.u_width = nullptr; a.u_depth = nullptr;
    a.f_lo = nullptr; a.f_step = nullptr; a.refine_k = 0; a.n_fine = 0; a.n_shift = 0;
    a.canon_count = p->d_canon;
    a.field_curves = 0;

    smem_out = smem;
    L.items = items;
    return BLS_OK;
}

// the plan-owned spectrum scratch (sr, ak, depth), `entries` each; growing synchronises the stream
int grow_spectrum_scratch(bls_plan *p, int64_t entries, cudaStream_t st)
{
    if (entries <= p->cap_entries && p->d_sr) return BLS_OK;
    if (p->d_sr) BLS_CUDA(p, cudaStreamSynchronize(st));
    release(p->d_sr); release(p->d_ak); release(p->d_depth);
    p->bytes_owned -= p->cap_entries * 12;
    p->cap_entries = 0;
    BLS_CUDA(p, cudaMalloc(&p->d_sr, (size_t)entries * sizeof(float)));
    BLS_CUDA(p, cudaMalloc(&p->d_ak, (size_t)entries * sizeof(uint32_t)));
    BLS_CUDA(p, cudaMalloc(&p->d_depth, (size_t)entries * sizeof(float)));
    p->cap_entries = entries;
    p->bytes_owned += entries * 12;
    return BLS_OK;
}

// Enqueue a host -> device copy of a caller's HOST array so that the array has been read when this returns, whatever
// memory it lives in: cudaMemcpyAsync straight from a pinned array reads it only when the stream gets there, so the
// bytes go through a private pageable block first (a copy out of pageable memory returns once the driver holds the
// bytes in its own staging buffer), which is freed at once.
cudaError_t copy_host_array_now(void *dst, const void *src, size_t bytes, cudaStream_t st)
{
    if (bytes == 0) return cudaSuccess;
    void *tmp = malloc(bytes);
    if (!tmp) return cudaErrorMemoryAllocation;
    memcpy(tmp, src, bytes);
    const cudaError_t e = cudaMemcpyAsync(dst, tmp, bytes, cudaMemcpyHostToDevice, st);
    free(tmp);
    return e;
}

void widths_from_q(int nb, double qmin, double qmax, int *kmin, int *kmax)
{
    int lo = (int)floor(qmin * (double)nb + 1e-9);
    int hi = (int)ceil(qmax * (double)nb - 1e-9);
    if (lo < 1) lo = 1;
    if (hi > nb - 1) hi = nb - 1;
    if (hi < lo) hi = lo;
    *kmin = lo; *kmax = hi;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

const char *bls_strerror(int status)
{
    switch (status) {
        case BLS_OK: return "ok";
        case BLS_ERR_NULL: return "required pointer is NULL";
        case BLS_ERR_CONFIG: return "invalid bls_config";
        case BLS_ERR_BATCH: return "invalid bls_batch";
        case BLS_ERR_ARG: return "invalid argument";
        case BLS_ERR_CUDA: return "CUDA failure (see bls_plan_last_cuda_error)";
        case BLS_ERR_UNSUPPORTED: return "shape not supported by the kernels";
        case BLS_ERR_CAPACITY: return "batch exceeds the built-in scratch of bls_variability_noalloc (BLS_NOALLOC_MAX_STARS / BLS_NOALLOC_MAX_CELLS); use bls_variability";
        default: return "unknown status";
    }
}

const char *bls_plan_last_cuda_error(const bls_plan *plan) { return plan ? plan->cuda_err : ""; }

int bls_plan_create(const bls_config *cfg, bls_plan **out_plan)
{
    if (!cfg || !out_plan) return BLS_ERR_NULL;
    if (cfg->struct_size != (int32_t)sizeof(bls_config)) return BLS_ERR_CONFIG;
    if (cfg->n_freq < 1 || cfg->n_freq > (int64_t)1 << 27) return BLS_ERR_CONFIG;   // 2^27 trial frequencies at most
    if (cfg->n_bins < 4 || cfg->n_bins > 2048) return BLS_ERR_CONFIG;
    if (!(cfg->q_min > 0.0) || !(cfg->q_max >= cfg->q_min) || !(cfg->q_max <= 0.5)) return BLS_ERR_CONFIG;
    if (cfg->max_top_k < 1 || cfg->max_top_k > 32) return BLS_ERR_CONFIG;
    if (cfg->scratch_bytes < 0) return BLS_ERR_CONFIG;

    struct HostGrid {                       // nothrow host copy of the grid (nothing may throw through the C ABI)
        double *v;
        explicit HostGrid(size_t n) : v((double *)malloc(n * sizeof(double))) {}
        ~HostGrid() { free(v); }
        double *data() { return v; }
    } grid((size_t)cfg->n_freq);
    if (!grid.v) return BLS_ERR_CUDA;
    double fmax = 0.0;
    for (int64_t k = 0; k < cfg->n_freq; ++k) {
        double f = cfg->freqs ? cfg->freqs[k] : cfg->f0 + (double)k * cfg->df;
        if (!isfinite(f) || !(f > 0.0)) return BLS_ERR_CONFIG;
        grid.v[k] = f;
        if (f > fmax) fmax = f;
    }

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) {
        cudaGetLastError();
        return BLS_ERR_CUDA;   // no CPU fallback
    }
    bls_plan *p = new (std::nothrow) bls_plan();
    if (!p) return BLS_ERR_CUDA;
    p->device = cfg->device;
    p->nf = cfg->n_freq;
    p->nb = cfg->n_bins;
    p->max_top_k = cfg->max_top_k;
    p->flags = cfg->flags;
    p->fmax = fmax;
    p->scratch_budget = cfg->scratch_bytes > 0 ? cfg->scratch_bytes : (int64_t)2 << 30;
    widths_from_q(p->nb, cfg->q_min, cfg->q_max, &p->kmin, &p->kmax);

    cudaError_t e = cudaSetDevice(p->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, p->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->max_smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, p->device);
    if (e == cudaSuccess) e = search_configure(p->max_smem_optin);
    if (e == cudaSuccess) e = cudaMalloc(&p->d_freqs, (size_t)p->nf * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(p->d_freqs, grid.data(), (size_t)p->nf * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&p->d_canon, sizeof(unsigned long long));
    if (e != cudaSuccess) {
        cudaGetLastError();
        release(p->d_freqs); release(p->d_canon);
        delete p;
        return BLS_ERR_CUDA;
    }
    p->bytes_owned = p->nf * (int64_t)sizeof(double) + 8;
    if (search_smem_bytes(p->nb, p->kmax, kMaxSearchWarps, 1, 0) > (size_t)p->max_smem_optin) {   // the bins alone must fit
        release(p->d_freqs); release(p->d_canon);
        delete p;
        return BLS_ERR_UNSUPPORTED;
    }
    *out_plan = p;
    return BLS_OK;
}

int bls_plan_destroy(bls_plan *p)
{
    if (!p) return BLS_OK;
    cudaSetDevice(p->device);
    release(p->d_freqs); release(p->d_pts); release(p->d_meta); release(p->d_offsets); release(p->d_poffsets);
    free(p->h_poffsets);
    release(p->d_origin); release(p->d_cand); release(p->d_sr); release(p->d_ak); release(p->d_depth);
    release(p->d_canon); release(p->d_ht); release(p->d_hmag); release(p->d_hsig);
    release(p->d_hpeaks); release(p->d_hstatus); release(p->d_sr_stats); release(p->d_flo); release(p->d_fstep);
    for (cudaEvent_t e : p->ev) cudaEventDestroy(e);
    delete p;
    return BLS_OK;
}

int bls_plan_query(const bls_plan *p, int32_t what, int64_t *value)
{
    if (!p || !value) return BLS_ERR_NULL;
    switch (what) {
        case BLS_QUERY_KMIN: *value = p->kmin; break;
        case BLS_QUERY_KMAX: *value = p->kmax; break;
        case BLS_QUERY_NBINS: *value = p->nb; break;
        case BLS_QUERY_NFREQ: *value = p->nf; break;
        case BLS_QUERY_SCRATCH_BYTES: *value = p->bytes_owned; break;
        case BLS_QUERY_LAST_LAUNCHES: *value = p->last_launches; break;
        case BLS_QUERY_TILE_FREQS: *value = (int64_t)p->last_tiles_per_item * kTileFreqs; break;
        case BLS_QUERY_SEARCH_CTAS: *value = p->last_search_ctas; break;
        case BLS_QUERY_SEARCH_KERNEL: *value = p->last_kernel; break;
        case BLS_QUERY_WS_SHAPE: *value = p->last_ws_shape; break;
        case BLS_QUERY_LAST_SEARCH_LAUNCHES: *value = (int64_t)(p->ev_used / 2); break;
        case BLS_QUERY_LAST_SEARCH_NS: {
            if (p->last_n_curves < 0) return BLS_ERR_ARG;
            if (cudaSetDevice(p->device) != cudaSuccess) return BLS_ERR_CUDA;
            double ns = 0.0;
            for (size_t i = 0; i + 1 < p->ev_used; i += 2) {
                float ms = 0.f;
                if (cudaEventSynchronize(p->ev[i + 1]) != cudaSuccess) return BLS_ERR_CUDA;
                if (cudaEventElapsedTime(&ms, p->ev[i], p->ev[i + 1]) != cudaSuccess) return BLS_ERR_CUDA;
                ns += (double)ms * 1e6;
            }
            *value = (int64_t)ns;
            break;
        }
        case BLS_QUERY_LAST_CANONICAL: {
            if (p->last_n_curves < 0) return BLS_ERR_ARG;
            unsigned long long v = 0;
            if (cudaSetDevice(p->device) != cudaSuccess) return BLS_ERR_CUDA;
            if (cudaStreamSynchronize(p->last_stream) != cudaSuccess) return BLS_ERR_CUDA;
            if (cudaMemcpy(&v, p->d_canon, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) return BLS_ERR_CUDA;
            *value = (int64_t)v;
            break;
        }
        default: return BLS_ERR_ARG;
    }
    return BLS_OK;
}

#pragma GCC visibility pop
}  // extern "C"

namespace {

// bls_run and bls_run_field.  field_epochs == 0: CSR batch `b`.  field_epochs > 0: b->offsets is NULL, every one
// of the b->n_curves stars has field_epochs entries (b->t shared, b->mag / b->sigma row-major) and b->t_origin
// points to ONE value.
int run_impl(bls_plan *p, const bls_batch *b, int64_t field_epochs, const bls_outputs *out, void *cuda_stream)
{
    const bool field = field_epochs > 0;
    const int64_t nc = b->n_curves;
    // Host staging owned by the plan, three arrays of nc + 1 entries: [prepared offsets | the caller's offsets | the
    // caller's origins].  The caller's HOST arrays are copied here before anything is enqueued, so they are "read
    // before the call returns" (bls.h) even when they live in pinned memory, where cudaMemcpyAsync straight from the
    // caller's pointer would read them only when the stream gets there.  This block is ordinary pageable memory: a
    // cudaMemcpyAsync from it returns once its contents are in the driver's own staging buffer, so the next run may
    // overwrite it.
    if (nc + 1 > p->cap_hpoff) {
        free(p->h_poffsets);
        p->h_poffsets = (int64_t *)malloc((size_t)(nc + 1) * 3 * sizeof(int64_t));
        p->cap_hpoff = p->h_poffsets ? nc + 1 : 0;
        if (!p->h_poffsets) return BLS_ERR_CUDA;
    }
    int64_t *const h_offsets = p->h_poffsets + p->cap_hpoff;
    double *const h_origin = (double *)(p->h_poffsets + 2 * p->cap_hpoff);
    if (!field) memcpy(h_offsets, b->offsets, (size_t)(nc + 1) * sizeof(int64_t));
    if (b->t_origin)
        for (int64_t c = 0; c < nc; ++c) h_origin[c] = field ? b->t_origin[0] : b->t_origin[c];
    int64_t max_n = 0, nrec = 0;
    for (int64_t c = 0; c < nc; ++c) {
        const int64_t n = field ? field_epochs : h_offsets[c + 1] - h_offsets[c];
        if (n < 0 || n > 2147483647LL / 64) return BLS_ERR_BATCH;
        if (n > max_n) max_n = n;
        p->h_poffsets[c] = nrec;
        nrec += (n + 3) & ~(int64_t)3;
    }
    p->h_poffsets[nc] = nrec;
    max_n = (max_n + 3) & ~(int64_t)3;                      // records per curve, padded
    const int64_t npts = field ? nc * field_epochs : h_offsets[nc];
    if (npts > 0 && (!b->t || !b->mag || !b->sigma)) return BLS_ERR_NULL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    BLS_CUDA(p, cudaSetDevice(p->device));
    p->last_n_curves = -1;
    p->last_launches = 0;
    p->last_stream = st;
    if (nc == 0) { p->last_n_curves = 0; return BLS_OK; }

    // ---- scratch (grows on demand; growing synchronises the stream) -----------------------------
    int rc;
    {
        if (nc > p->cap_curves || !p->d_meta) {
            if (p->d_meta) BLS_CUDA(p, cudaStreamSynchronize(st));
            release(p->d_meta); release(p->d_offsets); release(p->d_poffsets); release(p->d_origin); release(p->d_cand);
            release(p->d_sr_stats);
            p->bytes_owned -= p->cap_curves * (int64_t)(sizeof(CurveMeta) + 40 + sizeof(PeakCand) * p->max_top_k);
            p->cap_curves = 0;
            BLS_CUDA(p, cudaMalloc(&p->d_meta, (size_t)nc * sizeof(CurveMeta)));
            BLS_CUDA(p, cudaMalloc(&p->d_offsets, (size_t)(nc + 1) * sizeof(int64_t)));
            BLS_CUDA(p, cudaMalloc(&p->d_poffsets, (size_t)(nc + 1) * sizeof(int64_t)));
            BLS_CUDA(p, cudaMalloc(&p->d_origin, (size_t)nc * sizeof(double)));
            BLS_CUDA(p, cudaMalloc(&p->d_cand, (size_t)nc * p->max_top_k * sizeof(PeakCand)));
            BLS_CUDA(p, cudaMalloc(&p->d_sr_stats, (size_t)nc * sizeof(double2)));
            p->cap_curves = nc;
            p->bytes_owned += nc * (int64_t)(sizeof(CurveMeta) + 40 + sizeof(PeakCand) * p->max_top_k);
        }
    }
    if ((rc = grow(p, p->d_pts, p->cap_pts, nrec, true, st)) != BLS_OK) return rc;

    const int64_t per_curve = p->nf * 12;                       // sr + ak + depth
    int64_t chunk = p->scratch_budget / per_curve;
    if (chunk < 1) chunk = 1;
    if (chunk > nc) chunk = nc;
    if ((rc = grow_spectrum_scratch(p, chunk * p->nf, st)) != BLS_OK) return rc;

    // ---- metadata to the device, from the plan's staging block -----------------------------------
    if (!field)
        BLS_CUDA(p, cudaMemcpyAsync(p->d_offsets, h_offsets, (size_t)(nc + 1) * sizeof(int64_t),
                                    cudaMemcpyHostToDevice, st));
    BLS_CUDA(p, cudaMemcpyAsync(p->d_poffsets, p->h_poffsets, (size_t)(nc + 1) * sizeof(int64_t),
                                cudaMemcpyHostToDevice, st));
    p->last_has_origin = b->t_origin != nullptr;
    if (b->t_origin)                            // (a field's one origin was replicated per star above)
        BLS_CUDA(p, cudaMemcpyAsync(p->d_origin, h_origin, (size_t)nc * sizeof(double), cudaMemcpyHostToDevice, st));
    BLS_CUDA(p, cudaMemsetAsync(p->d_canon, 0, sizeof(unsigned long long), st));

    // ---- a0 prep -------------------------------------------------------------------------------
    BLS_CUDA(p, launch_prep(b->t, b->mag, b->sigma, p->d_offsets, p->d_poffsets, nc, field_epochs, p->fmax, p->d_pts,
                            p->d_meta, out ? out->status : nullptr, st));
    p->last_launches += 1;

    // ---- launch geometry of the search ---------------------------------------------------------
    SearchLaunch L;
    if ((rc = search_launch_setup(p, p->nf, max_n, chunk, L)) != BLS_OK) return rc;
    SearchArgs &a = L.a;
    a.u_sr = out ? out->sr : nullptr;
    a.u_start = out ? out->best_start : nullptr;
    a.u_width = out ? out->best_width : nullptr;
    a.u_depth = out ? out->depth : nullptr;
    int64_t units = chunk;                                       // CTAs of a launch = units x items
    if (field && !(p->flags & (BLS_FLAG_NO_FIELD_KERNEL | BLS_FLAG_SINGLE_BUFFER | BLS_FLAG_WARP_PER_TILE |
                               BLS_FLAG_WS_SHAPE(7) | BLS_FLAG_FOLD_WARPS(0xff) | BLS_FLAG_WARPS(0xff) | BLS_FLAG_MERGE_WARPS(7)))) {
        // f2: the field kernel (kernel 4) where its kFieldStars bin buffers and the field's records fit an SM at least
        // twice; same work-item sizing as search_launch_setup, over groups of stars instead of stars
        const int fw = kFieldWarps;                              // one pair of warps per star
        const size_t fsmem = field_smem_bytes(p->nb, p->kmax, fw, max_n);
        if (2 * (fsmem + 1024) <= (size_t)p->max_smem_sm && fsmem <= (size_t)p->max_smem_optin) {
            int ctas_per_sm = (int)((size_t)p->max_smem_sm / (fsmem + 1024));
            const int reg_ctas = 65536 / (96 * fw * 32);
            if (ctas_per_sm > reg_ctas) ctas_per_sm = reg_ctas;
            if (ctas_per_sm > 32) ctas_per_sm = 32;
            units = (chunk + kFieldStars - 1) / kFieldStars;
            const int ntiles = (int)((p->nf + kTileFreqs - 1) / kTileFreqs);
            int64_t it = ((int64_t)p->sm_count * ctas_per_sm * 24 + units - 1) / units;
            if (it < 1) it = 1;
            if (it > ntiles) it = ntiles;
            const int tpi = (int)((ntiles + it - 1) / it);
            L.items = (ntiles + tpi - 1) / tpi;
            L.smem = fsmem;
            L.tiles_per_item = tpi; L.kernel = 4; L.ws_shape = -1;
            a.kernel = 4; a.threads = fw * 32; a.pts_in_smem = 1; a.tiles_per_item = tpi; a.items_per_curve = (int)L.items;
            a.nrows = search_rows_for(p->nb, p->kmax, 0);
            a.merge_warps = 2;
        }
    }
    p->last_max_n = max_n;
    p->last_tiles_per_item = L.tiles_per_item;
    p->last_kernel = L.kernel;
    p->last_ws_shape = L.ws_shape;

    // ---- per chunk of curves: search -> peak candidates ------------------------------------------
    p->last_search_ctas = 0;
    p->ev_used = 0;
    for (int64_t base = 0; base < nc; base += chunk) {
        const int64_t cc = (nc - base < chunk) ? nc - base : chunk;
        a.curve_base = base;
        a.field_curves = cc;
        while (p->ev.size() < p->ev_used + 2) {
            cudaEvent_t e;
            BLS_CUDA(p, cudaEventCreate(&e));
            try { p->ev.push_back(e); } catch (...) { cudaEventDestroy(e); return BLS_ERR_CUDA; }
        }
        BLS_CUDA(p, cudaEventRecord(p->ev[p->ev_used], st));
        BLS_CUDA(p, launch_search(a, cc, L.smem, st));
        BLS_CUDA(p, cudaEventRecord(p->ev[p->ev_used + 1], st));
        p->ev_used += 2;
        BLS_CUDA(p, launch_peaks(p->d_sr, p->d_ak, p->d_depth, p->d_meta, base, cc, (int)p->nf,
                                 p->max_top_k, p->peak_min_sep, p->d_cand, p->d_sr_stats, st));
        p->last_launches += 2;
        p->last_search_ctas += (L.kernel == 4 ? (cc + kFieldStars - 1) / kFieldStars : cc) * L.items;
    }
    p->last_n_curves = nc;
    return BLS_OK;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

int bls_run(bls_plan *p, const bls_batch *b, const bls_outputs *out, void *cuda_stream)
{
    if (!p || !b) return BLS_ERR_NULL;
    if (b->n_curves < 0) return BLS_ERR_BATCH;
    if (!b->offsets) return BLS_ERR_NULL;
    if (b->offsets[0] != 0) return BLS_ERR_BATCH;
    return run_impl(p, b, 0, out, cuda_stream);
}

int bls_run_field(bls_plan *p, const bls_field_batch *fb, const bls_outputs *out, void *cuda_stream)
{
    if (!p || !fb) return BLS_ERR_NULL;
    if (fb->n_stars < 0 || fb->n_epochs < 1) return BLS_ERR_BATCH;
    bls_batch b;
    b.n_curves = fb->n_stars; b.offsets = nullptr; b.t = fb->t; b.mag = fb->mag; b.sigma = fb->sigma; b.t_origin = fb->t_origin;
    return run_impl(p, &b, fb->n_epochs, out, cuda_stream);
}

int bls_debug_fold_bins(int32_t device, const double *f, const double *t, int64_t n, int32_t n_bins,
                        uint32_t flags, int32_t *bins, int64_t *n_canonical)
{
    if (!f || !t || !bins) return BLS_ERR_NULL;
    if (n < 0 || n_bins < 4 || n_bins > 2048) return BLS_ERR_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    unsigned long long *d_cnt = nullptr, h_cnt = 0;
    if (cudaMalloc(&d_cnt, sizeof(h_cnt)) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaError_t e = cudaMemset(d_cnt, 0, sizeof(h_cnt));
    int sm_count = 1;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = launch_debug_bins(f, t, n, n_bins, (flags & BLS_FLAG_CANONICAL_PHASE) ? 1 : 0, bins, d_cnt, sm_count, nullptr);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(&h_cnt, d_cnt, sizeof(h_cnt), cudaMemcpyDeviceToHost);
    cudaFree(d_cnt);
    if (e != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    if (n_canonical) *n_canonical = (int64_t)h_cnt;
    return BLS_OK;
}

int bls_debug_fold_bins_shift(int32_t device, const double *f, const double *t, int64_t n, int32_t n_bins, int32_t h,
                              int32_t n_shift, uint32_t flags, int32_t *bins, int64_t *n_canonical)
{
    if (!f || !t || !bins) return BLS_ERR_NULL;
    if (n < 0 || n_bins < 4 || n_bins > 2048 || n_shift < 1 || n_shift > 8 || h < 0 || h >= n_shift) return BLS_ERR_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    unsigned long long *d_cnt = nullptr, h_cnt = 0;
    if (cudaMalloc(&d_cnt, sizeof(h_cnt)) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaError_t e = cudaMemset(d_cnt, 0, sizeof(h_cnt));
    int sm_count = 1;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess)
        e = launch_debug_bins_shift(f, t, n, n_bins, h, n_shift, (flags & BLS_FLAG_CANONICAL_PHASE) ? 1 : 0, bins, d_cnt, sm_count, nullptr);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(&h_cnt, d_cnt, sizeof(h_cnt), cudaMemcpyDeviceToHost);
    cudaFree(d_cnt);
    if (e != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    if (n_canonical) *n_canonical = (int64_t)h_cnt;
    return BLS_OK;
}

int bls_variability(int32_t device, const bls_variability_config *cfg, const bls_batch *b, const int32_t *group,
                    const bls_variability_outputs *out, void *cuda_stream)
{
    if (!cfg || !b || !out) return BLS_ERR_NULL;
    if (cfg->struct_size != (int32_t)sizeof(bls_variability_config)) return BLS_ERR_CONFIG;
    if (cfg->n_groups < 1 || cfg->n_mag_bins < 1 || (int64_t)cfg->n_groups * cfg->n_mag_bins > (1 << 24)) return BLS_ERR_CONFIG;
    if (!(cfg->mag_bin > 0.0) || !isfinite(cfg->mag_lo) || !(cfg->clip > 0.0) || !isfinite(cfg->nsig)) return BLS_ERR_CONFIG;
    if (cfg->max_iter < 0 || cfg->max_iter > 100 || cfg->min_members < 0) return BLS_ERR_CONFIG;
    if (b->n_curves < 0) return BLS_ERR_BATCH;
    if (!b->offsets) return BLS_ERR_NULL;
    const int64_t nc = b->n_curves;
    if (b->offsets[0] != 0) return BLS_ERR_BATCH;
    for (int64_t c = 0; c < nc; ++c)
        if (b->offsets[c + 1] < b->offsets[c]) return BLS_ERR_BATCH;
    if (b->offsets[nc] > 0 && (!b->t || !b->mag || !b->sigma)) return BLS_ERR_NULL;
    if (nc == 0) return BLS_OK;
    if (nc > 2147483647LL) return BLS_ERR_BATCH;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int64_t n_cells = (int64_t)cfg->n_groups * cfg->n_mag_bins;
    // one stream-ordered scratch block: offsets | status | cell | members | count | offset | cursor | mean | rms | keep
    size_t off = 0;
    auto take = [&off](size_t bytes) { const size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
    const size_t o_offsets = take((size_t)(nc + 1) * 8), o_status = take((size_t)nc * 4), o_cell = take((size_t)nc * 4);
    const size_t o_members = take((size_t)nc * 4), o_count = take((size_t)n_cells * 4), o_offset = take((size_t)(n_cells + 1) * 4);
    const size_t o_cursor = take((size_t)n_cells * 4), o_mean = take((size_t)nc * 8), o_rms = take((size_t)nc * 8);
    const size_t o_keep = take((size_t)nc);
    unsigned char *scr = nullptr;
    if (cudaMallocAsync((void **)&scr, off, st) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaError_t e = copy_host_array_now(scr + o_offsets, b->offsets, (size_t)(nc + 1) * 8, st);
    int32_t *status = out->status ? out->status : (int32_t *)(scr + o_status);
    int32_t *cell = out->cell ? out->cell : (int32_t *)(scr + o_cell);
    double *mean_mag = out->mean_mag ? out->mean_mag : (double *)(scr + o_mean);
    double *rms = out->rms ? out->rms : (double *)(scr + o_rms);
    if (e == cudaSuccess)
        e = launch_variability(b->t, b->mag, b->sigma, (const int64_t *)(scr + o_offsets), group, nc, *cfg, status, mean_mag,
                               rms, cell, (int32_t *)(scr + o_count), (int32_t *)(scr + o_offset), (int32_t *)(scr + o_cursor),
                               (int32_t *)(scr + o_members), scr + o_keep, out->expected, out->scatter, out->kept, out->flag, st);
    const cudaError_t e2 = cudaFreeAsync(scr, st);
    if (e != cudaSuccess || e2 != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    return BLS_OK;
}

int bls_detection_efficiency(int32_t device, const bls_batch *b, int64_t n_freq, const double *freqs, double duration,
                             int32_t n_phase, int32_t min_events, int32_t *count, double *efficiency, void *cuda_stream)
{
    if (!b || !freqs) return BLS_ERR_NULL;
    if (b->n_curves < 0 || b->n_curves > 65535) return BLS_ERR_BATCH;
    if (!b->offsets) return BLS_ERR_NULL;
    if (n_freq < 1 || n_freq > 2147483647LL || !(duration > 0.0) || !isfinite(duration)) return BLS_ERR_ARG;
    if (n_phase < 1 || n_phase > (1 << 20) || min_events < 1) return BLS_ERR_ARG;
    const int64_t nc = b->n_curves;
    if (b->offsets[0] != 0) return BLS_ERR_BATCH;
    for (int64_t c = 0; c < nc; ++c)
        if (b->offsets[c + 1] < b->offsets[c]) return BLS_ERR_BATCH;
    for (int64_t q = 0; q < n_freq; ++q)
        if (!isfinite(freqs[q]) || !(freqs[q] > 0.0)) return BLS_ERR_ARG;
    if (b->offsets[nc] > 0 && !b->t) return BLS_ERR_NULL;
    if (nc == 0) return BLS_OK;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    size_t off = 0;
    auto take = [&off](size_t bytes) { const size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
    const size_t o_off = take((size_t)(nc + 1) * 8), o_f = take((size_t)n_freq * 8);
    // the kernel writes both results; the one the caller does not want goes to scratch (none if both are wanted)
    const size_t o_cnt = count ? 0 : take((size_t)(nc * n_freq) * 4), o_eff = efficiency ? 0 : take((size_t)(nc * n_freq) * 8);
    unsigned char *scr = nullptr;
    if (cudaMallocAsync((void **)&scr, off, st) != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    cudaError_t e = copy_host_array_now(scr + o_off, b->offsets, (size_t)(nc + 1) * 8, st);
    if (e == cudaSuccess) e = copy_host_array_now(scr + o_f, freqs, (size_t)n_freq * 8, st);
    if (e == cudaSuccess)
        e = launch_window(b->t, (const int64_t *)(scr + o_off), nc, (int)n_freq, (const double *)(scr + o_f), duration, n_phase,
                          min_events, count ? count : (int32_t *)(scr + o_cnt), efficiency ? efficiency : (double *)(scr + o_eff), st);
    const cudaError_t e2 = cudaFreeAsync(scr, st);
    if (e != cudaSuccess || e2 != cudaSuccess) { cudaGetLastError(); return BLS_ERR_CUDA; }
    return BLS_OK;
}

int bls_plan_set_peak_min_sep(bls_plan *p, int32_t steps)
{
    if (!p) return BLS_ERR_NULL;
    if (steps < 0 || steps > (1 << 27)) return BLS_ERR_ARG;
    p->peak_min_sep = steps;
    return BLS_OK;
}

int bls_topk(bls_plan *p, int32_t k, bls_peak *peaks, void *cuda_stream)
{
    if (!p || !peaks) return BLS_ERR_NULL;
    if (p->last_n_curves < 0) return BLS_ERR_ARG;
    if (k < 1 || k > p->max_top_k) return BLS_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    BLS_CUDA(p, cudaSetDevice(p->device));
    BLS_CUDA(p, launch_format_peaks(p->d_cand, p->max_top_k, k, p->last_n_curves, p->nb, p->d_freqs,
                                    p->last_has_origin ? p->d_origin : nullptr, peaks, st));
    p->last_launches += 1;
    return BLS_OK;
}

int bls_refine(bls_plan *p, int32_t k, int32_t n_fine, int32_t n_shift, bls_refined_peak *out, void *cuda_stream)
{
    if (!p || !out) return BLS_ERR_NULL;
    if (p->last_n_curves < 0) return BLS_ERR_ARG;
    if (k < 1 || k > p->max_top_k) return BLS_ERR_ARG;
    if (n_fine < 1 || n_fine > 256 || n_shift < 1 || n_shift > 8) return BLS_ERR_ARG;
    const int64_t nc = p->last_n_curves;
    if (nc == 0) return BLS_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    BLS_CUDA(p, cudaSetDevice(p->device));
    int rc;
    if (nc * k > p->cap_refine || !p->d_flo) {
        if (p->d_flo) BLS_CUDA(p, cudaStreamSynchronize(st));
        release(p->d_flo); release(p->d_fstep);
        p->bytes_owned -= p->cap_refine * 16;
        p->cap_refine = 0;
        BLS_CUDA(p, cudaMalloc(&p->d_flo, (size_t)(nc * k) * sizeof(double)));
        BLS_CUDA(p, cudaMalloc(&p->d_fstep, (size_t)(nc * k) * sizeof(double)));
        p->cap_refine = nc * k;
        p->bytes_owned += nc * k * 16;
    }
    // the fine spectrum of a chunk of curves reuses the spectrum scratch of bls_run: [chunk][k*n_fine*n_shift]
    const int64_t nf = (int64_t)k * n_fine * n_shift;
    int64_t chunk = p->scratch_budget / (nf * 12);
    if (chunk < 1) chunk = 1;
    if (chunk > nc) chunk = nc;
    if ((rc = grow_spectrum_scratch(p, chunk * nf, st)) != BLS_OK) return rc;
    BLS_CUDA(p, launch_refine_grid(p->d_cand, p->max_top_k, k, nc, (int)p->nf, n_fine, p->d_freqs, p->d_flo, p->d_fstep, st));
    SearchLaunch L;
    if ((rc = search_launch_setup(p, nf, p->last_max_n, chunk, L)) != BLS_OK) return rc;
    SearchArgs &a = L.a;
    a.f_lo = p->d_flo; a.f_step = p->d_fstep; a.refine_k = k; a.n_fine = n_fine; a.n_shift = n_shift;
    a.canon_count = nullptr;
    for (int64_t base = 0; base < nc; base += chunk) {
        const int64_t cc = (nc - base < chunk) ? nc - base : chunk;
        a.curve_base = base;
        BLS_CUDA(p, launch_search(a, cc, L.smem, st));
        BLS_CUDA(p, launch_refine_reduce(p->d_sr, p->d_ak, p->d_depth, p->d_cand, p->max_top_k, k, base, cc, n_fine, n_shift,
                                         p->nb, p->d_flo, p->d_fstep, p->d_sr_stats, p->last_has_origin ? p->d_origin : nullptr,
                                         out, st));
        p->last_launches += 2;
    }
    p->last_launches += 1;
    return BLS_OK;
}

int bls_search_host(bls_plan *p, const bls_batch *hb, int32_t k, bls_peak *peaks, int32_t *status)
{
    if (!p || !hb || !peaks) return BLS_ERR_NULL;
    if (hb->n_curves < 0 || !hb->offsets) return BLS_ERR_BATCH;
    if (k < 1 || k > p->max_top_k) return BLS_ERR_ARG;
    const int64_t nc = hb->n_curves;
    const int64_t npts = hb->offsets[nc];
    if (npts < 0) return BLS_ERR_BATCH;
    if (npts > 0 && (!hb->t || !hb->mag || !hb->sigma)) return BLS_ERR_NULL;
    BLS_CUDA(p, cudaSetDevice(p->device));
    cudaStream_t st = nullptr;
    int rc;
    if (npts > p->cap_host_pts || !p->d_ht) {
        release(p->d_ht); release(p->d_hmag); release(p->d_hsig);
        p->bytes_owned -= p->cap_host_pts * 12;
        p->cap_host_pts = 0;
        const int64_t need = npts > 0 ? npts : 1;
        BLS_CUDA(p, cudaMalloc(&p->d_ht, (size_t)need * 4));
        BLS_CUDA(p, cudaMalloc(&p->d_hmag, (size_t)need * 4));
        BLS_CUDA(p, cudaMalloc(&p->d_hsig, (size_t)need * 4));
        p->cap_host_pts = need;
        p->bytes_owned += need * 12;
    }
    if ((rc = grow(p, p->d_hpeaks, p->cap_host_peaks, nc * k, false, st)) != BLS_OK) return rc;
    if ((rc = grow(p, p->d_hstatus, p->cap_host_status, nc, false, st)) != BLS_OK) return rc;
    if (npts > 0) {
        BLS_CUDA(p, cudaMemcpyAsync(p->d_ht, hb->t, (size_t)npts * 4, cudaMemcpyHostToDevice, st));
        BLS_CUDA(p, cudaMemcpyAsync(p->d_hmag, hb->mag, (size_t)npts * 4, cudaMemcpyHostToDevice, st));
        BLS_CUDA(p, cudaMemcpyAsync(p->d_hsig, hb->sigma, (size_t)npts * 4, cudaMemcpyHostToDevice, st));
    }
    bls_batch db = *hb;
    db.t = p->d_ht; db.mag = p->d_hmag; db.sigma = p->d_hsig;
    bls_outputs out;
    memset(&out, 0, sizeof(out));
    out.status = p->d_hstatus;
    if ((rc = bls_run(p, &db, &out, st)) != BLS_OK) return rc;
    if (nc > 0) {
        if ((rc = bls_topk(p, k, p->d_hpeaks, st)) != BLS_OK) return rc;
        BLS_CUDA(p, cudaMemcpyAsync(peaks, p->d_hpeaks, (size_t)(nc * k) * sizeof(bls_peak),
                                    cudaMemcpyDeviceToHost, st));
        if (status)
            BLS_CUDA(p, cudaMemcpyAsync(status, p->d_hstatus, (size_t)nc * sizeof(int32_t),
                                        cudaMemcpyDeviceToHost, st));
    }
    BLS_CUDA(p, cudaStreamSynchronize(st));
    return BLS_OK;
}

#pragma GCC visibility pop
}  // extern "C"
