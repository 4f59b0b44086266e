// a0 Prep: once per curve,
//   w_i = sigma_i^-2 / sum_j sigma_j^-2,  mu = sum_i w_i m_i,  x_i = m_i - mu      (readings R4, R5)
// all sums in fp64, then the fixed-point records the search kernel folds:
//   qw_i = rint(w_i * SW),        SW = 2^32 - 2N - 2            (sum_i qw_i < 2^32 for any subset)
//   qy_i = rint(w_i x_i * SY),    SY = (2^31 - N - 2) / (0.5 sqrt(sum_i w_i x_i^2) (1 + 1e-12))
// SY is safe for ANY subset of points: the least-squares residual of a two-level fit is >= 0, so
// s^2 <= r(1-r) sum w x^2 <= sum w x^2 / 4.
// One CTA per curve, fixed 256-thread strided accumulation + fixed tree => bitwise reproducible.
#include "bls_internal.cuh"

namespace bls {

// FIELD = false: CSR batch, curve c owns points [offsets[c], offsets[c+1]) of t / mag / sigma.
// FIELD = true (f2, field-shared cadence): every star shares the epoch list t[0..n_epochs) and owns row c of
// mag / sigma [n_curves][n_epochs]; an entry whose mag or sigma is not finite or whose sigma <= 0 is an ABSENT
// epoch of that star (a flagged measurement), not a data fault: it gets a weightless record.
template <bool FIELD>
__global__ void __launch_bounds__(kPrepThreads)
prep_kernel(const float *__restrict__ t, const float *__restrict__ mag, const float *__restrict__ sigma,
            const int64_t *__restrict__ offsets, const int64_t *__restrict__ poffsets, int64_t n_epochs, double fmax_grid,
            PointRec *__restrict__ pts, CurveMeta *__restrict__ meta, int32_t *__restrict__ u_status)
{
    __shared__ double sh[kPrepThreads / 32];
    __shared__ int s_flags;
    const int64_t c = blockIdx.x;
    const int64_t beg = FIELD ? c * n_epochs : offsets[c];
    const int64_t n = FIELD ? n_epochs : offsets[c + 1] - beg;
    const int64_t tbeg = FIELD ? 0 : beg;
    const int64_t pbeg = FIELD ? c * ((n_epochs + 3) & ~(int64_t)3) : poffsets[c];
    const int64_t n_pad = (n + 3) & ~(int64_t)3;                            // records: n rounded up to a multiple of 4
    auto present = [&](int64_t i) {
        if (!FIELD) return true;
        const float mi = mag[beg + i], si = sigma[beg + i];
        return isfinite(mi) && isfinite(si) && si > 0.0f;
    };
    if (threadIdx.x == 0) s_flags = 0;
    __syncthreads();

    // pass 1: validity, sum of inverse variances, max |t|, number of present points
    double acc = 0.0, tmax = 0.0, cnt = 0.0;
    int flags = 0;
    for (int64_t i = threadIdx.x; i < n; i += kPrepThreads) {
        const float ti = t[tbeg + i], mi = mag[beg + i], si = sigma[beg + i];
        if (!isfinite(ti)) flags |= 1;
        else if (FIELD && !present(i)) continue;
        else if (!isfinite(mi) || !isfinite(si)) flags |= 1;
        else if (!(si > 0.0f)) flags |= 2;
        else {
            double s = (double)si;
            acc += 1.0 / (s * s);
            tmax = fmax(tmax, fabs((double)ti));
            cnt += 1.0;
        }
    }
    if (flags) atomicOr(&s_flags, flags);
    double sw = block_sum(acc, sh);
    tmax = block_max_d(tmax, sh);
    const double n_present = block_sum(cnt, sh);
    __syncthreads();
    int status = BLS_CURVE_OK;
    if (s_flags & 1) status = BLS_CURVE_NONFINITE;
    else if (s_flags & 2) status = BLS_CURVE_BAD_SIGMA;
    else if (n_present < 2.0) status = BLS_CURVE_TOO_FEW;
    else if (!isfinite(sw) || !(sw > 0.0)) status = BLS_CURVE_NONFINITE;
    if (!FIELD && n < 2) status = BLS_CURVE_TOO_FEW;

    if (status != BLS_CURVE_OK) {
        for (int64_t i = threadIdx.x; i < n_pad; i += kPrepThreads) {
            PointRec r; r.t = 0.0; r.qw = 0u; r.qy = 0;
            pts[pbeg + i] = r;
        }
        if (threadIdx.x == 0) {
            CurveMeta m; m.ncw = 0.f; m.cy = 0.f; m.status = status; m.force_canonical = 0;
            m.swt = 0u; m.w0 = 0u; m.y0 = 0; m.pad_ = 0; m.sr_scale = 0.0; m.dp_scale = 0.0; m.wx2 = 0.0;
            meta[c] = m;
            if (u_status) u_status[c] = status;
        }
        return;
    }

    // pass 2: weighted mean
    acc = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += kPrepThreads) {
        if (!present(i)) continue;
        double s = (double)sigma[beg + i];
        acc += ((1.0 / (s * s)) / sw) * (double)mag[beg + i];
    }
    const double mu = block_sum(acc, sh);

    // pass 3: weighted variance (bounds every box sum, sets the fixed-point scale of qy)
    acc = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += kPrepThreads) {
        if (!present(i)) continue;
        double s = (double)sigma[beg + i];
        double w = (1.0 / (s * s)) / sw;
        double x = (double)mag[beg + i] - mu;
        acc += w * x * x;
    }
    const double wx2 = block_sum(acc, sh);

    const double SW = 4294967296.0 - 2.0 * n_present - 2.0;
    const double sigw = sqrt(wx2);
    const double SY = (sigw > 0.0 && isfinite(sigw))
                          ? (2147483648.0 - n_present - 2.0) / (0.5 * sigw * (1.0 + 1e-12)) : 0.0;

    // Records.  A zero-time point (t == 0, e.g. the curve's first epoch) sits exactly on a bin edge at every
    // frequency and always belongs to bin 0: it is summed into (w0, y0) instead and its record carries no
    // weight, so the fold's guard band is not triggered by it.  Weightless records (those, absent epochs of a
    // field and the padding to a multiple of 4) take the time max|t|: they add zero to whatever bin they hit.
    double qsum = 0.0, w0 = 0.0, y0 = 0.0;              // integers < 2^32: exact in fp64, any order
    const double t_pad = tmax;                          // inside the fast phase's range, not 0 unless all are
    for (int64_t i = threadIdx.x; i < n_pad; i += kPrepThreads) {
        PointRec r;
        r.t = t_pad; r.qw = 0u; r.qy = 0;
        if (i < n && present(i)) {
            double s = (double)sigma[beg + i];
            double w = (1.0 / (s * s)) / sw;
            double x = (double)mag[beg + i] - mu;
            const uint32_t qw = (uint32_t)__double2ll_rn(w * SW);
            const int32_t qy = (int32_t)__double2ll_rn(w * x * SY);
            qsum += (double)qw;
            if (t[tbeg + i] == 0.0f) { w0 += (double)qw; y0 += (double)qy; }
            else { r.t = (double)t[tbeg + i]; r.qw = qw; r.qy = qy; }
        }
        pts[pbeg + i] = r;
    }
    const double w0s = block_sum(w0, sh), y0s = block_sum(y0, sh);
    const double swt = block_sum(qsum, sh);             // SWT = sum_i qw_i <= SW + N/2 < 2^32
    if (threadIdx.x == 0) {
        CurveMeta m;
        m.ncw = (float)(-1.0 / swt);
        m.cy = SY > 0.0 ? (float)(1.0 / SY) : 0.f;
        m.status = BLS_CURVE_OK;
        // the fast phase needs |f t| < 2^18 cycles
        m.force_canonical = (fmax_grid * tmax < 262144.0) ? 0 : 1;
        m.swt = (uint32_t)swt;
        m.w0 = (uint32_t)w0s; m.y0 = (int32_t)y0s; m.pad_ = 0;
        m.sr_scale = SY > 0.0 ? (swt / SY) * (swt / SY) : 0.0;
        m.dp_scale = SY > 0.0 ? swt * (swt / SY) : 0.0;
        m.wx2 = wx2;
        meta[c] = m;
        if (u_status) u_status[c] = BLS_CURVE_OK;
    }
}

cudaError_t launch_prep(const float *t, const float *mag, const float *sigma, const int64_t *offsets,
                        const int64_t *poffsets, int64_t n_curves, int64_t field_epochs, double fmax, PointRec *pts,
                        CurveMeta *meta, int32_t *u_status, cudaStream_t st)
{
    if (n_curves <= 0) return cudaSuccess;
    if (field_epochs > 0)
        prep_kernel<true><<<(unsigned)n_curves, kPrepThreads, 0, st>>>(t, mag, sigma, offsets, poffsets, field_epochs, fmax, pts,
                                                                      meta, u_status);
    else
        prep_kernel<false><<<(unsigned)n_curves, kPrepThreads, 0, st>>>(t, mag, sigma, offsets, poffsets, 0, fmax, pts, meta,
                                                                       u_status);
    return cudaGetLastError();
}

}  // namespace bls
