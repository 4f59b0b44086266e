// a1 Load, a2 Fold, a3/a4 box search, per-frequency argmax (DESIGN.md
// section 6.3).  PAPER.md L145: "the light curve data is read into fast shared memory by each
// thread block (with memory accesses coalesced for speed), then each thread picks an untested
// period, phases the light curve at that period and then tests a range of durations and phases."
//
// What is kept from that design: the curve is resident in shared memory across a block of trial
// frequencies, and a LANE owns a trial frequency while folding.  What differs (Fermi -> sm_100a):
//   * a CTA owns one curve and a tile of 32 consecutive frequencies at a time; the fold warps fold
//     the curve into the tile's bins (each warp takes every NW-th group of points, every lane its
//     own frequency): bins[bin][{W,Y}][lane] puts lane l in bank l -> the native 32-bit ATOMS.ADD
//     is conflict-free by construction;
//   * bins are int32 fixed point and STAY integers for the whole life of a tile: sums are exact,
//     order independent and bitwise reproducible, and the statistic reported for a box is a
//     function of the box's point set alone (exact plateaus between adjacent frequencies);
//   * the phase is one DFMA with a magic constant whose low mantissa word is frac(f t) * 2^32;
//     one IMAD.WIDE gives (bin, position inside the bin); positions inside a guard band of a bin
//     edge fall back to the canonical 3-rounding fp64 rule, so bin indices equal the oracle's
//     bit for bit (DESIGN.md "Fold / fast phase" has the error bound);
//   * the box search ranks boxes in packed fp32 (add/fma/mul.f32x2): a thread owns TWO adjacent
//     frequencies and S consecutive start bins (S up to 8 at 96 registers, up to 13 with the registers the
//     other warp roles hand over); it walks the bin rows once, converting each row (one LDS.64 per plane,
//     I2FP) as it arrives, so a row feeds 2S boxes.  Per pair of boxes: FFMA2 (n -= W/SWT), FADD2 (s += Y),
//     FFMA2 (n^2 + n = -r(1-r)), 2 MUFU.RSQ, FMUL2, and one FMNMX3 per frequency that takes the boxes of
//     two consecutive rows of the SAME start.  Running sums are direct (no prefix differences).  The
//     maximum of |s| rsqrt(r(1-r)) is kept per start; the best start of the column goes to the merge step;
//   * the merge step (lane = frequency) re-walks that ONE start in EXACT integer arithmetic (its widths
//     split over a few warps), applies the canonical tie-break (reading R12) and writes SR and depth from
//     the integer box sums (R, S) in fp64, rounded once to fp32;
//   * three warp roles run concurrently on consecutive tiles (kernel 2): fold warps (zero / fold / extend
//     tile i+1), search warps (rank the boxes of tile i), merge warps (exact merge of tile i-1); registers
//     are moved from the fold and merge warps to the search warps with setmaxnreg.
#include "bls_internal.cuh"

namespace bls {

// Box-search geometry.  The nb start bins are dealt to the searching WARPS: warp w takes the starts
// [w nb / nsw, (w+1) nb / nsw); its two half-warps take ceil(P/2) starts each, the first from the front of that
// range and the second from its back (when P is odd they share the middle start: both halves of a warp always
// walk the same sequence of start tiles, so the warp never diverges).  A half-warp walks its starts as
// n = ceil(P_h / SMAX) start tiles of S = P_h/n or P_h/n + 1 consecutive starts.  SMAX is what the registers of
// the searching warps hold (8 at 96 registers, more for the register-rebalanced shapes).
// Bin rows of a buffer: the nb bins plus the cyclic extension the widest box of the last start reaches
// (row nb + kmax - 2) and one spare row for the search's one-row-ahead load.
int search_rows_for(int nb, int kmax, int) { return nb + kmax; }

// `buffers` = 1 (search_kernel) or 2 (search_ws_kernel); `warps` = box-search warps
size_t search_smem_bytes(int nb, int kmax, int warps, int buffers, int64_t n_points_in_smem)
{
    const size_t bins = (size_t)search_rows_for(nb, kmax, 2 * warps) * kTileFreqs * 8;
    // candidates (rank, code) per buffer; merge posts: kernel 2 kMergeWarps, kernel 1 all its warps
    const size_t cand = (size_t)buffers * warps * kTileFreqs * 8 + (size_t)(buffers == 2 ? kMergeWarps : warps) * kTileFreqs * 8 +
                        (buffers == 2 ? 16 : 0);                  // kernel 2: two mbarriers
    return (size_t)buffers * bins + cand + (size_t)n_points_in_smem * sizeof(PointRec);
}

__device__ __noinline__ int canonical_bin(double f, double t, int nb, double shift)
{
    double p = __dsub_rn(__dmul_rn(f, t), shift);        // shift = 0 (the plain rule R8) subtracts exactly nothing
    double phi = __dsub_rn(p, floor(p));
    double xb = __dmul_rn(phi, (double)nb);
    int b = (int)xb;
    return b >= nb ? nb - 1 : b;
}

__device__ __forceinline__ float fast_rsqrt(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <bool SMEM>
__device__ __forceinline__ PointRec load_point(const PointRec *p)
{
    PointRec r;
    // one 16-byte access at a warp-uniform address: LDS.128 broadcast (or LDG.128 through L1)
    const uint4 raw = SMEM ? *reinterpret_cast<const uint4 *>(p) : __ldg(reinterpret_cast<const uint4 *>(p));
    r.t = __hiloint2double((int)raw.y, (int)raw.x); r.qw = raw.z; r.qy = (int32_t)raw.w;
    return r;
}

// ---- packed fp32 pairs (sm_100a add/mul/fma.f32x2: one issue slot, two results) ---------------------
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b)
{
    uint64_t c;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(c) : "l"(a), "l"(b));
    return c;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b)
{
    uint64_t c;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(c) : "l"(a), "l"(b));
    return c;
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t d)
{
    uint64_t c;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(c) : "l"(a), "l"(b), "l"(d));
    return c;
}
__device__ __forceinline__ void unpack2(uint64_t v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t pack2(float lo, float hi)
{
    uint64_t v;
    asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(lo), "f"(hi));
    return v;
}

constexpr int kRowBytes = kTileFreqs * 8;   // one bin row: W plane [32 x u32] | Y plane [32 x i32]

// Shared memory is addressed by 32-bit shared-window addresses with immediate offsets in the hot
// loops (one address register per stream, no generic-pointer arithmetic).
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint2 lds64(uint32_t addr)
{
    uint2 v;
    asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds128(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, uint4 v)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void red_add(uint32_t addr, uint32_t v)      // ATOMS.ADD, no return value
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// base + row * kRowBytes as ONE instruction (kept opaque so the compiler does not fold it into a
// 64-bit shift of the IMAD.WIDE result it comes from)
__device__ __forceinline__ uint32_t row_addr(uint32_t base, uint32_t row)
{
    uint32_t a;
    asm volatile("mad.lo.u32 %0, %1, 256, %2;" : "=r"(a) : "r"(row), "r"(base));
    return a;
}
static_assert(kRowBytes == 256, "row_addr hard-codes the row pitch");

// ---- the phases of one tile (32 trial frequencies, one per lane), written for a GROUP of warps:
//      `gw` = this warp's index in the group, `gnw` = warps in the group -------------------------

// The trial frequency of a lane and the shift of its bin grid (0 except in bls_refine, reading S3).
struct LaneFreq {
    double f;        // cycles/day
    double shift;    // cycles; the bin grid starts at phase `shift`
    double magic;    // kPhaseMagic - shift: the fast phase's additive constant
};

// Frequency index q of curve cv.  Search mode: the plan's grid.  Refine mode (a.n_fine > 0): q =
// (peak * n_fine + j) * n_shift + h -> f = f_lo + j * step (two roundings, as the oracle's S2),
// shift = h / (n_shift * nb).  Indices past the end repeat the last one (ragged last tile).
__device__ __forceinline__ LaneFreq lane_freq(const SearchArgs &a, int64_t cv, int q)
{
    LaneFreq lf;
    q = min(q, a.nf - 1);
    if (a.n_fine > 0) {
        const int per_peak = a.n_fine * a.n_shift;
        const int peak = q / per_peak, rem = q - peak * per_peak;
        const int j = rem / a.n_shift, h = rem - j * a.n_shift;
        const int64_t pi = cv * a.refine_k + peak;
        lf.f = __dadd_rn(a.f_lo[pi], __dmul_rn((double)j, a.f_step[pi]));
        lf.shift = __ddiv_rn((double)h, (double)(a.n_shift * a.nb));
    } else {
        lf.f = a.freqs[q];
        lf.shift = 0.0;
    }
    lf.magic = kPhaseMagic - lf.shift;
    return lf;
}

struct TileCtx {
    int nb, nrows, kmin, kmax, n_pad;   // n_pad: prepared records of the curve (a multiple of 4)
    uint32_t G;
    uint32_t w0;              // integer weight / residual sums of the curve's zero-time points
    int32_t y0;
    bool force_canon;
    float ncw, cy, wx2;       // -1/SWT, 1/SY, sum w x^2
    uint32_t swt;             // exact total of the integer weights
    double sr_scale, dp_scale;
};

__device__ __forceinline__ void load_ctx(TileCtx &c, const SearchArgs &a, const CurveMeta &meta, int nrows)
{
    c.nb = a.nb; c.kmin = a.kmin; c.kmax = a.kmax; c.nrows = nrows;
    c.force_canon = (a.force_canonical != 0) || (meta.force_canonical != 0);
    c.ncw = meta.ncw; c.cy = meta.cy; c.wx2 = (float)meta.wx2;
    c.swt = meta.swt; c.sr_scale = meta.sr_scale; c.dp_scale = meta.dp_scale;
    c.w0 = meta.w0; c.y0 = meta.y0;
    // guard band, units of 2^-32 bin: fast phase error nb/2 (nb with a shifted grid: kPhaseMagic - shift
    // rounds the shift to 2^-32 cycle) + canonical rule error nb/8
    c.G = a.n_fine > 0 ? 2u * (uint32_t)a.nb + 8u : (uint32_t)a.nb + 8u;
}

__device__ __forceinline__ void zero_bins(uint32_t bins_s, int nb, int gtid, int gthreads)
{
    const int nvec = nb * (kRowBytes / 16);
    for (int i = gtid; i < nvec; i += gthreads)
        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(bins_s + i * 16), "r"(0u) : "memory");
}

// One prepared point of the curve: from shared memory (LDS.128 broadcast) or through L1 (LDG.128).
template <bool PTS_SMEM>
__device__ __forceinline__ uint4 point_raw(uint32_t pts_sa, const PointRec *pts_g, int i)
{
    return PTS_SMEM ? lds128(pts_sa + (uint32_t)i * 16u) : __ldg(reinterpret_cast<const uint4 *>(pts_g + i));
}

// a2 Fold: warp gw takes groups of 4 consecutive prepared points gw, gw+gnw, ... (the record list is
// padded to a multiple of 4 with zero-weight records: no tail); lane l folds them at its frequency.
// During the fold row b holds int32 planes W[b][lane] | Y[b][lane]: lane l always hits bank l (and Y
// sits 128 B after W, one address register), so the native ATOMS.ADD is conflict-free by construction.
//   main loop   branch-free: point load, DFMA (fast phase), IMAD.WIDE (bin, position), LEA, 2 ATOMS.ADD,
//               and a running minimum of the positions' distance to a bin edge (half a VIMNMX3);
//   repair      only if some position of this warp's points fell inside the guard band (~1e-7 per
//               point-fold): the warp re-walks its points, takes the canonical rule (R8) for those and
//               moves the few that the fast rule put in the neighbouring bin (integer adds: exact);
//   zero-time points (t == 0: always exactly on a bin edge, always bin 0) are not in the record list:
//               prep sums them into (w0, y0), added here to bin 0 (bin nb-1 on a shifted grid).
// Curves whose |f t| can exceed the fast phase's range take the canonical rule for every point.
template <bool PTS_SMEM, int NG = 1>
__device__ __forceinline__ void fold_tile(const TileCtx &c, const LaneFreq &lf, uint32_t bins_s, uint32_t pts_sa,
                                          const PointRec *pts_g, int lane, int gw, int gnw, unsigned int &n_canon)
{
    const int nb = c.nb;
    const uint32_t G = c.G;
    const uint32_t colw = bins_s + lane * 4;       // W plane of this lane's column, row 0
    const int ngroups = c.n_pad >> 2;
    if (gw == 0 && (c.w0 | (uint32_t)c.y0)) {      // the zero-time points
        const uint32_t addr = colw + (lf.shift == 0.0 ? 0 : nb - 1) * kRowBytes;
        red_add(addr, c.w0);
        red_add(addr + 128, (uint32_t)c.y0);
    }
    if (c.force_canon) {
        for (int g = gw; g < ngroups; g += gnw) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint4 raw = point_raw<PTS_SMEM>(pts_sa, pts_g, g * 4 + u);
                const int bin = canonical_bin(lf.f, __hiloint2double((int)raw.y, (int)raw.x), nb, lf.shift);
                ++n_canon;
                const uint32_t addr = colw + bin * kRowBytes;
                red_add(addr, raw.z);
                red_add(addr + 128, raw.w);
            }
        }
        return;
    }
    uint32_t lomin = 0xffffffffu;
    int g = gw;
    if (NG > 1) {
        constexpr int NP = 4 * NG;                   // points in flight
        for (; g + (NG - 1) * gnw < ngroups; g += NG * gnw) {
            uint4 raw[NP];
            unsigned long long pr[NP];
#pragma unroll
            for (int u = 0; u < NP; ++u) raw[u] = point_raw<PTS_SMEM>(pts_sa, pts_g, (g + (u >> 2) * gnw) * 4 + (u & 3));
#pragma unroll
            for (int u = 0; u < NP; ++u) pr[u] = fast_bin_pos(lf.f, __hiloint2double((int)raw[u].y, (int)raw[u].x), nb, G, lf.magic);
#pragma unroll
            for (int u = 0; u < NP; u += 2) lomin = min(lomin, min((uint32_t)pr[u], (uint32_t)pr[u + 1]));
#pragma unroll
            for (int u = 0; u < NP; ++u) {
                const uint32_t addr = row_addr(colw, (uint32_t)(pr[u] >> 32));
                red_add(addr, raw[u].z);
                red_add(addr + 128, raw[u].w);
            }
        }
    }
    for (; g < ngroups; g += gnw) {                  // 4 points in flight
        uint4 raw[4];
        unsigned long long pr[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) raw[u] = point_raw<PTS_SMEM>(pts_sa, pts_g, g * 4 + u);
#pragma unroll
        for (int u = 0; u < 4; ++u) pr[u] = fast_bin_pos(lf.f, __hiloint2double((int)raw[u].y, (int)raw[u].x), nb, G, lf.magic);
#pragma unroll
        for (int u = 0; u < 4; u += 2) lomin = min(lomin, min((uint32_t)pr[u], (uint32_t)pr[u + 1]));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t addr = row_addr(colw, (uint32_t)(pr[u] >> 32));
            red_add(addr, raw[u].z);
            red_add(addr + 128, raw[u].w);
        }
    }
    const bool mine = lomin < 2u * G;
    if (__any_sync(0xffffffffu, mine)) {             // repair (rare): some point sits within G of a bin edge
        for (g = gw; g < ngroups; g += gnw) {
            for (int u = 0; u < 4; ++u) {
                const uint4 raw = point_raw<PTS_SMEM>(pts_sa, pts_g, g * 4 + u);
                const double t = __hiloint2double((int)raw.y, (int)raw.x);
                const unsigned long long pr = fast_bin_pos(lf.f, t, nb, G, lf.magic);
                if (mine && (uint32_t)pr < 2u * G) {
                    const int fb = (int)(pr >> 32), cb = canonical_bin(lf.f, t, nb, lf.shift);
                    ++n_canon;
                    if (cb != fb) {
                        red_add(colw + fb * kRowBytes, 0u - raw.z);
                        red_add(colw + fb * kRowBytes + 128, 0u - raw.w);
                        red_add(colw + cb * kRowBytes, raw.z);
                        red_add(colw + cb * kRowBytes + 128, raw.w);
                    }
                }
            }
        }
    }
}

// Cyclic extension: rows nb .. nrows-1 repeat rows 0 .., so a box that crosses phase 1 needs no
// index arithmetic in the search (reading R11).  16-byte chunks dealt to the group's threads.
__device__ __forceinline__ void extend_rows(const TileCtx &c, uint32_t bins_s, int gtid, int gthreads)
{
    const int nvec = (c.nrows - c.nb) * (kRowBytes / 16);
    for (int i = gtid; i < nvec; i += gthreads) {
        const int row = i >> 4, col = i & 15;
        const int src = row % c.nb;
        sts128(bins_s + (c.nb + row) * kRowBytes + col * 16, lds128(bins_s + src * kRowBytes + col * 16));
    }
}

// ---- a3/a4 box search ------------------------------------------------------------------------------
// A start tile is S consecutive start bins a0 .. a0+S-1 walked over the rows x = 0 .. kmax+S-2 of the
// column (row x = bin a0+x; rows >= nb are the cyclic extension); box (u, k) = start a0+u, width k
// ends at row x = u+k-1.  The thread keeps the maximum rank PER START (one FMNMX3 takes two boxes of the
// same start, from two consecutive rows); at the end of the tile the best start goes into the running
// best of the column.  A candidate code is the start bin a0+u (bit 31: the column needs the exact full
// search); the merge step re-walks that one start in exact integer arithmetic.
struct Best {               // per thread: its two frequencies
    float t0, t1;           // best |s| rsqrt(r(1-r)) seen (units of 1/SY)
    uint32_t c0, c1;        // candidate codes (start bins)
    float nmin0, nmin1;     // min over starts of n = -r at width kmax
};

struct RowI { uint2 w, y; };
__device__ __forceinline__ RowI ld_row(uint32_t p)
{
    RowI r;
    r.w = lds64(p);             // W plane: (qW[f0], qW[f1])
    r.y = lds64(p + 128);       // Y plane
    return r;
}
__device__ __forceinline__ void cvt_row(const RowI &r, uint64_t &W, uint64_t &Y)
{
    W = pack2(__uint2float_rn(r.w.x), __uint2float_rn(r.w.y));
    Y = pack2(__int2float_rn((int)r.y.x), __int2float_rn((int)r.y.y));
}
__device__ __forceinline__ void box_acc(uint64_t &n, uint64_t &s, uint64_t W, uint64_t Y, uint64_t ncw2)
{
    n = fma2(W, ncw2, n);       // n = -r
    s = add2(s, Y);
}
// rank |s| rsqrt(r(1-r)); n^2 + n = -r(1-r).  An empty box gives 0 * inf = NaN, which never wins an
// FMNMX; r == 1 gives inf, which the merge step recognises as impossible.
__device__ __forceinline__ void box_rank(uint64_t n, uint64_t s, float &t0, float &t1)
{
    const uint64_t d = fma2(n, n, n);
    float d0, d1;
    unpack2(d, d0, d1);
    const uint64_t t = mul2(s, pack2(fast_rsqrt(fabsf(d0)), fast_rsqrt(fabsf(d1))));
    unpack2(t, t0, t1);
}
// one row into start u: accumulate, rank, keep the start's maximum
__device__ __forceinline__ void box_step(uint64_t &n, uint64_t &s, uint64_t W, uint64_t Y, uint64_t ncw2, float &m0, float &m1)
{
    float t0, t1;
    box_acc(n, s, W, Y, ncw2);
    box_rank(n, s, t0, t1);
    m0 = fmaxf(m0, fabsf(t0));
    m1 = fmaxf(m1, fabsf(t1));
}
// two consecutive rows into start u: the two ranks share one three-input maximum per frequency
__device__ __forceinline__ void box_step2(uint64_t &n, uint64_t &s, uint64_t WA, uint64_t YA, uint64_t WB, uint64_t YB,
                                          uint64_t ncw2, float &m0, float &m1)
{
    float a0, a1, b0, b1;
    box_acc(n, s, WA, YA, ncw2);
    box_rank(n, s, a0, a1);
    box_acc(n, s, WB, YB, ncw2);
    box_rank(n, s, b0, b1);
    m0 = fmaxf(fmaxf(m0, fabsf(a0)), fabsf(b0));
    m1 = fmaxf(fmaxf(m1, fabsf(a1)), fabsf(b1));
}

template <int S>
__device__ __forceinline__ void search_tile(uint32_t p, int kmin, int kmax, uint64_t ncw2, uint32_t a0, Best &b)
{
    uint64_t rn[S], rs[S];
    float m0[S], m1[S];
#pragma unroll
    for (int u = 0; u < S; ++u) { rn[u] = 0ull; rs[u] = 0ull; m0[u] = 0.f; m1[u] = 0.f; }
    RowI nx = ld_row(p);
    uint64_t W, Y;
    if (kmin == 1 && kmax >= S - 1) {
        uint64_t WB, YB;
#pragma unroll
        for (int x = 0; x + 1 < S - 1; x += 2) {             // head, rows x and x+1: row x serves starts u <= x
            const RowI ra = nx;
            const RowI rb = ld_row(p + kRowBytes);
            p += 2 * kRowBytes; nx = ld_row(p);
            cvt_row(ra, W, Y);
            cvt_row(rb, WB, YB);
#pragma unroll
            for (int u = 0; u <= x; ++u) box_step2(rn[u], rs[u], W, Y, WB, YB, ncw2, m0[u], m1[u]);
            box_step(rn[x + 1], rs[x + 1], WB, YB, ncw2, m0[x + 1], m1[x + 1]);
        }
        if ((S - 1) & 1) {                                   // the odd last head row S-2
            const RowI cur = nx;
            p += kRowBytes; nx = ld_row(p);
            cvt_row(cur, W, Y);
#pragma unroll
            for (int u = 0; u <= S - 2; ++u) box_step(rn[u], rs[u], W, Y, ncw2, m0[u], m1[u]);
        }
        int x = S - 1;
        for (; x + 2 <= kmax; x += 2) {                      // full rows, two at a time: every start, no checks
            const RowI ra = nx;
            const RowI rb = ld_row(p + kRowBytes);
            p += 2 * kRowBytes; nx = ld_row(p);
            cvt_row(ra, W, Y);
            cvt_row(rb, WB, YB);
#pragma unroll
            for (int u = 0; u < S; ++u) box_step2(rn[u], rs[u], W, Y, WB, YB, ncw2, m0[u], m1[u]);
        }
        if (x < kmax) {
            const RowI cur = nx;
            p += kRowBytes; nx = ld_row(p);
            cvt_row(cur, W, Y);
#pragma unroll
            for (int u = 0; u < S; ++u) box_step(rn[u], rs[u], W, Y, ncw2, m0[u], m1[u]);
        }
#pragma unroll
        for (int d = 0; d + 1 < S - 1; d += 2) {             // tail, rows kmax+d and kmax+d+1: row kmax+d serves starts u > d
            const RowI ra = nx;
            const RowI rb = ld_row(p + kRowBytes);
            p += 2 * kRowBytes;
            if (d + 2 < S - 1) nx = ld_row(p);
            cvt_row(ra, W, Y);
            cvt_row(rb, WB, YB);
            box_step(rn[d + 1], rs[d + 1], W, Y, ncw2, m0[d + 1], m1[d + 1]);
#pragma unroll
            for (int u = d + 2; u < S; ++u) box_step2(rn[u], rs[u], W, Y, WB, YB, ncw2, m0[u], m1[u]);
        }
        if ((S - 1) & 1) {                                   // the odd last tail row kmax+S-2 serves start S-1
            cvt_row(nx, W, Y);
            box_step(rn[S - 1], rs[S - 1], W, Y, ncw2, m0[S - 1], m1[S - 1]);
        }
    } else {
        const int xend = kmax + S - 1;
        for (int x = 0; x < xend; ++x) {
            const RowI cur = nx;
            p += kRowBytes; nx = ld_row(p);                  // the last one reads one row too far (unused)
            cvt_row(cur, W, Y);
#pragma unroll
            for (int u = 0; u < S; ++u) {
                const int k = x - u + 1;
                if (k >= 1 && k <= kmax) {
                    if (k >= kmin) box_step(rn[u], rs[u], W, Y, ncw2, m0[u], m1[u]);
                    else box_acc(rn[u], rs[u], W, Y, ncw2);
                }
            }
        }
    }
#pragma unroll
    for (int u = 0; u < S; ++u) {
        if (m0[u] > b.t0) { b.t0 = m0[u]; b.c0 = a0 + u; }
        if (m1[u] > b.t1) { b.t1 = m1[u]; b.c1 = a0 + u; }
        float n0, n1;                                        // rn[u] = -r(start u, width kmax)
        unpack2(rn[u], n0, n1);
        b.nmin0 = fminf(b.nmin0, n0);
        b.nmin1 = fminf(b.nmin1, n1);
    }
}

// The starts of half-warp `half` of searching warp `sw` of `nsw`, as start tiles of at most SMAX starts.  `col` is
// the shared address of row 0 of this thread's frequency pair (W plane).
template <int SMAX>
__device__ __forceinline__ void search_slot(uint32_t col, const TileCtx &c, int sw, int nsw, int half, Best &b)
{
    const int w0 = (sw * c.nb) / nsw, w1 = ((sw + 1) * c.nb) / nsw;
    const int P = (w1 - w0 + 1) >> 1;
    if (P <= 0) return;
    int a0 = half ? w1 - P : w0;
    const int n = (P + SMAX - 1) / SMAX, base = P / n, extra = P - base * n;
    const uint64_t ncw2 = pack2(c.ncw, c.ncw);
    for (int i = 0; i < n; ++i) {
        const int S = base + (i < extra ? 1 : 0);
        const uint32_t p = col + a0 * kRowBytes;
#define BLS_TILE_CASE(N) \
    case N: if constexpr (N <= SMAX) search_tile<N>(p, c.kmin, c.kmax, ncw2, (uint32_t)a0, b); break;
        switch (S) {
            BLS_TILE_CASE(1) BLS_TILE_CASE(2) BLS_TILE_CASE(3) BLS_TILE_CASE(4) BLS_TILE_CASE(5) BLS_TILE_CASE(6)
            BLS_TILE_CASE(7) BLS_TILE_CASE(8) BLS_TILE_CASE(9) BLS_TILE_CASE(10) BLS_TILE_CASE(11) BLS_TILE_CASE(12)
            BLS_TILE_CASE(13)
            default: break;
        }
#undef BLS_TILE_CASE
        a0 += S;
    }
}
static_assert(kSmaxWide <= 13, "search_slot dispatches start tiles of up to 13 starts");

// Box search of one tile by one warp: lanes l and l+16 own the frequency pair (2l', 2l'+1),
// l' = l & 15, and different slots.  Writes the warp's 32 candidates (rank, code) to cand_t/cand_c.
template <int SMAX>
__device__ __forceinline__ void search_warp(uint32_t bins_s, const TileCtx &c, int lane, int sw, int nsw,
                                            float *cand_t, uint32_t *cand_c)
{
    Best b;
    b.t0 = 0.f; b.t1 = 0.f; b.c0 = 0u; b.c1 = 0u; b.nmin0 = 0.f; b.nmin1 = 0.f;
    const int half = lane >> 4, lp = lane & 15;
    search_slot<SMAX>(bins_s + lp * 8, c, sw, nsw, half, b);
    __syncwarp();
    const float ot0 = __shfl_xor_sync(0xffffffffu, b.t0, 16), ot1 = __shfl_xor_sync(0xffffffffu, b.t1, 16);
    const uint32_t oc0 = __shfl_xor_sync(0xffffffffu, b.c0, 16), oc1 = __shfl_xor_sync(0xffffffffu, b.c1, 16);
    const float on0 = __shfl_xor_sync(0xffffffffu, b.nmin0, 16), on1 = __shfl_xor_sync(0xffffffffu, b.nmin1, 16);
    if (ot0 > b.t0) { b.t0 = ot0; b.c0 = oc0; }
    if (ot1 > b.t1) { b.t1 = ot1; b.c1 = oc1; }
    // a box holding more than 0.9 of the weight: r(1-r) loses precision in fp32 -> exact full search
    if (fminf(b.nmin0, on0) < -0.9f) b.c0 |= 0x80000000u;
    if (fminf(b.nmin1, on1) < -0.9f) b.c1 |= 0x80000000u;
    if (half == 0) {
        *reinterpret_cast<float2 *>(cand_t + sw * 32 + 2 * lp) = make_float2(b.t0, b.t1);
        *reinterpret_cast<uint2 *>(cand_c + sw * 32 + 2 * lp) = make_uint2(b.c0, b.c1);
    }
}

// ---- merge: exact integer re-evaluation of the winning start, canonical ties, outputs -----------------

// Outputs of one (curve, frequency).
struct OutPtrs {
    float *sr; uint32_t *ak; float *depth;        // chunk scratch, row of this curve
    float *u_sr; uint16_t *u_start; uint16_t *u_width; float *u_depth;   // user rows or NULL
};

// One integer column of a bin buffer: row b holds qW at colw + b*256 and qY 128 bytes later.
struct IntColumn {
    uint32_t colw;
    int nb;
    __device__ __forceinline__ uint32_t W(int b) const { return lds32(colw + b * kRowBytes); }
    __device__ __forceinline__ int32_t Y(int b) const { return (int32_t)lds32(colw + b * kRowBytes + 128); }
    __device__ __forceinline__ bool empty(int b) const { return W(b) == 0u && Y(b) == 0; }
};

struct ExactBest {
    float v;            // S^2 / (R (SWT - R)) evaluated in fp32 from the exact integers: ranking only
    int a, k;
    uint32_t R;
    int32_t S;
};

// Reading R10: a box is valid iff r(1-r) > 0, decided exactly on the integers.  v is a deterministic
// function of (R, S), so boxes holding the same point set tie exactly.
__device__ __forceinline__ float exact_value(uint32_t R, int32_t S, uint32_t swt)
{
    const float Sf = (float)S;
    return __fdividef(Sf * Sf, (float)R * (float)(swt - R));
}

// Reading R12 for the full search: among equal values the smallest width wins, then the smallest start.
__device__ __forceinline__ void exact_eval(uint32_t R, int32_t S, uint32_t swt, int a, int k, ExactBest &e)
{
    if (R == 0u || R >= swt) return;
    const float v = exact_value(R, S, swt);
    if (v > e.v || (v == e.v && v > 0.f && (k < e.k || (k == e.k && a < e.a)))) {
        e.v = v; e.a = a; e.k = k; e.R = R; e.S = S;
    }
}

// every box of the column, in the oracle's order (guarded path: degenerate columns only)
__device__ __noinline__ void exact_full(IntColumn c, int kmin, int kmax, uint32_t swt, ExactBest &e)
{
    for (int a = 0; a < c.nb; ++a) {
        uint32_t R = 0u;
        int32_t Sy = 0;
        for (int k = 1; k <= kmax; ++k) {
            int j = a + k - 1; if (j >= c.nb) j -= c.nb;
            R += c.W(j); Sy += c.Y(j);
            if (k >= kmin) exact_eval(R, Sy, swt, a, k, e);
        }
    }
}

// Reading R12: among boxes holding the same point set take the smallest width, then the smallest
// start.  Given any box of that family: drop empty bins at both ends; if that falls below kmin,
// re-grow to kmin over empty bins, as far left as the numeric start index allows.
__device__ __forceinline__ void canonicalise(const IntColumn &c, int kmin, int &a, int &k)
{
    const int nb = c.nb;
    while (k > 1 && c.empty(a)) { a = a + 1 == nb ? 0 : a + 1; --k; }
    while (k > 1) { int e = a + k - 1; if (e >= nb) e -= nb; if (!c.empty(e)) break; --k; }
    if (k < kmin) {
        const int need = kmin - k;
        int L = 0, R = 0;
        while (L < need) { int b = a - 1 - L; if (b < 0) b += nb; if (!c.empty(b)) break; ++L; }
        while (R < need) { int b = a + k + R; if (b >= nb) b -= nb; if (!c.empty(b)) break; ++R; }
        const int d_hi = L, d_lo = need - R;          // feasible left shifts: d_lo <= d <= d_hi
        const int d = (d_lo <= a) ? min(d_hi, a) : d_hi;
        a -= d; if (a < 0) a += nb;
        k = kmin;
    }
}

// boxes (a, k), klo <= k <= khi, of ONE start: exact integer running sums in bin order.  Widths go up, so
// among equal values the smallest width stays (R12); equal values at other starts are boxes holding the
// same point set, which canonicalise() maps to the same answer.
__device__ __forceinline__ void exact_start(const IntColumn &c, uint32_t swt, int a, int klo, int khi, ExactBest &e)
{
    if (khi < klo) return;
    uint32_t R = 0u;
    int32_t Sy = 0;
    uint32_t p = c.colw + a * kRowBytes;
    int k = 1;
    for (; k + 3 < klo; k += 4, p += 4 * kRowBytes) {      // below klo: sums only, four rows in flight
        const uint32_t w0 = lds32(p), w1 = lds32(p + kRowBytes), w2 = lds32(p + 2 * kRowBytes), w3 = lds32(p + 3 * kRowBytes);
        const uint32_t y0 = lds32(p + 128), y1 = lds32(p + kRowBytes + 128), y2 = lds32(p + 2 * kRowBytes + 128),
                       y3 = lds32(p + 3 * kRowBytes + 128);
        R += (w0 + w1) + (w2 + w3);
        Sy += (int32_t)((y0 + y1) + (y2 + y3));
    }
    for (; k < klo; ++k, p += kRowBytes) { R += lds32(p); Sy += (int32_t)lds32(p + 128); }
    for (; k <= khi; ++k, p += kRowBytes) {
        R += lds32(p); Sy += (int32_t)lds32(p + 128);
        if (R != 0u && R < swt) {
            const float v = exact_value(R, Sy, swt);
            if (v > e.v) { e.v = v; e.k = k; e.R = R; e.S = Sy; }
        }
    }
}

// Merge of one tile by `mw` warps (warp `w` of them, lane = frequency column):
//   A  best of the `ncand` candidates (rank, start bin) of the column -> the winning start;
//   B  warp w re-evaluates its share of the widths kmin..kmax of that start in exact integer arithmetic
//      and posts its best (value, width << 16 | start);
//   C  after `sync`, the warp that holds the column's best box (value, then smallest width: reading R12)
//      canonicalises it and writes
//      SR = S^2/(R(SWT-R)) * sr_scale, depth = S/(R(SWT-R)) * dp_scale   (fp64, rounded once).
// cand_t/cand_c: [ncand][32] written by search_warp (and made visible by the caller's barrier);
// post_v/post_k: [mw][32] scratch.  Warps w >= mw of the group only take part in `sync`.
template <typename Sync>
__device__ __forceinline__ void merge_tile(const TileCtx &c, uint32_t bins_s, const float *cand_t, const uint32_t *cand_c,
                                           float *post_v, uint32_t *post_k, int ncand, int mw, int w, int lane, int q,
                                           int nf, const OutPtrs &o, Sync sync)
{
    if (w >= mw) { if (mw > 1) sync(); return; }
    float bt = 0.f;
    uint32_t bc = 0u, flag = 0u;
    for (int p = 0; p < ncand; ++p) {
        const float t = cand_t[p * 32 + lane];
        const uint32_t cc = cand_c[p * 32 + lane];
        flag |= cc;
        if (t > bt) { bt = t; bc = cc; }
    }
    const IntColumn col{bins_s + (uint32_t)lane * 4u, c.nb};
    ExactBest e;
    e.v = 0.f; e.a = 0; e.k = c.kmin; e.R = 0u; e.S = 0;
    const float tv = bt * c.cy;
    if ((flag >> 31) || !(tv * tv <= 1.001f * c.wx2 + 1e-30f)) {     // a box near r = 1, or inf / NaN
        if (w == 0) exact_full(col, c.kmin, c.kmax, c.swt, e);
    } else if (bt > 0.f) {
        const int a = (int)(bc & 0x7fffffffu);
        const int nk = c.kmax - c.kmin + 1, per = (nk + mw - 1) / mw;
        const int klo = c.kmin + w * per;
        e.a = a >= c.nb ? a - c.nb : a;                      // starts in the cyclic extension
        exact_start(col, c.swt, a, klo, min(c.kmax, klo + per - 1), e);
    }
    int win = 0;
    if (mw > 1) {
        post_v[w * 32 + lane] = e.v;
        post_k[w * 32 + lane] = ((uint32_t)e.k << 16) | (uint32_t)e.a;
        sync();
        float bv = 0.f;
        uint32_t bkey = 0xffffffffu;
        for (int p = 0; p < mw; ++p) {
            const float v = post_v[p * 32 + lane];
            const uint32_t key = post_k[p * 32 + lane];
            if (v > bv || (v == bv && v > 0.f && key < bkey)) { bv = v; bkey = key; win = p; }
        }
        if (!(bv > 0.f)) { win = 0; e.v = 0.f; }
    }
    if (win != w) return;
    float sr = 0.f, dp = 0.f;
    int ba = 0, bk = c.kmin;
    if (e.v > 0.f) {
        ba = e.a; bk = e.k;
        canonicalise(col, c.kmin, ba, bk);
        const double Rd = (double)e.R, Cd = (double)(c.swt - e.R), Sd = (double)e.S;
        const double inv = 1.0 / (Rd * Cd);
        sr = (float)(Sd * Sd * inv * c.sr_scale);
        dp = (float)(Sd * inv * c.dp_scale);
    }
    if (q < nf) {
        o.sr[q] = sr; o.ak[q] = ((uint32_t)bk << 16) | (uint32_t)ba; o.depth[q] = dp;
        if (o.u_sr) o.u_sr[q] = sr;
        if (o.u_start) o.u_start[q] = (uint16_t)ba;
        if (o.u_width) o.u_width[q] = (uint16_t)bk;
        if (o.u_depth) o.u_depth[q] = dp;
    }
}

__device__ __forceinline__ OutPtrs out_rows(const SearchArgs &a, int64_t curve_local, int64_t c)
{
    OutPtrs o;
    o.sr = a.sr + curve_local * a.nf; o.ak = a.ak + curve_local * a.nf; o.depth = a.depth + curve_local * a.nf;
    o.u_sr = a.u_sr ? a.u_sr + c * a.nf : nullptr;
    o.u_start = a.u_start ? a.u_start + c * a.nf : nullptr;
    o.u_width = a.u_width ? a.u_width + c * a.nf : nullptr;
    o.u_depth = a.u_depth ? a.u_depth + c * a.nf : nullptr;
    return o;
}

// data fault: zero-filled spectrum (include/bls.h)
__device__ __forceinline__ void zero_fill_outputs(const OutPtrs &o, int q_begin, int q_end, int kmin, int tid, int nthr)
{
    for (int q = q_begin + tid; q < q_end; q += nthr) {
        o.sr[q] = 0.f; o.ak[q] = (uint32_t)kmin << 16; o.depth[q] = 0.f;
        if (o.u_sr) o.u_sr[q] = 0.f;
        if (o.u_start) o.u_start[q] = 0;
        if (o.u_width) o.u_width[q] = (uint16_t)kmin;
        if (o.u_depth) o.u_depth[q] = 0.f;
    }
}

__device__ __forceinline__ void count_canonical(const SearchArgs &a, unsigned int n_canon, int lane)
{
    if (a.canon_count) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) n_canon += __shfl_xor_sync(0xffffffffu, n_canon, o);
        if (lane == 0 && n_canon) atomicAdd(a.canon_count, (unsigned long long)n_canon);
    }
}

// ---- common prologue: which curve / tiles this CTA owns; stage the curve (a1 Load) -------------------
struct WorkItem {
    int64_t curve_local, cv, beg;
    int tile0, tile1;
    CurveMeta meta;
    OutPtrs out;
};

__device__ __forceinline__ WorkItem work_item(const SearchArgs &a, TileCtx &c)
{
    WorkItem w;
    w.curve_local = blockIdx.x / a.items_per_curve;
    const int item = blockIdx.x % a.items_per_curve;
    w.cv = a.curve_base + w.curve_local;
    w.beg = a.poffsets[w.cv];                                  // prepared records: padded to multiples of 4
    c.n_pad = (int)(a.poffsets[w.cv + 1] - w.beg);
    w.meta = a.meta[w.cv];
    const int ntiles = (a.nf + kTileFreqs - 1) / kTileFreqs;
    w.tile0 = item * a.tiles_per_item;
    w.tile1 = min(w.tile0 + a.tiles_per_item, ntiles);
    w.out = out_rows(a, w.curve_local, w.cv);
    load_ctx(c, a, w.meta, a.nrows);
    return w;
}

template <bool PTS_SMEM>
__device__ __forceinline__ void stage_curve(const PointRec *pts_g, PointRec *pts_s, int n, int tid, int nthr)
{
    if (PTS_SMEM) {                               // coalesced LDG.128 -> STS.128, once per work item
        const uint4 *src = reinterpret_cast<const uint4 *>(pts_g);
        uint4 *dst = reinterpret_cast<uint4 *>(pts_s);
        for (int i = tid; i < n; i += nthr) dst[i] = __ldg(src + i);
    }
}

// ---- kernel 1: every warp does every phase, phases separated by CTA barriers.  Used where the
//      double-buffered bins of kernel 2 do not fit shared memory (nb above ~420 at wide boxes). ------
template <bool PTS_SMEM>
__global__ void __launch_bounds__(kMaxSearchWarps * 32, 2)
search_kernel(const SearchArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nw = nthr >> 5;
    TileCtx c;
    const WorkItem w = work_item(a, c);
    // smem: bins [nrows][256 B] | cand_t, cand_c, post_v, post_k [nw][32] each | points [n] (if PTS_SMEM)
    float *cand_t = reinterpret_cast<float *>(smem_raw + (size_t)c.nrows * kRowBytes);
    uint32_t *cand_c = reinterpret_cast<uint32_t *>(cand_t + nw * 32);
    float *post_v = reinterpret_cast<float *>(cand_c + nw * 32);
    uint32_t *post_k = reinterpret_cast<uint32_t *>(post_v + nw * 32);
    PointRec *pts_s = reinterpret_cast<PointRec *>(post_k + nw * 32);

    if (w.meta.status != BLS_CURVE_OK) {
        zero_fill_outputs(w.out, w.tile0 * kTileFreqs, min(w.tile1 * kTileFreqs, a.nf), a.kmin, tid, nthr);
        return;
    }
    const PointRec *pts_g = a.pts + w.beg;
    stage_curve<PTS_SMEM>(pts_g, pts_s, c.n_pad, tid, nthr);
    const uint32_t bins_s = smem_u32(smem_raw), pts_sa = smem_u32(pts_s);
    unsigned int n_canon = 0;

    LaneFreq lf_next = lane_freq(a, w.cv, w.tile0 * kTileFreqs + lane);     // ragged last tile: surplus lanes repeat the last f
    for (int tile = w.tile0; tile < w.tile1; ++tile) {
        const int q0 = tile * kTileFreqs;
        const LaneFreq lf = lf_next;
        zero_bins(bins_s, c.nb, tid, nthr);
        __syncthreads();
        if (a.fold_depth == 2) fold_tile<PTS_SMEM, 2>(c, lf, bins_s, pts_sa, pts_g, lane, warp, nw, n_canon);
        else fold_tile<PTS_SMEM, 1>(c, lf, bins_s, pts_sa, pts_g, lane, warp, nw, n_canon);
        if (tile + 1 < w.tile1) lf_next = lane_freq(a, w.cv, q0 + kTileFreqs + lane);   // in flight during the search
        __syncthreads();
        extend_rows(c, bins_s, tid, nthr);
        __syncthreads();
        search_warp<kSmax>(bins_s, c, lane, warp, nw, cand_t, cand_c);
        __syncthreads();
        merge_tile(c, bins_s, cand_t, cand_c, post_v, post_k, nw, min(nw, a.merge_warps), warp, lane, q0 + lane, a.nf, w.out,
                   [] { __syncthreads(); });
        __syncthreads();
    }
    count_canonical(a, n_canon, lane);
}

// ---- kernel 2: warp-specialised, double-buffered.  The fold is bound by the shared-memory pipe
//      (atomics + point broadcasts), the box search by the XU pipe (one MUFU.RSQ per box), the exact
//      merge by latency: they run CONCURRENTLY on different warps.  "Search warps" rank the boxes of
//      tile i in one bin buffer while "fold warps" zero / fold / extend tile i+1 into the other and
//      "merge warps" (shapes 1, 2; in shape 0 the fold warps, in front of their fold) finish tile i-1.
//      A buffer's life: fold -> FULL[b] -> search -> DONE[b] -> merge -> FREE[b] -> fold ...
//        FULL[b]  mbarrier: every fold thread arrives, every search warp polls on its own;
//        DONE[b]  named barrier: bar.arrive by the search warps, bar.sync by the merging warps;
//        FREE[b]  named barrier (shapes 1, 2): bar.arrive by the merge warps, bar.sync by the fold warps;
//      one named barrier for the fold group and one for the merge group.
__device__ __forceinline__ void named_sync(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void named_arrive(int id, int count)
{
    __threadfence_block();
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}
enum { kBarFree0 = 1, kBarFree1 = 2, kBarDone0 = 3, kBarDone1 = 4, kBarFoldGroup = 5, kBarMergeGroup = 6 };

// FULL[b] (fold -> search) is an mbarrier in shared memory: every fold thread arrives (release), every search
// warp polls on its own, so the search warps are not re-aligned at every tile: they drift apart and one warp's
// tile prologue / epilogue overlaps the steady loops of the others on the XU pipe.
__device__ __forceinline__ void mbar_init(uint32_t addr, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(addr), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t addr)
{
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t addr, uint32_t parity)
{
    uint32_t ok;
    for (;;) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(addr), "r"(parity), "r"(20000u) : "memory");        // suspend-time hint (ns)
        if (ok) break;                   // (a __nanosleep between polls measured no better: C1 573 against 568)
    }
}

// Launch shapes of kernel 2.  Shape 0: up to 20 warps at equal registers (96), the search / fold split chosen at
// run time (BLS_FLAG_WARPS / BLS_FLAG_FOLD_WARPS); the fold warps also do the exact merge.  Shapes 1 and 2: 28 warps
// launched at 72 registers in three roles.  The low-register warps (whole warpgroups) give registers back with
// setmaxnreg.dec and the search warps take them with setmaxnreg.inc, so a search thread holds start tiles of up to
// kTileStarts starts (fewer row loads and conversions per box: 3.9 instructions per box in the steady loop at 13
// starts, 4.4 at 7) and more warps are resident to hide each other's latencies.  Four of the low-register warps do
// nothing except the exact merge: the merge of tile i (latency-bound: a few dependent walks over one start's rows)
// runs beside the fold of tile i+1 instead of in front of the fold of tile i+2, which takes it off the fold warps'
// critical path (measured with clock64 per role: the fold warps never waited for the search warps, and spent a
// fifth of their time in the merge).
template <int SHAPE> struct WsShape;
template <> struct WsShape<0> { static constexpr int kWarps = kWsMaxWarps, kSearchWarps = 0, kMergeRole = 0, kTileStarts = kSmax, kSearchRegs = 0, kFoldRegs = 0; };
template <> struct WsShape<1> { static constexpr int kWarps = 28, kSearchWarps = 8, kMergeRole = 4, kTileStarts = kSmaxWide, kSearchRegs = 128, kFoldRegs = 48; };
template <> struct WsShape<2> { static constexpr int kWarps = 28, kSearchWarps = 12, kMergeRole = 4, kTileStarts = 9, kSearchRegs = 104, kFoldRegs = 48; };
int ws_shape_warps(int shape, int *search_warps)
{
    switch (shape) {
        case 1: *search_warps = WsShape<1>::kSearchWarps; return WsShape<1>::kWarps;
        case 2: *search_warps = WsShape<2>::kSearchWarps; return WsShape<2>::kWarps;
        default: *search_warps = 0; return kWsMaxWarps;
    }
}

template <bool PTS_SMEM, int SHAPE>
__global__ void __launch_bounds__(WsShape<SHAPE>::kWarps * 32, 1)
search_ws_kernel(const SearchArgs a)
{
    using Shape = WsShape<SHAPE>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x;
    constexpr int nmw = Shape::kMergeRole;                          // warps of the merge role (0: the fold warps merge)
    const int nsw = SHAPE ? Shape::kSearchWarps : a.search_warps, nlow = (nthr >> 5) - nsw, nfw = nlow - nmw;
    const int mw = nmw ? nmw : min(nfw, a.merge_warps);
    // the scheduler favours the highest warp ids (B300_MICROARCH.md: "hi-wid-first"): the XU-bound search
    // warps take them, the fold (and merge) warps the low ids
    const bool search_role = warp >= nlow;
    const int sw = warp - nlow;
    TileCtx c;
    const WorkItem w = work_item(a, c);
    // smem: bins[2] [nrows][256 B] | cand_t[2], cand_c[2] [nsw][32] | post_v, post_k [kMergeWarps][32] | FULL[2] | points [n]
    const size_t buf_bytes = (size_t)c.nrows * kRowBytes;
    float *cand_t = reinterpret_cast<float *>(smem_raw + 2 * buf_bytes);
    uint32_t *cand_c = reinterpret_cast<uint32_t *>(cand_t + 2 * nsw * 32);
    float *post_v = reinterpret_cast<float *>(cand_c + 2 * nsw * 32);
    uint32_t *post_k = reinterpret_cast<uint32_t *>(post_v + kMergeWarps * 32);
    const uint32_t full_bar = smem_u32(post_k + kMergeWarps * 32);          // two 8-byte mbarriers
    PointRec *pts_s = reinterpret_cast<PointRec *>(post_k + kMergeWarps * 32 + 4);

    if (w.meta.status != BLS_CURVE_OK) {
        zero_fill_outputs(w.out, w.tile0 * kTileFreqs, min(w.tile1 * kTileFreqs, a.nf), a.kmin, tid, nthr);
        return;
    }
    const PointRec *pts_g = a.pts + w.beg;
    stage_curve<PTS_SMEM>(pts_g, pts_s, c.n_pad, tid, nthr);        // a1 Load, by all warps
    if (tid == 0) { mbar_init(full_bar, nfw * 32); mbar_init(full_bar + 8, nfw * 32); }
    __syncthreads();
    const uint32_t bins_s = smem_u32(smem_raw), pts_sa = smem_u32(pts_s);
    const int nt = w.tile1 - w.tile0;

    if (search_role) {
        // ================= search warps: a3/a4 ranking only =================
        if constexpr (SHAPE != 0) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(Shape::kSearchRegs));
        for (int it = 0; it < nt; ++it) {
            const int b = it & 1;
            mbar_wait(full_bar + 8 * b, (it >> 1) & 1);           // buffer b holds the tile's integer rows
            search_warp<Shape::kTileStarts>(bins_s + b * (uint32_t)buf_bytes, c, lane, sw, nsw, cand_t + b * nsw * 32,
                                      cand_c + b * nsw * 32);
            named_arrive(kBarDone0 + b, nmw ? (nsw + nmw) * 32 : nthr);   // candidates posted, done reading buffer b
        }
    } else if (nmw > 0 && warp >= nfw) {
        // ================= merge warps (shapes 1 / 2): exact merge of tile i while the fold warps fold tile i+1 =================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Shape::kFoldRegs));
        for (int it = 0; it < nt; ++it) {
            const int b = it & 1;
            named_sync(kBarDone0 + b, (nsw + nmw) * 32);
            merge_tile(c, bins_s + b * (uint32_t)buf_bytes, cand_t + b * nsw * 32, cand_c + b * nsw * 32, post_v, post_k, nsw, nmw,
                       warp - nfw, lane, (w.tile0 + it) * kTileFreqs + lane, a.nf, w.out, [] { named_sync(kBarMergeGroup, nmw * 32); });
            if (it + 2 < nt) named_arrive(kBarFree0 + b, (nfw + nmw) * 32);   // every column has left the buffer
        }
    } else {
        // ================= fold warps: exact merge of tile i-2, then zero, a2 fold, cyclic extension =================
        if constexpr (SHAPE != 0) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Shape::kFoldRegs));
        const int gw = warp, gtid = tid, gthreads = nfw * 32;
        unsigned int n_canon = 0;
        auto merge = [&](int it) {
            const int b = it & 1;
            named_sync(kBarDone0 + b, nthr);
            merge_tile(c, bins_s + b * (uint32_t)buf_bytes, cand_t + b * nsw * 32, cand_c + b * nsw * 32, post_v, post_k, nsw, mw,
                       gw, lane, (w.tile0 + it) * kTileFreqs + lane, a.nf, w.out,
                       [gthreads] { named_sync(kBarFoldGroup, gthreads); });
            named_sync(kBarFoldGroup, gthreads);                  // every column has left the buffer
        };
        for (int it = 0; it < nt; ++it) {
            const int b = it & 1, tile = w.tile0 + it;
            const uint32_t buf = bins_s + b * (uint32_t)buf_bytes;
            if (it >= 2) {
                if (nmw) named_sync(kBarFree0 + b, (nfw + nmw) * 32);
                else merge(it - 2);
            }
            const LaneFreq lf = lane_freq(a, w.cv, tile * kTileFreqs + lane);
            zero_bins(buf, c.nb, gtid, gthreads);
            named_sync(kBarFoldGroup, gthreads);
            if (a.fold_depth == 2) fold_tile<PTS_SMEM, 2>(c, lf, buf, pts_sa, pts_g, lane, gw, nfw, n_canon);
            else fold_tile<PTS_SMEM, 1>(c, lf, buf, pts_sa, pts_g, lane, gw, nfw, n_canon);
            named_sync(kBarFoldGroup, gthreads);
            extend_rows(c, buf, gtid, gthreads);
            mbar_arrive(full_bar + 8 * b);
        }
        if (!nmw) for (int it = max(nt - 2, 0); it < nt; ++it) merge(it);   // drain
        count_canonical(a, n_canon, lane);
    }
}

// ---- kernel 3: one warp per tile.  For small shapes (C4: 200 epochs, 64 bins) a tile is a few
//      thousand instructions and the hand-offs of kernels 1/2 cost more than the work.  Here every
//      warp owns private bins and runs zero / fold / extend / search / merge of its own tiles with
//      warp syncs only; warps of an SM sit in different phases, so the LSU-bound fold of one overlaps
//      the XU-bound search of another without any CTA-level barrier. ------------------------------
template <bool PTS_SMEM>
__global__ void __launch_bounds__(kWtWarps * 32, 2)
search_wt_kernel(const SearchArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nw = nthr >> 5;
    TileCtx c;
    const WorkItem w = work_item(a, c);
    // smem: per warp { bins [nrows][256 B] | cand_t [32] | cand_c [32] } ... | points [n]
    const size_t per_warp = (size_t)c.nrows * kRowBytes + 256;
    unsigned char *mine = smem_raw + warp * per_warp;
    float *cand_t = reinterpret_cast<float *>(mine + (size_t)c.nrows * kRowBytes);
    uint32_t *cand_c = reinterpret_cast<uint32_t *>(cand_t + 32);
    PointRec *pts_s = reinterpret_cast<PointRec *>(smem_raw + nw * per_warp);

    if (w.meta.status != BLS_CURVE_OK) {
        zero_fill_outputs(w.out, w.tile0 * kTileFreqs, min(w.tile1 * kTileFreqs, a.nf), a.kmin, tid, nthr);
        return;
    }
    const PointRec *pts_g = a.pts + w.beg;
    stage_curve<PTS_SMEM>(pts_g, pts_s, c.n_pad, tid, nthr);
    __syncthreads();                              // the only CTA barrier
    const uint32_t buf = smem_u32(mine), pts_sa = smem_u32(pts_s);
    unsigned int n_canon = 0;

    for (int tile = w.tile0 + warp; tile < w.tile1; tile += nw) {
        const int q0 = tile * kTileFreqs;
        const LaneFreq lf = lane_freq(a, w.cv, q0 + lane);
        zero_bins(buf, c.nb, lane, 32);
        __syncwarp();
        fold_tile<PTS_SMEM, 2>(c, lf, buf, pts_sa, pts_g, lane, 0, 1, n_canon);
        __syncwarp();
        extend_rows(c, buf, lane, 32);
        __syncwarp();
        search_warp<kSmax>(buf, c, lane, 0, 1, cand_t, cand_c);
        __syncwarp();
        merge_tile(c, buf, cand_t, cand_c, nullptr, nullptr, 1, 1, 0, lane, q0 + lane, a.nf, w.out, [] {});
        __syncwarp();
    }
    count_canonical(a, n_canon, lane);
}

// ---- kernel 4 (row f2, field-shared cadence): kFieldStars stars of a field per CTA ---------------------
// All stars of a pointing share their epochs, so the phase and the bin index of an epoch at a
// trial frequency are the same for every star: this kernel computes them ONCE per (epoch, frequency) and adds the
// epoch's (qw, qy) of S stars into S bin buffers.  Measured as an instruction mix (profiles/r03_microbench.md):
// 9.6 point-folds per clock per SM at S = 3 against 5.7 for the per-star fold -- the DFMA, the slow IMAD.WIDE
// (18 lane-ops per clock per SM) and the row address are shared by S stars, and the stars' integers come two to
// an LDS.128.  Everything after the fold (extension rows, box search, exact merge, outputs) is kernel 1's, once per
// star on that star's buffer, so results are those of the per-star kernels (bins are exact integers).
//   shared memory: bins [S][nrows][256 B] | cand_t, cand_c, post_v, post_k [nw][32] | field records | S CurveMeta
//   field record of epoch e, (S + 1) / 2 uint4: (t lo, t hi, qw0, qy0), (qw1, qy1, qw2, qy2), ...
// The prepared records of a field are per star (prep_kernel<true>): a star's record of an epoch it has no
// measurement for carries no weight and a placeholder time.  Staging takes the epoch's time from the first star of
// the group whose record carries weight (all such records hold the same fp32 epoch time); if none does, the epoch
// adds zero to whatever bin it lands in.
template <int S>
__device__ __forceinline__ void field_add(uint32_t addr, uint32_t buf_bytes, uint32_t rec_sa, const uint4 &v0, bool negate)
{
    constexpr int REC = (S + 1) / 2;
    const uint32_t sg = negate ? 0xffffffffu : 0u, one = negate ? 1u : 0u;       // two's complement: -x = (x ^ ~0) + 1
    red_add(addr, (v0.z ^ sg) + one);
    red_add(addr + 128, (v0.w ^ sg) + one);
#pragma unroll
    for (int r = 1; r < REC; ++r) {
        const uint4 w = lds128(rec_sa + r * 16);
        const uint32_t a1 = addr + (uint32_t)(2 * r - 1) * buf_bytes, a2 = a1 + buf_bytes;
        red_add(a1, (w.x ^ sg) + one);
        red_add(a1 + 128, (w.y ^ sg) + one);
        red_add(a2, (w.z ^ sg) + one);
        red_add(a2 + 128, (w.w ^ sg) + one);
    }
}

template <int S>
__device__ __forceinline__ void fold_field_tile(int nb, uint32_t G, bool force_canon, const LaneFreq &lf, uint32_t bins_s,
                                                uint32_t buf_bytes, uint32_t frec_sa, int n_pad, const CurveMeta *metas,
                                                int lane, int gw, int gnw, unsigned int &n_canon)
{
    constexpr int REC = (S + 1) / 2;
    const uint32_t colw = bins_s + lane * 4;
    const int ngroups = n_pad >> 2;
    if (gw == 0) {                                   // the zero-time epoch of each star (bin 0)
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const uint32_t w0 = metas[s].w0;
            const int32_t y0 = metas[s].y0;
            if (w0 | (uint32_t)y0) {
                red_add(colw + s * buf_bytes, w0);
                red_add(colw + s * buf_bytes + 128, (uint32_t)y0);
            }
        }
    }
    if (force_canon) {
        for (int g = gw; g < ngroups; g += gnw)
            for (int u = 0; u < 4; ++u) {
                const uint32_t ra = frec_sa + (uint32_t)(g * 4 + u) * (REC * 16);
                const uint4 v0 = lds128(ra);
                const int bin = canonical_bin(lf.f, __hiloint2double((int)v0.y, (int)v0.x), nb, 0.0);
                n_canon += S;
                field_add<S>(colw + bin * kRowBytes, buf_bytes, ra, v0, false);
            }
        return;
    }
    uint32_t lomin = 0xffffffffu;
    for (int g = gw; g < ngroups; g += gnw) {        // 4 epochs in flight, S stars each
        uint4 v0[4];
        unsigned long long pr[4];
        const uint32_t ra = frec_sa + (uint32_t)(g * 4) * (REC * 16);
#pragma unroll
        for (int u = 0; u < 4; ++u) v0[u] = lds128(ra + u * (REC * 16));
#pragma unroll
        for (int u = 0; u < 4; ++u) pr[u] = fast_bin_pos(lf.f, __hiloint2double((int)v0[u].y, (int)v0[u].x), nb, G, lf.magic);
#pragma unroll
        for (int u = 0; u < 4; u += 2) lomin = min(lomin, min((uint32_t)pr[u], (uint32_t)pr[u + 1]));
#pragma unroll
        for (int u = 0; u < 4; ++u)
            field_add<S>(row_addr(colw, (uint32_t)(pr[u] >> 32)), buf_bytes, ra + u * (REC * 16), v0[u], false);
    }
    const bool mine = lomin < 2u * G;
    if (__any_sync(0xffffffffu, mine)) {             // repair (rare), as in fold_tile: move the epoch's S contributions
        for (int g = gw; g < ngroups; g += gnw)
            for (int u = 0; u < 4; ++u) {
                const uint32_t ra = frec_sa + (uint32_t)(g * 4 + u) * (REC * 16);
                const uint4 v0 = lds128(ra);
                const double t = __hiloint2double((int)v0.y, (int)v0.x);
                const unsigned long long pr = fast_bin_pos(lf.f, t, nb, G, lf.magic);
                if (mine && (uint32_t)pr < 2u * G) {
                    const int fb = (int)(pr >> 32), cb = canonical_bin(lf.f, t, nb, 0.0);
                    n_canon += S;
                    if (cb != fb) {
                        field_add<S>(colw + fb * kRowBytes, buf_bytes, ra, v0, true);
                        field_add<S>(colw + cb * kRowBytes, buf_bytes, ra, v0, false);
                    }
                }
            }
    }
}

size_t field_smem_bytes(int nb, int kmax, int warps, int64_t n_pad)
{
    return (size_t)kFieldStars * search_rows_for(nb, kmax, 0) * kRowBytes + (size_t)4 * warps * kTileFreqs * 4 +
           (size_t)n_pad * ((kFieldStars + 1) / 2) * 16 + (size_t)kFieldStars * sizeof(CurveMeta);
}

template <int S>
__global__ void __launch_bounds__(kMaxSearchWarps * 32, 2)
search_field_kernel(const SearchArgs a)
{
    constexpr int REC = (S + 1) / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nw = nthr >> 5;
    const int64_t local0 = (int64_t)(blockIdx.x / a.items_per_curve) * S;     // first star of the group, within the launch
    const int item = blockIdx.x % a.items_per_curve;
    const int ns = (int)min((int64_t)S, a.field_curves - local0);            // the last group of a launch may be short
    const int64_t cv0 = a.curve_base + local0;
    const int64_t rec0 = a.poffsets[cv0];
    const int n_pad = (int)(a.poffsets[cv0 + 1] - rec0);                      // the same for every star of a field
    const int ntiles = (a.nf + kTileFreqs - 1) / kTileFreqs;
    const int tile0 = item * a.tiles_per_item, tile1 = min(tile0 + a.tiles_per_item, ntiles);
    const uint32_t buf_bytes = (uint32_t)a.nrows * kRowBytes;
    float *cand_t = reinterpret_cast<float *>(smem_raw + (size_t)S * buf_bytes);
    uint32_t *cand_c = reinterpret_cast<uint32_t *>(cand_t + nw * 32);
    float *post_v = reinterpret_cast<float *>(cand_c + nw * 32);
    uint32_t *post_k = reinterpret_cast<uint32_t *>(post_v + nw * 32);
    uint4 *frec = reinterpret_cast<uint4 *>(post_k + nw * 32);
    CurveMeta *metas = reinterpret_cast<CurveMeta *>(frec + (size_t)n_pad * REC);

    if (tid < S) {
        CurveMeta m;
        if (tid < ns) m = a.meta[cv0 + tid];
        else {
            m.ncw = 0.f; m.cy = 0.f; m.status = BLS_CURVE_TOO_FEW; m.force_canonical = 0; m.swt = 0u; m.w0 = 0u; m.y0 = 0;
            m.pad_ = 0; m.sr_scale = 0.0; m.dp_scale = 0.0; m.wx2 = 0.0;
        }
        metas[tid] = m;
    }
    for (int e = tid; e < n_pad; e += nthr) {        // a1 Load: the group's records -> field records
        uint4 r[S];
#pragma unroll
        for (int s = 0; s < S; ++s)
            r[s] = s < ns ? __ldg(reinterpret_cast<const uint4 *>(a.pts + rec0 + (int64_t)s * n_pad + e)) : make_uint4(0u, 0u, 0u, 0u);
        uint32_t tl = r[0].x, th = r[0].y;
        bool weighted = (r[0].z | r[0].w) != 0u, timed = (tl | th) != 0u;
#pragma unroll
        for (int s = 1; s < S; ++s) {
            const bool ws = (r[s].z | r[s].w) != 0u, ts = (r[s].x | r[s].y) != 0u;
            if ((ws && !weighted) || (ts && !timed && !weighted)) { tl = r[s].x; th = r[s].y; }
            weighted |= ws; timed |= ts;
        }
        frec[e * REC] = make_uint4(tl, th, r[0].z, r[0].w);
#pragma unroll
        for (int q = 1; q < REC; ++q) frec[e * REC + q] = make_uint4(r[2 * q - 1].z, r[2 * q - 1].w, r[2 * q].z, r[2 * q].w);
    }
    __syncthreads();
    bool any_ok = false, force_canon = a.force_canonical != 0;
    for (int s = 0; s < ns; ++s) {
        if (metas[s].status != BLS_CURVE_OK)
            zero_fill_outputs(out_rows(a, local0 + s, cv0 + s), tile0 * kTileFreqs, min(tile1 * kTileFreqs, a.nf), a.kmin, tid, nthr);
        else any_ok = true;
        force_canon |= metas[s].force_canonical != 0;
    }
    if (!any_ok) return;
    const uint32_t bins_s = smem_u32(smem_raw), frec_sa = smem_u32(frec);
    const uint32_t G = (uint32_t)a.nb + 8u;
    unsigned int n_canon = 0;

    // After the shared fold the CTA splits into S pairs of warps, one pair per star, each with its own named barrier:
    // pair s extends, searches and merges star s's buffer exactly as a two-warp CTA of kernel 1 would, then zeroes
    // that buffer for the next tile.  Two CTA barriers per tile: bins zeroed -> fold, fold -> pairs.
    const int s_mine = warp >> 1, pw = warp & 1, ptid = tid & 63;
    const bool mine_ok = metas[s_mine].status == BLS_CURVE_OK;                 // uniform over the pair
    const uint32_t buf = bins_s + s_mine * buf_bytes;
    float *pc_t = cand_t + s_mine * 64, *pp_v = post_v + s_mine * 64;
    uint32_t *pc_c = cand_c + s_mine * 64, *pp_k = post_k + s_mine * 64;
    const int bar = 1 + s_mine;
    TileCtx c;
    load_ctx(c, a, metas[s_mine], a.nrows);
    c.n_pad = n_pad;
    const OutPtrs outp = out_rows(a, local0 + min(s_mine, ns - 1), cv0 + min(s_mine, ns - 1));
    zero_bins(buf, a.nb, ptid, 64);
    __syncthreads();
    LaneFreq lf_next = lane_freq(a, cv0, tile0 * kTileFreqs + lane);
    for (int tile = tile0; tile < tile1; ++tile) {
        const int q0 = tile * kTileFreqs;
        const LaneFreq lf = lf_next;
        fold_field_tile<S>(a.nb, G, force_canon, lf, bins_s, buf_bytes, frec_sa, n_pad, metas, lane, warp, nw, n_canon);
        if (tile + 1 < tile1) lf_next = lane_freq(a, cv0, q0 + kTileFreqs + lane);
        __syncthreads();
        if (mine_ok) {
            extend_rows(c, buf, ptid, 64);
            named_sync(bar, 64);
            search_warp<kSmax>(buf, c, lane, pw, 2, pc_t, pc_c);
            named_sync(bar, 64);
            merge_tile(c, buf, pc_t, pc_c, pp_v, pp_k, 2, 2, pw, lane, q0 + lane, a.nf, outp, [bar] { named_sync(bar, 64); });
            named_sync(bar, 64);
            zero_bins(buf, a.nb, ptid, 64);
        }
        __syncthreads();
    }
    count_canonical(a, n_canon, lane);
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
        bins[i] = fold_bin(f[i], t[i], nb, G, force_canon != 0, n_canon, kPhaseMagic, 0.0);
    if (n_canon && n_canon_out) atomicAdd(n_canon_out, (unsigned long long)n_canon);
}

cudaError_t launch_debug_bins(const double *f, const double *t, int64_t n, int nb, int force_canon,
                              int32_t *bins, unsigned long long *n_canon, int sm_count, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    int64_t blocks = (n + 255) / 256;
    if (blocks > (int64_t)sm_count * 16) blocks = (int64_t)sm_count * 16;
    debug_bins_kernel<<<(unsigned)blocks, 256, 0, st>>>(f, t, n, nb, force_canon, bins, n_canon);
    return cudaGetLastError();
}

// The same for the shifted bin grids of bls_refine (reading S3): shift = h / (n_shift * nb) cycles, the additive
// constant kPhaseMagic - shift and the wider guard band 2 nb + 8, exactly as lane_freq / load_ctx set them up.
__global__ void debug_bins_shift_kernel(const double *__restrict__ f, const double *__restrict__ t, int64_t n, int nb,
                                        int h, int n_shift, int force_canon, int32_t *__restrict__ bins,
                                        unsigned long long *__restrict__ n_canon_out)
{
    const uint32_t G = 2u * (uint32_t)nb + 8u;
    const double shift = __ddiv_rn((double)h, (double)(n_shift * nb));
    const double magic = kPhaseMagic - shift;
    unsigned int n_canon = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        bins[i] = fold_bin(f[i], t[i], nb, G, force_canon != 0, n_canon, magic, shift);
    if (n_canon && n_canon_out) atomicAdd(n_canon_out, (unsigned long long)n_canon);
}

cudaError_t launch_debug_bins_shift(const double *f, const double *t, int64_t n, int nb, int h, int n_shift, int force_canon,
                                    int32_t *bins, unsigned long long *n_canon, int sm_count, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    int64_t blocks = (n + 255) / 256;
    if (blocks > (int64_t)sm_count * 16) blocks = (int64_t)sm_count * 16;
    debug_bins_shift_kernel<<<(unsigned)blocks, 256, 0, st>>>(f, t, n, nb, h, n_shift, force_canon, bins, n_canon);
    return cudaGetLastError();
}

cudaError_t search_configure(int max_smem_optin)
{
    const void *fns[] = {(const void *)search_kernel<true>,    (const void *)search_kernel<false>,
                         (const void *)search_ws_kernel<true, 0>, (const void *)search_ws_kernel<false, 0>,
                         (const void *)search_ws_kernel<true, 1>, (const void *)search_ws_kernel<false, 1>,
                         (const void *)search_ws_kernel<true, 2>, (const void *)search_ws_kernel<false, 2>,
                         (const void *)search_wt_kernel<true>, (const void *)search_wt_kernel<false>,
                         (const void *)search_field_kernel<kFieldStars>};
    for (const void *f : fns) {
        cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_search(const SearchArgs &a, int64_t chunk_curves, size_t smem, cudaStream_t st)
{
    const int64_t units = a.kernel == 4 ? (chunk_curves + kFieldStars - 1) / kFieldStars : chunk_curves;   // kernel 4: groups of stars
    const int64_t grid = units * (int64_t)a.items_per_curve;
    if (grid <= 0) return cudaSuccess;
    if (grid > 2147483647LL) return cudaErrorInvalidConfiguration;
    const unsigned g = (unsigned)grid;
#define BLS_LAUNCH(K)                                                  \
    do {                                                               \
        if (a.pts_in_smem) K<true><<<g, a.threads, smem, st>>>(a);     \
        else K<false><<<g, a.threads, smem, st>>>(a);                  \
    } while (0)
    if (a.kernel == 4) search_field_kernel<kFieldStars><<<g, a.threads, smem, st>>>(a);
    else if (a.kernel == 3) BLS_LAUNCH(search_wt_kernel);
    else if (a.kernel == 2) {
#define BLS_LAUNCH_WS(SH)                                                           \
    do {                                                                            \
        if (a.pts_in_smem) search_ws_kernel<true, SH><<<g, a.threads, smem, st>>>(a); \
        else search_ws_kernel<false, SH><<<g, a.threads, smem, st>>>(a);            \
    } while (0)
        switch (a.ws_shape) {
            case 1: BLS_LAUNCH_WS(1); break;
            case 2: BLS_LAUNCH_WS(2); break;
            default: BLS_LAUNCH_WS(0); break;
        }
#undef BLS_LAUNCH_WS
    }
    else BLS_LAUNCH(search_kernel);
#undef BLS_LAUNCH
    return cudaGetLastError();
}

}  // namespace bls
