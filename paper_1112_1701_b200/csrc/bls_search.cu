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
//     frequency and slides an 8-row window over the bins, so one shared load feeds 4 boxes; sums
//     are direct running sums in bin order (no prefix differences), so boxes holding the same
//     point set tie bitwise;
//   * boxes are ranked by |s| * rsqrt(r(1-r)) (one MUFU.RSQ + one FMUL; monotone in SR); a thread
//     keeps only the maximum per block of 16 boxes (FMNMX3 tree) and the block's id, re-walks its
//     winning block once at the end to find the box, and the merge step canonicalises exact ties
//     (trim empty edge bins -> smallest width, then smallest start: reading R12).
#include "bls_internal.cuh"

namespace bls {

// `buffers` = 1 (search_kernel) or 2 (search_ws_kernel); `warps` = warps that write partial results
size_t search_smem_bytes(int nb, int kmax, int warps, int buffers, int64_t n_points_in_smem)
{
    size_t bins = (size_t)search_rows(nb, kmax) * kTileFreqs * 8;
    size_t red = (size_t)2 * warps * kTileFreqs * 4;
    return (size_t)buffers * (bins + red) + (size_t)n_points_in_smem * sizeof(PointRec);
}

// Geometry of the box search: a thread owns S consecutive start bins (S = 4 or 5), the
// ceil(nb/S) start tiles of a column are dealt to the warps.  Pick (S, warps in [6,10]) that wastes
// the fewest thread-tiles; ties go to S = 5 (fewer loads per box), then to more warps.
void search_geometry(int nb, int max_warps, int *starts_per_thread, int *warps)
{
    int best_s = 4, best_w = 8;
    double best_cost = 1e30;
    for (int s = 4; s <= 5; ++s) {
        const int nst = (nb + s - 1) / s;
        for (int w = 6; w <= max_warps; ++w) {
            const int per = (nst + w - 1) / w;
            const double cost = (double)per * w * s / nb;      // thread-starts issued per useful start
            if (cost < best_cost - 1e-9 || (cost < best_cost + 1e-9 && (s > best_s || (s == best_s && w > best_w)))) {
                best_cost = cost; best_s = s; best_w = w;
            }
        }
    }
    *starts_per_thread = best_s;
    *warps = best_w;
}

__device__ __noinline__ int canonical_bin(double f, double t, int nb)
{
    double p = __dmul_rn(f, t);
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

// Bins of one frequency column after the convert pass: row b holds the pair (W, Y) at col[b*32].
struct Column {
    const float2 *col;
    int nb;
    __device__ __forceinline__ float W(int b) const { return col[b * 32].x; }
    __device__ __forceinline__ float Y(int b) const { return col[b * 32].y; }
};

// Scalar, guarded re-search of one frequency column in canonical order; only used when the fast
// search produced a non-finite or impossible value (a box holding the entire weight, r == 1.0f).
__device__ __noinline__ void careful_search(Column c, int kmin, int kmax, float &bv, uint32_t &bkey)
{
    bv = 0.f; bkey = ((uint32_t)kmin << 16);
    for (int a = 0; a < c.nb; ++a) {
        float r = 0.f, s = 0.f;
        for (int k = 1; k <= kmax; ++k) {
            int j = a + k - 1; if (j >= c.nb) j -= c.nb;
            r += c.W(j); s += c.Y(j);
            if (k < kmin) continue;
            float den = fmaf(-r, r, r);
            if (!(den > 0.f) || !(r < 1.f)) continue;
            float v = s * s / den;
            uint32_t key = ((uint32_t)k << 16) | (uint32_t)a;
            if (v > bv || (v == bv && v > 0.f && key < bkey)) { bv = v; bkey = key; }
        }
    }
}

// Reading R12: among boxes holding the same point set take the smallest width, then the smallest
// start.  Given any box of that family: drop empty bins at both ends; if that falls below kmin,
// re-grow to kmin over empty bins, as far left as the numeric start index allows.
__device__ __forceinline__ void canonicalise(Column c, int kmin, int &a, int &k)
{
    const int nb = c.nb;
    auto empty = [&](int b) { return c.W(b) == 0.f && c.Y(b) == 0.f; };
    while (k > 1 && empty(a)) { a = a + 1 == nb ? 0 : a + 1; --k; }
    while (k > 1) { int e = a + k - 1; if (e >= nb) e -= nb; if (!empty(e)) break; --k; }
    if (k < kmin) {
        const int need = kmin - k;
        int L = 0, R = 0;
        while (L < need) { int b = a - 1 - L; if (b < 0) b += nb; if (!empty(b)) break; ++L; }
        while (R < need) { int b = a + k + R; if (b >= nb) b -= nb; if (!empty(b)) break; ++R; }
        const int d_hi = L, d_lo = need - R;          // feasible left shifts: d_lo <= d <= d_hi
        const int d = (d_lo <= a) ? min(d_hi, a) : d_hi;
        a -= d; if (a < 0) a += nb;
        k = kmin;
    }
}

// ---- packed fp32 pairs -------------------------------------------------------------------------
// After the fold a bin row holds, per frequency column, the pair (W, Y) as one 64-bit word, so a
// box's running sums (r, s) advance with ONE packed add (FADD2) fed by ONE LDS.64.
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b)
{
    uint64_t c;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(c) : "l"(a), "l"(b));
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

constexpr int kRowBytes = kTileFreqs * 8;   // one bin row: 32 columns x (W, Y)

// Shared memory is addressed by 32-bit shared-window addresses with immediate offsets in the hot
// loops (one address register per stream, no generic-pointer arithmetic).
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t lds64(uint32_t addr)
{
    uint64_t v;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
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
__device__ __forceinline__ void sts64(uint32_t addr, uint64_t v)
{
    asm volatile("st.shared.b64 [%0], %1;" ::"r"(addr), "l"(v) : "memory");
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

// rows g .. g+3 of this thread's column; `p` is the shared address of row g of the column
__device__ __forceinline__ void load4(uint32_t p, uint64_t (&v)[4])
{
#pragma unroll
    for (int i = 0; i < 4; ++i) v[i] = lds64(p + i * kRowBytes);
}

// 16 boxes: starts u = 0..3 (rows of the window), widths k0+1 .. k0+4.  Running sums advance by one
// row per width; returns the largest |s| * rsqrt(r(1-r)).  NaN (empty box: 0 * inf, or r > 1 by
// rounding: rsqrt of a negative, or an invalid start seeded with NaN) never wins an FMNMX.
// The 8-row window is two halves (cur = rows g..g+3, nxt = rows g+4..g+7) so the caller can
// ping-pong them instead of shifting registers.
#define WIN(cur, nxt, i) ((i) < 4 ? cur[(i) & 3] : nxt[(i) & 3])

template <int S, bool CHECK>
__device__ __forceinline__ float block_max(uint64_t (&rs)[S], const uint64_t (&cur)[4], const uint64_t (&nxt)[4],
                                           int k0, int kmin, int kmax)
{
    float mj[4] = {0.f, 0.f, 0.f, 0.f};           // one short FMNMX chain per width, joined at the end
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int u = 0; u < S; ++u) rs[u] = add2(rs[u], WIN(cur, nxt, u + j));
        if (!CHECK || (k0 + j + 1 >= kmin && k0 + j + 1 <= kmax)) {
#pragma unroll
            for (int u = 0; u < S; ++u) {
                float r, s;
                unpack2(rs[u], r, s);
                const float den = fmaf(-r, r, r);       // r (1 - r)
                const float t = s * fast_rsqrt(den);
                mj[j] = fmaxf(mj[j], fabsf(t));
            }
        }
    }
    return fmaxf(fmaxf(mj[0], mj[1]), fmaxf(mj[2], mj[3]));
}

// Box search of one frequency column by one thread: start tiles tl = first, first+stride, ... of
// S consecutive start bins each (S = 4 or 5: S + 3 rows fit the 8-row window).
// `col` is the shared address of row 0 of the column; rows nb .. are copies of rows 0 .. (cyclic
// boxes without index arithmetic).  Returns the best |t| (t^2 = SR) and its (width << 16 | start)
// key; ties in any order.
template <int S>
__device__ __forceinline__ void search_column(uint32_t col, int nb, int kmin, int kmax, int first, int stride,
                                              float &out_t, uint32_t &out_key)
{
    static_assert(S == 4 || S == 5, "the 8-row window holds S + 3 rows");
    const int nst = (nb + S - 1) / S;
    const int nkb = (kmax + 3) >> 2;
    const int kb_full_lo = (kmin + 2) >> 2;          // blocks kb in [kb_full_lo, kb_full_hi) need no width check
    const int kb_full_hi = kmax >> 2;
    const uint64_t nan2 = pack2(__int_as_float(0x7fc00000), 0.f);
    float best = 0.f;
    int bcode = -1;
    for (int tl = first; tl < nst; tl += stride) {
        uint32_t p = col + tl * (S * kRowBytes);
        const int tcode = tl << 10;
        uint64_t rs[S], wa[4], wb[4];
#pragma unroll
        for (int u = 0; u < S; ++u) rs[u] = (tl * S + u < nb) ? 0ull : nan2;
        load4(p, wa);
        int kb = 0;
        // head blocks below kmin (only when kmin > 4), one at a time, window shifted through registers
        for (; kb < kb_full_lo && kb < nkb; ++kb) {
            p += 4 * kRowBytes;
            load4(p, wb);
            const float m = block_max<S, true>(rs, wa, wb, kb * 4, kmin, kmax);
            if (m > best) { best = m; bcode = tcode | kb; }
#pragma unroll
            for (int i = 0; i < 4; ++i) wa[i] = wb[i];
        }
        // two full blocks per iteration, the window halves ping-pong
        for (; kb + 2 <= kb_full_hi; kb += 2) {
            load4(p + 4 * kRowBytes, wb);
            float m = block_max<S, false>(rs, wa, wb, 0, 0, 0);
            if (m > best) { best = m; bcode = tcode | kb; }
            load4(p + 8 * kRowBytes, wa);
            m = block_max<S, false>(rs, wb, wa, 0, 0, 0);
            if (m > best) { best = m; bcode = tcode | (kb + 1); }
            p += 8 * kRowBytes;
        }
        // tail: at most one full block and the block that holds kmax
        if (kb + 2 <= nkb) {
            load4(p + 4 * kRowBytes, wb);
            float m = block_max<S, true>(rs, wa, wb, kb * 4, kmin, kmax);
            if (m > best) { best = m; bcode = tcode | kb; }
            load4(p + 8 * kRowBytes, wa);
            m = block_max<S, true>(rs, wb, wa, kb * 4 + 4, kmin, kmax);
            if (m > best) { best = m; bcode = tcode | (kb + 1); }
        } else if (kb < nkb) {
            load4(p + 4 * kRowBytes, wb);
            const float m = block_max<S, true>(rs, wa, wb, kb * 4, kmin, kmax);
            if (m > best) { best = m; bcode = tcode | kb; }
        }
    }
    out_t = 0.f;
    out_key = (uint32_t)kmin << 16;
    if (bcode < 0) return;
    // Re-walk to the winning block: first only the running sums (lanes differ in how far they
    // go, so this loop holds nothing else), then that block's boxes once, with the argmax.
    // Identical operations in identical order, so identical values.
    const int tl = bcode >> 10, kbs = bcode & 1023;
    uint32_t p = col + tl * (S * kRowBytes);
    uint64_t rs[S], w[8];
#pragma unroll
    for (int u = 0; u < S; ++u) rs[u] = (tl * S + u < nb) ? 0ull : nan2;
#pragma unroll
    for (int i = 0; i < 4; ++i) w[i] = lds64(p + i * kRowBytes);
    for (int kb = 0; kb < kbs; ++kb) {
        p += 4 * kRowBytes;
#pragma unroll
        for (int i = 0; i < 4; ++i) w[4 + i] = lds64(p + i * kRowBytes);
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int u = 0; u < S; ++u) rs[u] = add2(rs[u], w[u + j]);
#pragma unroll
        for (int i = 0; i < 4; ++i) w[i] = w[i + 4];
    }
    p += 4 * kRowBytes;
#pragma unroll
    for (int i = 0; i < 4; ++i) w[4 + i] = lds64(p + i * kRowBytes);
    float bt = 0.f;
    int bk = kmin, bu = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int u = 0; u < S; ++u) rs[u] = add2(rs[u], w[u + j]);
        const int k = kbs * 4 + j + 1;
        if (k >= kmin && k <= kmax) {
#pragma unroll
            for (int u = 0; u < S; ++u) {
                float r, s;
                unpack2(rs[u], r, s);
                const float den = fmaf(-r, r, r);
                const float t = fabsf(s * fast_rsqrt(den));
                if (t > bt) { bt = t; bk = k; bu = u; }
            }
        }
    }
    out_t = bt;
    out_key = ((uint32_t)bk << 16) | (uint32_t)(tl * S + bu);
}

// ---- the phases of one tile (32 trial frequencies, one per lane), written for a GROUP of warps:
//      `gw` = this warp's index in the group, `gnw` = warps in the group -------------------------

struct TileCtx {
    int nb, nrows, kmin, kmax, n;
    uint32_t G;
    bool force_canon;
    float cw, cy, wx2;
};

__device__ __forceinline__ void zero_bins(uint32_t bins_s, int nb, int gtid, int gthreads)
{
    const int nvec = nb * (kRowBytes / 16);
    for (int i = gtid; i < nvec; i += gthreads)
        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(bins_s + i * 16), "r"(0u) : "memory");
}

// NG groups of 4 consecutive points (group g at shared address pa + g*step) folded at frequency f:
// all loads first, then the phases, then the atomics, so 4*NG points are in flight per warp.
template <int NG>
__device__ __forceinline__ void fold_groups(const TileCtx &c, double f, uint32_t colw, uint32_t pa, uint32_t step,
                                            unsigned int &n_canon)
{
    constexpr int NP = 4 * NG;
    const int nb = c.nb;
    const uint32_t G = c.G;
    uint4 raw[NP];
    unsigned long long pr[NP];
#pragma unroll
    for (int u = 0; u < NP; ++u) raw[u] = lds128(pa + (u >> 2) * step + (u & 3) * 16);
    uint32_t lomin = 0xffffffffu;
#pragma unroll
    for (int u = 0; u < NP; ++u) {
        pr[u] = fast_bin_pos(f, __hiloint2double((int)raw[u].y, (int)raw[u].x), nb, G);
        lomin = min(lomin, (uint32_t)pr[u]);
    }
    if (!c.force_canon && lomin >= 2u * G) {
#pragma unroll
        for (int u = 0; u < NP; ++u) {
            const uint32_t addr = row_addr(colw, (uint32_t)(pr[u] >> 32));
            red_add(addr, raw[u].z);
            red_add(addr + 128, raw[u].w);
        }
    } else {                       // rare: some point sits within G of a bin edge
#pragma unroll
        for (int u = 0; u < NP; ++u) {
            int bin = (int)(pr[u] >> 32);
            if (c.force_canon || (uint32_t)pr[u] < 2u * G) {
                bin = canonical_bin(f, __hiloint2double((int)raw[u].y, (int)raw[u].x), nb);
                ++n_canon;
            }
            const uint32_t addr = colw + bin * kRowBytes;
            red_add(addr, raw[u].z);
            red_add(addr + 128, raw[u].w);
        }
    }
}

// a2 Fold: warp gw takes groups of 4 consecutive points gw, gw+gnw, ...; lane l folds them at its
// frequency f.  During the fold row b holds int32 planes W[b][lane] | Y[b][lane]: lane l always
// hits bank l (and Y sits 128 B after W, one address register), so the native ATOMS.ADD is
// conflict-free by construction.  Four points in flight hide the LDS / DFMA latency.
template <bool PTS_SMEM, int NG = 1>
__device__ __forceinline__ void fold_tile(const TileCtx &c, double f, uint32_t bins_s, uint32_t pts_sa,
                                          const PointRec *pts_g, int lane, int gw, int gnw, unsigned int &n_canon)
{
    const int nb = c.nb;
    const uint32_t G = c.G;
    const bool force_canon = c.force_canon;
    const uint32_t colw = bins_s + lane * 4;       // W plane of this lane's column, row 0
    const int ngroups = c.n >> 2;
    if (PTS_SMEM) {
        const uint32_t pa_end = pts_sa + ngroups * 64, step = gnw * 64;
        uint32_t pa = pts_sa + gw * 64;
        if (NG == 2)
            for (; pa + step < pa_end; pa += 2 * step) fold_groups<2>(c, f, colw, pa, step, n_canon);
        for (; pa < pa_end; pa += step) fold_groups<1>(c, f, colw, pa, step, n_canon);
    } else {
        for (int g = gw; g < ngroups; g += gnw) {
            PointRec p[4];
            int bin[4];
            uint32_t lo[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) p[u] = load_point<false>(pts_g + g * 4 + u);
#pragma unroll
            for (int u = 0; u < 4; ++u) bin[u] = fast_bin(f, p[u].t, nb, G, lo[u]);
            if (force_canon || min(min(lo[0], lo[1]), min(lo[2], lo[3])) < 2u * G) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (force_canon || lo[u] < 2u * G) { bin[u] = canonical_bin(f, p[u].t, nb); ++n_canon; }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t addr = colw + bin[u] * kRowBytes;
                red_add(addr, p[u].qw);
                red_add(addr + 128, (uint32_t)p[u].qy);
            }
        }
    }
    if (gw == ngroups % gnw) {             // the n % 4 points after the last whole group
        for (int i = ngroups * 4; i < c.n; ++i) {
            PointRec p;
            if (PTS_SMEM) {
                const uint4 raw = lds128(pts_sa + i * 16);
                p.t = __hiloint2double((int)raw.y, (int)raw.x); p.qw = raw.z; p.qy = (int32_t)raw.w;
            } else {
                p = load_point<false>(pts_g + i);
            }
            const int bin = fold_bin(f, p.t, nb, G, force_canon, n_canon);
            const uint32_t addr = colw + bin * kRowBytes;
            red_add(addr, p.qw);
            red_add(addr + 128, (uint32_t)p.qy);
        }
    }
}

// fixed point -> fp32 pairs (weight fraction, weighted residual), in place, plus the cyclic
// extension rows nb .. nrows-1.  A warp owns whole rows, so reading both int planes before
// writing the pairs needs only a warp sync.
__device__ __forceinline__ void convert_rows(const TileCtx &c, uint32_t bins_s, int lane, int gw, int gnw)
{
    const int nb = c.nb;
    const int next = c.nrows - nb;                // extension rows
    uint32_t ra = bins_s + gw * kRowBytes + lane * 4;
    if (next <= nb) {                             // every shape but tiny nb with wide boxes
        int j = gw;
        for (; j + gnw < nb; j += 2 * gnw, ra += 2 * gnw * kRowBytes) {     // two rows in flight
            const uint32_t rb = ra + gnw * kRowBytes;
            const uint32_t qw0 = lds32(ra), qw1 = lds32(rb);
            const int32_t qy0 = (int32_t)lds32(ra + 128), qy1 = (int32_t)lds32(rb + 128);
            __syncwarp();
            const uint64_t v0 = pack2((float)qw0 * c.cw, (float)qy0 * c.cy);
            const uint64_t v1 = pack2((float)qw1 * c.cw, (float)qy1 * c.cy);
            const uint32_t wa = ra + lane * 4, wb = rb + lane * 4;
            sts64(wa, v0);
            sts64(wb, v1);
            if (j < next) sts64(wa + nb * kRowBytes, v0);
            if (j + gnw < next) sts64(wb + nb * kRowBytes, v1);
        }
        for (; j < nb; j += gnw, ra += gnw * kRowBytes) {
            const uint32_t qw = lds32(ra);
            const int32_t qy = (int32_t)lds32(ra + 128);
            __syncwarp();
            const uint64_t v = pack2((float)qw * c.cw, (float)qy * c.cy);
            const uint32_t wa = ra + lane * 4;
            sts64(wa, v);
            if (j < next) sts64(wa + nb * kRowBytes, v);
        }
    } else {
        for (int j = gw; j < nb; j += gnw, ra += gnw * kRowBytes) {
            const uint32_t qw = lds32(ra);
            const int32_t qy = (int32_t)lds32(ra + 128);
            __syncwarp();
            const uint64_t v = pack2((float)qw * c.cw, (float)qy * c.cy);
            uint32_t wa = ra + lane * 4;
            sts64(wa, v);
            for (int x = j + nb; x < c.nrows; x += nb) { wa += nb * kRowBytes; sts64(wa, v); }
        }
    }
}

// Outputs of one (curve, frequency).
struct OutPtrs {
    float *sr; uint32_t *ak; float *depth;        // chunk scratch, row of this curve
    float *u_sr; uint16_t *u_start; uint16_t *u_width; float *u_depth;   // user rows or NULL
};

// Merge the per-warp partial results of column `lane`, canonicalise exact ties (R12), recompute
// (r, s) of the chosen box by direct summation and write SR = s^2/den, depth = s/den (IEEE
// division).  The chains below are serial per column, so callers spread the 32 columns over
// several warps.
__device__ __forceinline__ void merge_column(const TileCtx &c, const float2 *rows2, const float *red_v,
                                             const uint32_t *red_key, int nparts, int lane, int q, int nf,
                                             const OutPtrs &o)
{
    const int nb = c.nb, kmin = c.kmin, kmax = c.kmax;
    float bt = red_v[lane];
    uint32_t bkey = red_key[lane];
#pragma unroll 4
    for (int w = 1; w < nparts; ++w) {
        const float v = red_v[w * 32 + lane];
        const uint32_t key = red_key[w * 32 + lane];
        if (v > bt) { bt = v; bkey = key; }
    }
    const Column col{rows2 + lane, nb};
    float bv = bt * bt;
    if (!(bv <= 1.001f * c.wx2 + 1e-30f)) {   // inf / impossible: r == 1.0f box
        careful_search(col, kmin, kmax, bv, bkey);
        bt = bv;
    }
    int bk = (int)(bkey >> 16), ba = (int)(bkey & 0xffffu);
    if (bt > 0.f) canonicalise(col, kmin, ba, bk);
    else { bk = kmin; ba = 0; }
    float r = 0.f, s = 0.f;
    {   // bins in order (as the oracle sums them); rows nb .. repeat rows 0 .., so no wrap; loads 4 ahead
        const float2 *pr = col.col + ba * 32;
        int j = 0;
        for (; j + 4 <= bk; j += 4, pr += 128) {
            const float2 v0 = pr[0], v1 = pr[32], v2 = pr[64], v3 = pr[96];
            r += v0.x; s += v0.y; r += v1.x; s += v1.y; r += v2.x; s += v2.y; r += v3.x; s += v3.y;
        }
        for (; j < bk; ++j, pr += 32) { r += pr[0].x; s += pr[0].y; }
    }
    const float den = fmaf(-r, r, r);
    float sr = 0.f, dp = 0.f;
    if (bt > 0.f && den > 0.f) { sr = (s * s) / den; dp = s / den; }
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

// ---- kernel 1: every warp does every phase, phases separated by CTA barriers.  Used where the
//      double-buffered bins of kernel 2 do not fit shared memory (e.g. nb = 400).  Two CTAs per
//      SM overlap each other's LSU-bound fold and XU-bound box search only by chance. -----------
template <bool PTS_SMEM, int S>
__global__ void __launch_bounds__(kMaxSearchWarps * 32, 2)
search_kernel(const SearchArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nw = nthr >> 5;
    TileCtx c;
    c.nb = a.nb; c.kmin = a.kmin; c.kmax = a.kmax;
    c.nrows = search_rows(a.nb, a.kmax);
    // smem: bins [nrows][256 B] | red_v [nw][32] | red_key [nw][32] | points [n] (if PTS_SMEM)
    float *red_v = reinterpret_cast<float *>(smem_raw + (size_t)c.nrows * kRowBytes);
    uint32_t *red_key = reinterpret_cast<uint32_t *>(red_v + nw * 32);
    PointRec *pts_s = reinterpret_cast<PointRec *>(red_key + nw * 32);
    const float2 *rows2 = reinterpret_cast<const float2 *>(smem_raw);

    const int64_t curve_local = blockIdx.x / a.items_per_curve;
    const int item = blockIdx.x % a.items_per_curve;
    const int64_t cv = a.curve_base + curve_local;
    const int64_t beg = a.offsets[cv];
    c.n = (int)(a.offsets[cv + 1] - beg);
    const CurveMeta meta = a.meta[cv];
    const int ntiles = (a.nf + kTileFreqs - 1) / kTileFreqs;
    const int tile0 = item * a.tiles_per_item;
    const int tile1 = min(tile0 + a.tiles_per_item, ntiles);
    const OutPtrs out = out_rows(a, curve_local, cv);

    if (meta.status != BLS_CURVE_OK) {
        zero_fill_outputs(out, tile0 * kTileFreqs, min(tile1 * kTileFreqs, a.nf), a.kmin, tid, nthr);
        return;
    }

    // ---- a1 Load: the curve becomes resident for every tile of this work item -------------------
    const PointRec *pts_g = a.pts + beg;
    if (PTS_SMEM) {
        const uint4 *src = reinterpret_cast<const uint4 *>(pts_g);
        uint4 *dst = reinterpret_cast<uint4 *>(pts_s);
        for (int i = tid; i < c.n; i += nthr) dst[i] = __ldg(src + i);
    }
    const uint32_t bins_s = smem_u32(smem_raw), pts_sa = smem_u32(pts_s);
    c.force_canon = (a.force_canonical != 0) || (meta.force_canonical != 0);
    c.cw = meta.cw; c.cy = meta.cy; c.wx2 = (float)meta.wx2;
    c.G = (uint32_t)a.nb + 8u;                    // guard band, units of 2^-32 bin
    unsigned int n_canon = 0;

    for (int tile = tile0; tile < tile1; ++tile) {
        const int q0 = tile * kTileFreqs;
        const double f = a.freqs[min(q0 + lane, a.nf - 1)];   // ragged last tile: surplus lanes repeat the last f
        zero_bins(bins_s, c.nb, tid, nthr);
        __syncthreads();
        fold_tile<PTS_SMEM>(c, f, bins_s, pts_sa, pts_g, lane, warp, nw, n_canon);
        __syncthreads();
        convert_rows(c, bins_s, lane, warp, nw);
        __syncthreads();
        // ---- a3/a4 box search: this thread owns start tiles warp, warp+nw, ... of column `lane` --
        {
            float t_best; uint32_t key_best;
            search_column<S>(bins_s + lane * 8, c.nb, c.kmin, c.kmax, warp, nw, t_best, key_best);
            red_v[warp * 32 + lane] = t_best;
            red_key[warp * 32 + lane] = key_best;
        }
        __syncthreads();
        if (warp < 4 && (lane >> 3) == warp)      // 4 warps x 8 columns
            merge_column(c, rows2, red_v, red_key, nw, lane, q0 + lane, a.nf, out);
        __syncthreads();
    }
    count_canonical(a, n_canon, lane);
}

// ---- kernel 2: warp-specialised, double-buffered.  The fold is bound by the LSU pipe (shared
//      atomics + point broadcasts), the box search by the XU pipe (one MUFU.RSQ per box): run
//      them CONCURRENTLY on different warps so the SM is busy for max(fold, search), not their
//      sum.  "Fold warps" zero / fold / convert tile i+1 (and merge tile i-1) into one bin buffer
//      while "search warps" walk the boxes of tile i in the other.  Hand-off by named barriers
//      (bar.arrive by the producer side, bar.sync by the consumer side). --------------------------
__device__ __forceinline__ void named_sync(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void named_arrive(int id, int count)
{
    __threadfence_block();
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}
enum { kBarFull0 = 1, kBarFull1 = 2, kBarDone0 = 3, kBarDone1 = 4, kBarFoldGroup = 5 };

template <bool PTS_SMEM, int S>
__global__ void __launch_bounds__(kWsMaxWarps * 32, 1)
search_ws_kernel(const SearchArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x;
    const int nsw = a.search_warps, nfw = (nthr >> 5) - nsw;      // search warps come first
    TileCtx c;
    c.nb = a.nb; c.kmin = a.kmin; c.kmax = a.kmax;
    c.nrows = search_rows(a.nb, a.kmax);
    // smem: bins[2] [nrows][256 B] | red_v[2] [nsw][32] | red_key[2] [nsw][32] | points [n]
    const size_t buf_bytes = (size_t)c.nrows * kRowBytes;
    float *red_v = reinterpret_cast<float *>(smem_raw + 2 * buf_bytes);
    uint32_t *red_key = reinterpret_cast<uint32_t *>(red_v + 2 * nsw * 32);
    PointRec *pts_s = reinterpret_cast<PointRec *>(red_key + 2 * nsw * 32);

    const int64_t curve_local = blockIdx.x / a.items_per_curve;
    const int item = blockIdx.x % a.items_per_curve;
    const int64_t cv = a.curve_base + curve_local;
    const int64_t beg = a.offsets[cv];
    c.n = (int)(a.offsets[cv + 1] - beg);
    const CurveMeta meta = a.meta[cv];
    const int ntiles = (a.nf + kTileFreqs - 1) / kTileFreqs;
    const int tile0 = item * a.tiles_per_item;
    const int tile1 = min(tile0 + a.tiles_per_item, ntiles);
    const OutPtrs out = out_rows(a, curve_local, cv);

    if (meta.status != BLS_CURVE_OK) {
        zero_fill_outputs(out, tile0 * kTileFreqs, min(tile1 * kTileFreqs, a.nf), a.kmin, tid, nthr);
        return;
    }

    const PointRec *pts_g = a.pts + beg;
    if (PTS_SMEM) {                               // a1 Load, by all warps
        const uint4 *src = reinterpret_cast<const uint4 *>(pts_g);
        uint4 *dst = reinterpret_cast<uint4 *>(pts_s);
        for (int i = tid; i < c.n; i += nthr) dst[i] = __ldg(src + i);
    }
    __syncthreads();
    const uint32_t bins_s = smem_u32(smem_raw), pts_sa = smem_u32(pts_s);
    c.force_canon = (a.force_canonical != 0) || (meta.force_canonical != 0);
    c.cw = meta.cw; c.cy = meta.cy; c.wx2 = (float)meta.wx2;
    c.G = (uint32_t)a.nb + 8u;

    if (warp < nsw) {
        // ================= search warps: a3/a4 only =================
        for (int tile = tile0, it = 0; tile < tile1; ++tile, ++it) {
            const int b = it & 1;
            named_sync(kBarFull0 + b, nthr);                      // buffer b holds tile's fp32 rows
            float t_best; uint32_t key_best;
            search_column<S>(bins_s + b * (uint32_t)buf_bytes + lane * 8, c.nb, c.kmin, c.kmax, warp, nsw, t_best, key_best);
            red_v[(b * nsw + warp) * 32 + lane] = t_best;
            red_key[(b * nsw + warp) * 32 + lane] = key_best;
            named_arrive(kBarDone0 + b, nthr);                    // done with buffer b
        }
    } else {
        // ================= fold warps: zero, a2 fold, convert, merge =================
        const int gw = warp - nsw, gtid = tid - nsw * 32, gthreads = nfw * 32;
        unsigned int n_canon = 0;
        auto merge = [&](int tile, int b) {
            const int mw = min(nfw, 4), per = (32 + mw - 1) / mw;  // mw warps x ceil(32/mw) columns
            if (gw < mw && lane / per == gw)
                merge_column(c, reinterpret_cast<const float2 *>(smem_raw + b * buf_bytes), red_v + b * nsw * 32,
                             red_key + b * nsw * 32, nsw, lane, tile * kTileFreqs + lane, a.nf, out);
        };
        for (int tile = tile0, it = 0; tile < tile1; ++tile, ++it) {
            const int b = it & 1;
            const uint32_t buf = bins_s + b * (uint32_t)buf_bytes;
            if (it >= 2) {                                        // tile-2 used this buffer: wait, then merge it
                named_sync(kBarDone0 + b, nthr);
                merge(tile - 2, b);
                named_sync(kBarFoldGroup, gthreads);
            }
            const double f = a.freqs[min(tile * kTileFreqs + lane, a.nf - 1)];
            zero_bins(buf, c.nb, gtid, gthreads);
            named_sync(kBarFoldGroup, gthreads);
            fold_tile<PTS_SMEM>(c, f, buf, pts_sa, pts_g, lane, gw, nfw, n_canon);
            named_sync(kBarFoldGroup, gthreads);
            convert_rows(c, buf, lane, gw, nfw);
            named_arrive(kBarFull0 + b, nthr);
        }
        // drain: the last (up to) two tiles
        const int nt = tile1 - tile0;
        for (int it = max(nt - 2, 0); it < nt; ++it) {
            const int b = it & 1;
            named_sync(kBarDone0 + b, nthr);
            merge(tile0 + it, b);
        }
        count_canonical(a, n_canon, lane);
    }
}

// ---- kernel 3: one warp per tile.  For small shapes (C4: 200 epochs, 64 bins) a tile is a few
//      thousand instructions and the hand-offs of kernels 1/2 cost more than the work.  Here every
//      warp owns private bins and runs zero / fold / convert / search / merge of its own tiles with
//      warp syncs only; warps of an SM sit in different phases, so the LSU-bound fold of one overlaps
//      the XU-bound search of another without any CTA-level barrier. ------------------------------
template <bool PTS_SMEM, int S>
__global__ void __launch_bounds__(kWtWarps * 32, 2)
search_wt_kernel(const SearchArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nw = nthr >> 5;
    TileCtx c;
    c.nb = a.nb; c.kmin = a.kmin; c.kmax = a.kmax;
    c.nrows = search_rows(a.nb, a.kmax);
    // smem: per warp { bins [nrows][256 B] | red_v [32] | red_key [32] } ... | points [n]
    const size_t per_warp = (size_t)c.nrows * kRowBytes + 256;
    unsigned char *mine = smem_raw + warp * per_warp;
    float *red_v = reinterpret_cast<float *>(mine + (size_t)c.nrows * kRowBytes);
    uint32_t *red_key = reinterpret_cast<uint32_t *>(red_v + 32);
    PointRec *pts_s = reinterpret_cast<PointRec *>(smem_raw + nw * per_warp);

    const int64_t curve_local = blockIdx.x / a.items_per_curve;
    const int item = blockIdx.x % a.items_per_curve;
    const int64_t cv = a.curve_base + curve_local;
    const int64_t beg = a.offsets[cv];
    c.n = (int)(a.offsets[cv + 1] - beg);
    const CurveMeta meta = a.meta[cv];
    const int ntiles = (a.nf + kTileFreqs - 1) / kTileFreqs;
    const int tile0 = item * a.tiles_per_item;
    const int tile1 = min(tile0 + a.tiles_per_item, ntiles);
    const OutPtrs out = out_rows(a, curve_local, cv);

    if (meta.status != BLS_CURVE_OK) {
        zero_fill_outputs(out, tile0 * kTileFreqs, min(tile1 * kTileFreqs, a.nf), a.kmin, tid, nthr);
        return;
    }
    const PointRec *pts_g = a.pts + beg;
    if (PTS_SMEM) {
        const uint4 *src = reinterpret_cast<const uint4 *>(pts_g);
        uint4 *dst = reinterpret_cast<uint4 *>(pts_s);
        for (int i = tid; i < c.n; i += nthr) dst[i] = __ldg(src + i);
    }
    __syncthreads();                              // the only CTA barrier
    const uint32_t buf = smem_u32(mine), pts_sa = smem_u32(pts_s);
    c.force_canon = (a.force_canonical != 0) || (meta.force_canonical != 0);
    c.cw = meta.cw; c.cy = meta.cy; c.wx2 = (float)meta.wx2;
    c.G = (uint32_t)a.nb + 8u;
    unsigned int n_canon = 0;

    for (int tile = tile0 + warp; tile < tile1; tile += nw) {
        const int q0 = tile * kTileFreqs;
        const double f = a.freqs[min(q0 + lane, a.nf - 1)];
        zero_bins(buf, c.nb, lane, 32);
        __syncwarp();
        fold_tile<PTS_SMEM, 2>(c, f, buf, pts_sa, pts_g, lane, 0, 1, n_canon);
        __syncwarp();
        convert_rows(c, buf, lane, 0, 1);
        __syncwarp();
        float t_best; uint32_t key_best;
        search_column<S>(buf + lane * 8, c.nb, c.kmin, c.kmax, 0, 1, t_best, key_best);
        red_v[lane] = t_best;
        red_key[lane] = key_best;
        __syncwarp();
        merge_column(c, reinterpret_cast<const float2 *>(mine), red_v, red_key, 1, lane, q0 + lane, a.nf, out);
        __syncwarp();
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
    const void *fns[] = {(const void *)search_kernel<true, 4>,    (const void *)search_kernel<false, 4>,
                         (const void *)search_kernel<true, 5>,    (const void *)search_kernel<false, 5>,
                         (const void *)search_ws_kernel<true, 4>, (const void *)search_ws_kernel<false, 4>,
                         (const void *)search_ws_kernel<true, 5>, (const void *)search_ws_kernel<false, 5>,
                         (const void *)search_wt_kernel<true, 4>, (const void *)search_wt_kernel<false, 4>,
                         (const void *)search_wt_kernel<true, 5>, (const void *)search_wt_kernel<false, 5>};
    for (const void *f : fns) {
        cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_search(const SearchArgs &a, int64_t chunk_curves, size_t smem, cudaStream_t st)
{
    const int64_t grid = chunk_curves * (int64_t)a.items_per_curve;
    if (grid <= 0) return cudaSuccess;
    if (grid > 2147483647LL) return cudaErrorInvalidConfiguration;
    const unsigned g = (unsigned)grid;
#define BLS_LAUNCH(K)                                                                   \
    do {                                                                                \
        if (a.starts_per_thread == 5) {                                                 \
            if (a.pts_in_smem) K<true, 5><<<g, a.threads, smem, st>>>(a);               \
            else K<false, 5><<<g, a.threads, smem, st>>>(a);                            \
        } else {                                                                        \
            if (a.pts_in_smem) K<true, 4><<<g, a.threads, smem, st>>>(a);               \
            else K<false, 4><<<g, a.threads, smem, st>>>(a);                            \
        }                                                                               \
    } while (0)
    if (a.kernel == 3) BLS_LAUNCH(search_wt_kernel);
    else if (a.kernel == 2) BLS_LAUNCH(search_ws_kernel);
    else BLS_LAUNCH(search_kernel);
#undef BLS_LAUNCH
    return cudaGetLastError();
}

}  // namespace bls
