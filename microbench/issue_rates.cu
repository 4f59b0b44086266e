// Issue-rate microbenchmarks behind the "stated roofline" of the BLS search kernel (DESIGN.md
// "Roofline").  The fold and box-search stages are bound by per-SM
// issue rates, not by HBM or tensor throughput, so the denominators of bench.py's roofline are
// measured here, on the box the bench runs on, in lane-operations per clock per SM:
//
//   atoms_add_cf    native 32-bit shared ATOMS.ADD, lane l -> bank l (the fold's access pattern)
//   atoms_add_rand  same, pseudo-random banks (what a lane = point layout would see)
//   lds128_bcast    LDS.128 at a warp-uniform address (how the fold reads one point)
//   lds32_cf        LDS.32, lane l -> bank l (how the box search reads a bin row)
//   mufu_rsq        MUFU.RSQ (one per box in the search)
//   fadd / fadd2    FADD vs the packed FADD2 (add.rn.f32x2)
//   ffma / ffma2    FFMA vs FFMA2
//   fmnmx3          3-input FMNMX
//   dfma            fp64 FMA (the fold's phase)
//   imad_wide       IMAD.WIDE.U32 (phase -> bin)
//   fold_mix        the fold's per-point-fold instruction mix (LDS.128 bcast amortised over 32 lanes,
//                   DFMA, IMAD.WIDE, 2 x ATOMS.ADD)
//   box_mix         the search's per-box mix (2 FADD, FFMA, MUFU.RSQ, FMUL, 1/2 FMNMX3)
//   fold_mix_nb64, fold_field_s3, fold_field_s7, fold_field_stars
//                   row f2 (field-shared cadence): the fold when the stars of a pointing share their epochs, so that
//                   one bin index per (epoch, frequency) serves several stars; two designs against today's mix
//
// One CTA of 1024 threads per SM; cycles are clock64() deltas between two __syncthreads(), so the
// numbers do not depend on the SM clock.  Prints one line per test: median and best over SMs.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -o issue_rates issue_rates.cu && ./issue_rates
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>
#include <vector>

constexpr int kThreads = 1024;
constexpr int kIters = 2048;

enum Test { ATOMS_CF, ATOMS_RAND, LDS128_BCAST, LDS32_CF, MUFU_RSQ, FADD, FADD2, FFMA, FFMA2, FMNMX3, DFMA, IMAD_WIDE,
            FOLD_MIX, BOX_MIX, BOX_MIX2, ATOMS_CF2, LDS64_BCAST, LDS32_BCAST, LDS64_CF, I2FP, MUFU_I2FP, FMUL2, BOX_PACKED, BOX_PACKED_CVT, BOX_PACKED_THRESH, BOX_PACKED_PAIRDIV, FFMA2_ALU, FFMA2_MUFU, FFMA_ALU, MUFU_ALU,
            FOLD_MIX64, FOLD_FIELD_S3, FOLD_FIELD_S7, FOLD_FIELD_STARS, N_TESTS };
static const char *kNames[N_TESTS] = {"atoms_add_cf", "atoms_add_rand", "lds128_bcast", "lds32_cf", "mufu_rsq", "fadd",
                                      "fadd2", "ffma", "ffma2", "fmnmx3", "dfma", "imad_wide", "fold_mix", "box_mix",
                                      "box_mix_fadd2", "atoms_add_cf_min", "lds64_bcast", "lds32_bcast", "lds64_cf", "i2fp",
                                      "mufu_plus_i2fp", "fmul2", "box_packed", "box_packed_cvt", "box_nodiv_thresh", "box_nodiv_pair", "ffma2_plus_alu", "ffma2_plus_mufu", "ffma_plus_alu", "mufu_plus_alu",
                                      "fold_mix_nb64", "fold_field_s3", "fold_field_s7", "fold_field_stars"};
// lane-operations each thread performs per inner iteration (what the rate is quoted in)
static const double kOpsPerIter[N_TESTS] = {8, 8, 8, 8, 8, 8, 8, 8, 8, 8, 8, 8, 4, 8, 8, 8, 8, 8, 8, 8, 8, 8, 14, 14, 14, 12, 16, 12, 16, 12, 4, 12, 28, 4};
static const char *kUnit[N_TESTS] = {"ATOMS lane-ops", "ATOMS lane-ops", "LDS.128 lane-loads", "LDS.32 lane-loads",
                                     "MUFU lane-ops", "FADD lane-ops", "FADD2 lane-instr (2 adds each)", "FFMA lane-ops",
                                     "FFMA2 lane-instr (2 fmas each)", "FMNMX3 lane-ops (+1/8 FADD)", "DFMA lane-ops",
                                     "IMAD.WIDE lane-ops", "point-folds", "boxes", "boxes", "ATOMS lane-ops", "LDS.64 lane-loads", "LDS.32 lane-loads", "LDS.64 lane-loads",
                                     "I2FP lane-ops", "MUFU lane-ops (each with one I2FP beside it)", "FMUL2 lane-instr (2 muls each)",
                                     "boxes (packed f32x2 search mix, rows already fp32)", "boxes (packed f32x2 search mix, int rows converted on the fly)",
                                     "boxes (no division: excess s^2 - B r(1-r) against a threshold B, FMNMX3; finds no argmax by itself)",
                                     "boxes (division-free compare of two boxes: cross-multiplied, one MUFU.RCP per two boxes)",
                                     "warp-instr lanes (8 FFMA2 + 8 LOP3 per iteration: does a packed instruction hold the issue port for 2 clocks?)",
                                     "warp-instr lanes (8 FFMA2 + 4 MUFU.RSQ per iteration)",
                                     "warp-instr lanes (8 FFMA + 8 LOP3 per iteration)",
                                     "warp-instr lanes (4 MUFU.RSQ + 8 LOP3 per iteration)",
                                     "point-folds (fold_mix at nb = 64: the baseline of the three field lines)",
                                     "point-folds (f2, lanes = frequencies, 3 stars per epoch read: bin index once per (epoch, frequency), 2 LDS.128 + 6 ATOMS per 3 stars)",
                                     "point-folds (f2, lanes = frequencies, 7 stars per epoch read: 4 LDS.128 + 14 ATOMS per 7 stars)",
                                     "point-folds (f2 as VERDICT r2 #6 words it, lanes = stars: warp-uniform phase from an LDS.64 broadcast of t, per-lane LDS.64 of (qw, qy), 2 ATOMS)"};

__device__ __forceinline__ float rsq(float x) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ unsigned long long add2(unsigned long long a, unsigned long long b)
{ unsigned long long c; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(c) : "l"(a), "l"(b)); return c; }
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c)
{ unsigned long long d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b)
{ unsigned long long c; asm volatile("mul.rn.f32x2 %0, %1, %2;" : "=l"(c) : "l"(a), "l"(b)); return c; }
__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{ unsigned long long v; asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(lo), "f"(hi)); return v; }
__device__ __forceinline__ void unpack2(unsigned long long v, float &lo, float &hi)
{ asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ float fmax3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }

template <int T>
__global__ void __launch_bounds__(kThreads, 1) bench(long long *cycles, float *sink, int nb)
{
    extern __shared__ __align__(16) uint32_t sm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < nb * 64 + 4096; i += kThreads) sm[i] = (uint32_t)i * 2654435761u >> 20;
    __syncthreads();
    float f0 = 1.0f + tid * 1e-3f, f1 = 1.5f, f2 = 0.25f, f3 = 0.75f, f4 = 1.25f, f5 = 2.f, f6 = 3.f, f7 = 0.5f;
    unsigned long long p0 = 0x3f8000003f800000ull, p1 = p0 + tid, p2 = p0 + 7, p3 = p0 + 11, p4 = p0, p5 = p1, p6 = p2, p7 = p3;
    double d0 = 1.0 + tid, d1 = 2.0, d2 = 3.0, d3 = 4.0, d4 = 5.0, d5 = 6.0, d6 = 7.0, d7 = 8.0;
    const double fr = 0.3712345 + 1e-6 * lane, dc = 1e-3 * (1 + lane), frw = 0.3712345 + 1e-3 * warp;
    float fc = 1e-3f * (1 + lane);
    const float fm = 0.999f + 1e-6f * lane;
    const unsigned long long pc = 0x3a83126f3a83126full + lane, pm = 0x3f7fbe773f7fbe77ull + lane;
    uint32_t x = tid * 747796405u + 2891336453u;
    unsigned long long acc = 0;
    unsigned long long q[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) q[u] = ((unsigned long long)x << 20) + u * 77777ull;
    uint32_t *pts = sm + nb * 64;            // 4096 words of "points" for the broadcast loads
    long long t0 = 0, t1 = 0;
    __syncthreads();
    t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
        if (T == ATOMS_CF) {
#pragma unroll
            for (int u = 0; u < 8; ++u) { x = x * 1664525u + 1013904223u; atomicAdd(&sm[((x >> 8) & 127) * 64 + (u & 1) * 32 + lane], x); }
        } else if (T == ATOMS_CF2) {
            uint32_t *b = sm + ((it * 8) & 63) * 64 + lane;
#pragma unroll
            for (int u = 0; u < 8; ++u) atomicAdd(b + u * 64 * 9 + (u & 1) * 32, x);
        } else if (T == LDS64_BCAST) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint2 v = *reinterpret_cast<const uint2 *>(pts + (((it * 8 + u) * 37 + warp * 4) & 1023) * 4);
                acc += v.x ^ v.y;
            }
        } else if (T == LDS32_BCAST) {
#pragma unroll
            for (int u = 0; u < 8; ++u) acc += pts[(((it * 8 + u) * 37 + warp * 4) & 1023) * 4];
        } else if (T == LDS64_CF) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint2 v = *reinterpret_cast<const uint2 *>(sm + (((it * 8 + u) * 5 + warp) & 127) * 64 + lane * 2);
                acc += v.x ^ v.y;
            }
        } else if (T == ATOMS_RAND) {
#pragma unroll
            for (int u = 0; u < 8; ++u) { x = x * 1664525u + 1013904223u; atomicAdd(&sm[(x >> 8) & 8191], x); }
        } else if (T == LDS128_BCAST) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint4 v = *reinterpret_cast<const uint4 *>(pts + (((it * 8 + u) * 37 + warp * 4) & 1023) * 4);
                acc += v.x ^ v.y ^ v.z ^ v.w;
            }
        } else if (T == LDS32_CF) {
#pragma unroll
            for (int u = 0; u < 8; ++u) acc += sm[(((it * 8 + u) * 5 + warp) & 127) * 64 + lane];
        } else if (T == MUFU_RSQ) {
            f0 = rsq(f0); f1 = rsq(f1); f2 = rsq(f2); f3 = rsq(f3); f4 = rsq(f4); f5 = rsq(f5); f6 = rsq(f6); f7 = rsq(f7);
        } else if (T == FADD) {
            f0 += fc; f1 += fc; f2 += fc; f3 += fc; f4 += fc; f5 += fc; f6 += fc; f7 += fc;
        } else if (T == FADD2) {
            p0 = add2(p0, pc); p1 = add2(p1, pc); p2 = add2(p2, pc); p3 = add2(p3, pc);
            p4 = add2(p4, pc); p5 = add2(p5, pc); p6 = add2(p6, pc); p7 = add2(p7, pc);
        } else if (T == FFMA) {
            f0 = fmaf(f0, fm, fc); f1 = fmaf(f1, fm, fc); f2 = fmaf(f2, fm, fc); f3 = fmaf(f3, fm, fc);
            f4 = fmaf(f4, fm, fc); f5 = fmaf(f5, fm, fc); f6 = fmaf(f6, fm, fc); f7 = fmaf(f7, fm, fc);
        } else if (T == FFMA2) {
            p0 = fma2(p0, pm, pc); p1 = fma2(p1, pm, pc); p2 = fma2(p2, pm, pc); p3 = fma2(p3, pm, pc);
            p4 = fma2(p4, pm, pc); p5 = fma2(p5, pm, pc); p6 = fma2(p6, pm, pc); p7 = fma2(p7, pm, pc);
        } else if (T == FMNMX3) {
            f0 = fmax3(f0, fc, fm); f1 = fmax3(f1, fm, fc); f2 = fmax3(f2, fc, fm); f3 = fmax3(f3, fm, fc);
            fc += 1.0f; f4 = fmax3(f4, fc, fm); f5 = fmax3(f5, fm, fc); f6 = fmax3(f6, fc, fm); f7 = fmax3(f7, fm, fc);
        } else if (T == DFMA) {
            d0 = fma(d0, fr, dc); d1 = fma(d1, fr, dc); d2 = fma(d2, fr, dc); d3 = fma(d3, fr, dc);
            d4 = fma(d4, fr, dc); d5 = fma(d5, fr, dc); d6 = fma(d6, fr, dc); d7 = fma(d7, fr, dc);
        } else if (T == IMAD_WIDE) {
#pragma unroll
            for (int u = 0; u < 8; ++u) { q[u] = (unsigned long long)(uint32_t)(q[u] >> 32) * (uint32_t)nb + q[u]; }
        } else if (T == FOLD_FIELD_S3 || T == FOLD_FIELD_S7) {
            // Row f2 with lanes = frequencies: S stars of a field share their epochs, so one phase / bin index per
            // (epoch, frequency) serves S stars, each with its own [64 bins][W | Y][32 lanes] buffer (16 KB apart: an
            // immediate offset).  Epoch record: (t fp64, qw0, qy0), then (qw, qy) pairs of the other stars, 16 B each.
            // 4 epochs per iteration.
            constexpr int S = T == FOLD_FIELD_S3 ? 3 : 7;
            constexpr int REC = (S + 1) / 2;            // LDS.128 per epoch
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint4 *rec = reinterpret_cast<const uint4 *>(pts + ((((it * 4 + u) * 8 + warp) * REC) & 1020) * 4);
                const uint4 v = rec[0];
                const double t = __hiloint2double((int)(v.y & 0xfffffu) | 0x40000000, (int)v.x);
                const double y = fma(fr, t, 1572864.0);
                const unsigned long long pr = (unsigned long long)(uint32_t)__double2loint(y) * 64u;
                uint32_t *b = &sm[(int)(pr >> 32) * 64 + lane];
                atomicAdd(b, v.z);
                atomicAdd(b + 32, v.w + (uint32_t)pr);
#pragma unroll
                for (int r = 1; r < REC; ++r) {
                    const uint4 w = rec[r];
                    atomicAdd(b + (2 * r - 1) * 4096, w.x);
                    atomicAdd(b + (2 * r - 1) * 4096 + 32, w.y);
                    atomicAdd(b + (2 * r) * 4096, w.z);
                    atomicAdd(b + (2 * r) * 4096 + 32, w.w);
                }
            }
        } else if (T == FOLD_FIELD_STARS) {
            // Row f2 with lanes = stars: the warp folds ONE frequency for 32 stars.  Per epoch: t from an LDS.64
            // broadcast, the phase and bin index computed identically by every lane (warp-uniform), the star's
            // (qw, qy) from a conflict-free per-lane LDS.64 of the [epoch][32 stars] tile, 2 ATOMS into the warp's own
            // columns bins[bin][W | Y][star].  4 epochs per iteration; the tile is the 64-epoch "points" area.
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int e = ((it * 4 + u) * 8 + warp) & 63;
                const uint2 tt = *reinterpret_cast<const uint2 *>(sm + (e & 31) * 2);
                const double t = __hiloint2double((int)(tt.y & 0xfffffu) | 0x40000000, (int)tt.x);
                const double y = fma(frw, t, 1572864.0);
                const unsigned long long pr = (unsigned long long)(uint32_t)__double2loint(y) * 64u;
                const uint2 v = *reinterpret_cast<const uint2 *>(pts + e * 64 + lane * 2);
                uint32_t *b = &sm[(int)(pr >> 32) * 64 + lane];
                atomicAdd(b, v.x);
                atomicAdd(b + 32, v.y + (uint32_t)pr);
            }
        } else if (T == FOLD_MIX || T == FOLD_MIX64) {
            // 4 points per iteration: LDS.128 broadcast, DFMA with the magic constant, IMAD.WIDE, 2 ATOMS.ADD
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint4 v = *reinterpret_cast<const uint4 *>(pts + (((it * 4 + u) * 8 + warp) & 1023) * 4);
                const double t = __hiloint2double((int)(v.y & 0xfffffu) | 0x40000000, (int)v.x);
                const double y = fma(fr, t, 1572864.0);
                const unsigned long long pr = (unsigned long long)(uint32_t)__double2loint(y) * (uint32_t)nb;
                const int bin = (int)(pr >> 32);
                atomicAdd(&sm[bin * 64 + lane], v.z);
                atomicAdd(&sm[bin * 64 + 32 + lane], v.w + (uint32_t)pr);
            }
        } else if (T == BOX_MIX) {
            // 8 boxes: running sums of (r, s), den = r - r^2, t = |s| * rsqrt(den), max
            const float w = __uint_as_float(sm[(it % nb) * 64 + lane]) * 1e-12f, y = w * 0.5f;
            f0 += w; f1 += y; { float t = fabsf(f1) * rsq(fmaf(-f0, f0, f0)); float w2 = f0 + w, y2 = f1 + y;
            float t2 = fabsf(y2) * rsq(fmaf(-w2, w2, w2)); f7 = fmax3(f7, t, t2); f0 = w2; f1 = y2; }
            f2 += w; f3 += y; { float t = fabsf(f3) * rsq(fmaf(-f2, f2, f2)); float w2 = f2 + w, y2 = f3 + y;
            float t2 = fabsf(y2) * rsq(fmaf(-w2, w2, w2)); f7 = fmax3(f7, t, t2); f2 = w2; f3 = y2; }
            f4 += w; f5 += y; { float t = fabsf(f5) * rsq(fmaf(-f4, f4, f4)); float w2 = f4 + w, y2 = f5 + y;
            float t2 = fabsf(y2) * rsq(fmaf(-w2, w2, w2)); f6 = fmax3(f6, t, t2); f4 = w2; f5 = y2; }
            p0 = add2(p0, p1); p0 = add2(p0, p1);   // stand-ins for the 4th start: keeps the mix at 8 boxes
            { float r = __uint_as_float((uint32_t)p0), s = __uint_as_float((uint32_t)(p0 >> 32));
              float t = fabsf(s) * rsq(fmaf(-r, r, r)); float t2 = fabsf(s + y) * rsq(fmaf(-(r + w), r + w, r + w)); f6 = fmax3(f6, t, t2); }
        } else if (T == I2FP) {
            f0 = __int2float_rn(__float_as_int(f0)); f1 = __int2float_rn(__float_as_int(f1)); f2 = __int2float_rn(__float_as_int(f2));
            f3 = __int2float_rn(__float_as_int(f3)); f4 = __int2float_rn(__float_as_int(f4)); f5 = __int2float_rn(__float_as_int(f5));
            f6 = __int2float_rn(__float_as_int(f6)); f7 = __int2float_rn(__float_as_int(f7));
        } else if (T == MUFU_I2FP) {
            f0 = rsq(__int2float_rn(__float_as_int(f0))); f1 = rsq(__int2float_rn(__float_as_int(f1)));
            f2 = rsq(__int2float_rn(__float_as_int(f2))); f3 = rsq(__int2float_rn(__float_as_int(f3)));
            f4 = rsq(__int2float_rn(__float_as_int(f4))); f5 = rsq(__int2float_rn(__float_as_int(f5)));
            f6 = rsq(__int2float_rn(__float_as_int(f6))); f7 = rsq(__int2float_rn(__float_as_int(f7)));
        } else if (T == FMUL2) {
            p0 = mul2(p0, pm); p1 = mul2(p1, pm); p2 = mul2(p2, pm); p3 = mul2(p3, pm);
            p4 = mul2(p4, pm); p5 = mul2(p5, pm); p6 = mul2(p6, pm); p7 = mul2(p7, pm);
        } else if (T == BOX_PACKED || T == BOX_PACKED_CVT) {
            // one bin row -> 7 starts x 2 frequencies = 14 boxes: per box pair FFMA2 (n -= W c), FADD2, FFMA2 (n^2 + n),
            // 2 MUFU.RSQ, FMUL2, and one FMNMX3 per two box pairs and frequency
            const uint2 wi = *reinterpret_cast<const uint2 *>(sm + (it % nb) * 64 + (lane & 15) * 2);
            const uint2 yi = *reinterpret_cast<const uint2 *>(sm + (it % nb) * 64 + 32 + (lane & 15) * 2);
            unsigned long long W, Y;
            if (T == BOX_PACKED_CVT) {
                W = pack2(__uint2float_rn(wi.x), __uint2float_rn(wi.y));
                Y = pack2(__int2float_rn((int)yi.x), __int2float_rn((int)yi.y));
            } else {
                W = ((unsigned long long)(wi.y & 0x3fffffffu) << 32) | (wi.x & 0x3fffffffu);
                Y = ((unsigned long long)(yi.y & 0x3fffffffu) << 32) | (yi.x & 0x3fffffffu);
            }
            unsigned long long *rn = q;                 // q[0..6] = n, p0..p6 = s
            unsigned long long rs[7] = {p0, p1, p2, p3, p4, p5, p6};
#pragma unroll
            for (int u = 0; u < 7; ++u) {
                rn[u] = fma2(W, pm, rn[u]);
                rs[u] = add2(rs[u], Y);
                const unsigned long long d = fma2(rn[u], rn[u], rn[u]);
                float d0, d1; unpack2(d, d0, d1);
                const unsigned long long t = mul2(rs[u], pack2(rsq(fabsf(d0)), rsq(fabsf(d1))));
                float t0, t1; unpack2(t, t0, t1);
                f6 = fmaxf(f6, fabsf(t0)); f7 = fmaxf(f7, fabsf(t1));
            }
            p0 = rs[0]; p1 = rs[1]; p2 = rs[2]; p3 = rs[3]; p4 = rs[4]; p5 = rs[5]; p6 = rs[6];
        } else if (T == BOX_PACKED_THRESH) {
            // DESIGN.md section 7, "division-free evaluate", form 1: per box pair FFMA2, FADD2, FFMA2 (n^2 + n), FMUL2 (s^2),
            // FFMA2 (s^2 - B r(1-r)), and one FMNMX3 per box pair: no MUFU at all.  It only says whether a box beats the
            // threshold B; the argmax needs a second pass over the groups that did.
            const uint2 wi = *reinterpret_cast<const uint2 *>(sm + (it % nb) * 64 + (lane & 15) * 2);
            const uint2 yi = *reinterpret_cast<const uint2 *>(sm + (it % nb) * 64 + 32 + (lane & 15) * 2);
            const unsigned long long W = pack2(__uint2float_rn(wi.x), __uint2float_rn(wi.y));
            const unsigned long long Y = pack2(__int2float_rn((int)yi.x), __int2float_rn((int)yi.y));
            unsigned long long *rn = q;
            unsigned long long rs[7] = {p0, p1, p2, p3, p4, p5, p6};
#pragma unroll
            for (int u = 0; u < 7; ++u) {
                rn[u] = fma2(W, pm, rn[u]);
                rs[u] = add2(rs[u], Y);
                const unsigned long long d = fma2(rn[u], rn[u], rn[u]);
                const unsigned long long e = fma2(p7, d, mul2(rs[u], rs[u]));
                float e0, e1; unpack2(e, e0, e1);
                f6 = fmax3(f6, e0, e1);
            }
            p0 = rs[0]; p1 = rs[1]; p2 = rs[2]; p3 = rs[3]; p4 = rs[4]; p5 = rs[5]; p6 = rs[6];
        } else if (T == BOX_PACKED_PAIRDIV) {
            // form 2: boxes A, B of the same frequency share one reciprocal: SR_A = s_A^2 d_B / (d_A d_B).  Per two box
            // pairs (4 boxes): 2 FFMA2 + 2 FADD2 + 2 FFMA2 (sums, d), FMUL2 (d_A d_B), 2 FMUL2 (s^2), 2 FMUL2 (cross),
            // 2 MUFU.RCP, 2 FMUL2, 2 FMNMX3 = 17 instructions
            const uint2 wi = *reinterpret_cast<const uint2 *>(sm + (it % nb) * 64 + (lane & 15) * 2);
            const uint2 yi = *reinterpret_cast<const uint2 *>(sm + (it % nb) * 64 + 32 + (lane & 15) * 2);
            const unsigned long long W = pack2(__uint2float_rn(wi.x), __uint2float_rn(wi.y));
            const unsigned long long Y = pack2(__int2float_rn((int)yi.x), __int2float_rn((int)yi.y));
            unsigned long long *rn = q;
            unsigned long long rs[6] = {p0, p1, p2, p3, p4, p5};
#pragma unroll
            for (int u = 0; u < 6; u += 2) {
                rn[u] = fma2(W, pm, rn[u]); rn[u + 1] = fma2(W, pm, rn[u + 1]);
                rs[u] = add2(rs[u], Y); rs[u + 1] = add2(rs[u + 1], Y);
                const unsigned long long dA = fma2(rn[u], rn[u], rn[u]), dB = fma2(rn[u + 1], rn[u + 1], rn[u + 1]);
                const unsigned long long P = mul2(dA, dB);
                const unsigned long long xA = mul2(mul2(rs[u], rs[u]), dB), xB = mul2(mul2(rs[u + 1], rs[u + 1]), dA);
                float P0, P1; unpack2(P, P0, P1);
                float i0, i1;
                asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(i0) : "f"(P0));
                asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(i1) : "f"(P1));
                const unsigned long long inv = pack2(i0, i1);
                float a0, a1, b0, b1;
                unpack2(mul2(xA, inv), a0, a1); unpack2(mul2(xB, inv), b0, b1);
                f6 = fmax3(f6, a0, b0); f7 = fmax3(f7, a1, b1);
            }
            p0 = rs[0]; p1 = rs[1]; p2 = rs[2]; p3 = rs[3]; p4 = rs[4]; p5 = rs[5];
        } else if (T == FFMA2_ALU) {
            // if FFMA2 only held the FMA pipe for 2 clocks, the 8 LOP3 would issue in its shadow: 16 clocks per
            // iteration per SM sub-partition warp slot; if it holds the issue port, 24
            p0 = fma2(p0, pm, pc); x ^= (x >> 3) | 0x11u; p1 = fma2(p1, pm, pc); acc ^= (acc >> 5) | 0x101ull;
            p2 = fma2(p2, pm, pc); x ^= (x >> 7) | 0x21u; p3 = fma2(p3, pm, pc); acc ^= (acc >> 9) | 0x201ull;
            p4 = fma2(p4, pm, pc); x ^= (x >> 11) | 0x41u; p5 = fma2(p5, pm, pc); acc ^= (acc >> 13) | 0x401ull;
            p6 = fma2(p6, pm, pc); x ^= (x >> 15) | 0x81u; p7 = fma2(p7, pm, pc); acc ^= (acc >> 17) | 0x801ull;
        } else if (T == FFMA_ALU) {
            f0 = fmaf(f0, fm, fc); x ^= (x >> 3) | 0x11u; f1 = fmaf(f1, fm, fc); acc ^= (acc >> 5) | 0x101ull;
            f2 = fmaf(f2, fm, fc); x ^= (x >> 7) | 0x21u; f3 = fmaf(f3, fm, fc); acc ^= (acc >> 9) | 0x201ull;
            f4 = fmaf(f4, fm, fc); x ^= (x >> 11) | 0x41u; f5 = fmaf(f5, fm, fc); acc ^= (acc >> 13) | 0x401ull;
            f6 = fmaf(f6, fm, fc); x ^= (x >> 15) | 0x81u; f7 = fmaf(f7, fm, fc); acc ^= (acc >> 17) | 0x801ull;
        } else if (T == FFMA2_MUFU) {
            p0 = fma2(p0, pm, pc); p1 = fma2(p1, pm, pc); f0 = rsq(f0); p2 = fma2(p2, pm, pc); p3 = fma2(p3, pm, pc); f1 = rsq(f1);
            p4 = fma2(p4, pm, pc); p5 = fma2(p5, pm, pc); f2 = rsq(f2); p6 = fma2(p6, pm, pc); p7 = fma2(p7, pm, pc); f3 = rsq(f3);
        } else if (T == MUFU_ALU) {
            f0 = rsq(f0); x ^= (x >> 3) | 0x11u; acc ^= (acc >> 5) | 0x101ull; f1 = rsq(f1); x ^= (x >> 7) | 0x21u; acc ^= (acc >> 9) | 0x201ull;
            f2 = rsq(f2); x ^= (x >> 11) | 0x41u; acc ^= (acc >> 13) | 0x401ull; f3 = rsq(f3); x ^= (x >> 15) | 0x81u; acc ^= (acc >> 17) | 0x801ull;
        } else if (T == BOX_MIX2) {
            // 8 boxes with packed (r, s) running sums: FADD2, FFMA, MUFU, FMUL, 1/2 FMNMX3 per box
            const unsigned long long wy = ((unsigned long long)sm[(it % nb) * 64 + lane] << 32) | 0x2b8cbccbu;
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                p0 = add2(p0, wy); p1 = add2(p1, wy); p2 = add2(p2, wy); p3 = add2(p3, wy);
                float r0 = __uint_as_float((uint32_t)p0), s0 = __uint_as_float((uint32_t)(p0 >> 32));
                float r1 = __uint_as_float((uint32_t)p1), s1 = __uint_as_float((uint32_t)(p1 >> 32));
                float r2 = __uint_as_float((uint32_t)p2), s2 = __uint_as_float((uint32_t)(p2 >> 32));
                float r3 = __uint_as_float((uint32_t)p3), s3 = __uint_as_float((uint32_t)(p3 >> 32));
                float t0 = fabsf(s0) * rsq(fmaf(-r0, r0, r0)), t1 = fabsf(s1) * rsq(fmaf(-r1, r1, r1));
                float t2 = fabsf(s2) * rsq(fmaf(-r2, r2, r2)), t3 = fabsf(s3) * rsq(fmaf(-r3, r3, r3));
                f6 = fmax3(f6, t0, t1); f7 = fmax3(f7, t2, t3);
            }
        }
    }
    __syncthreads();
    t1 = clock64();
    if (tid == 0) cycles[blockIdx.x] = t1 - t0;
    float out = f0 + f1 + f2 + f3 + f4 + f5 + f6 + f7 + (float)(d0 + d1 + d2 + d3 + d4 + d5 + d6 + d7) + (float)acc + (float)x + (float)(q[0] ^ q[1] ^ q[2] ^ q[3] ^ q[4] ^ q[5] ^ q[6] ^ q[7]) +
                (float)(p0 ^ p1 ^ p2 ^ p3 ^ p4 ^ p5 ^ p6 ^ p7);
    if (out == 12345.678f) sink[tid] = out + (float)sm[tid];
}

template <int T>
void run(int n_sm, int nb, long long *d_cyc, float *d_sink)
{
    const size_t smem = (size_t)(nb * 64 + 4096) * 4;
    cudaFuncSetAttribute(bench<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    std::vector<long long> h(n_sm);
    double best = 0, med = 0;
    for (int rep = 0; rep < 3; ++rep) {
        bench<T><<<n_sm, kThreads, smem>>>(d_cyc, d_sink, nb);
        cudaError_t e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { printf("%s: CUDA error %s\n", kNames[T], cudaGetErrorString(e)); exit(1); }
        cudaMemcpy(h.data(), d_cyc, sizeof(long long) * n_sm, cudaMemcpyDeviceToHost);
        std::sort(h.begin(), h.end());
        const double ops = (double)kThreads * kIters * kOpsPerIter[T];
        med = ops / (double)h[n_sm / 2];
        best = std::max(best, ops / (double)h[0]);
    }
    printf("%-16s %8.2f %8.2f  %s / clk / SM\n", kNames[T], med, best, kUnit[T]);
}

int main()
{
    int n_sm = 0, clk = 0;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { printf("no CUDA device\n"); return 1; }
    n_sm = prop.multiProcessorCount;
    cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0);
    printf("# %s, %d SMs, max SM clock %d MHz; %d threads/SM, %d iterations; nb = 200 bins x 64 columns\n", prop.name, n_sm,
           clk / 1000, kThreads, kIters);
    printf("# %-14s %8s %8s\n", "test", "median", "best");
    long long *d_cyc; float *d_sink;
    cudaMalloc(&d_cyc, sizeof(long long) * n_sm);
    cudaMalloc(&d_sink, sizeof(float) * kThreads);
    const int nb = 200;
    run<ATOMS_CF>(n_sm, nb, d_cyc, d_sink);
    run<ATOMS_RAND>(n_sm, nb, d_cyc, d_sink);
    run<LDS128_BCAST>(n_sm, nb, d_cyc, d_sink);
    run<LDS32_CF>(n_sm, nb, d_cyc, d_sink);
    run<MUFU_RSQ>(n_sm, nb, d_cyc, d_sink);
    run<FADD>(n_sm, nb, d_cyc, d_sink);
    run<FADD2>(n_sm, nb, d_cyc, d_sink);
    run<FFMA>(n_sm, nb, d_cyc, d_sink);
    run<FFMA2>(n_sm, nb, d_cyc, d_sink);
    run<FMNMX3>(n_sm, nb, d_cyc, d_sink);
    run<DFMA>(n_sm, nb, d_cyc, d_sink);
    run<IMAD_WIDE>(n_sm, nb, d_cyc, d_sink);
    run<FOLD_MIX>(n_sm, nb, d_cyc, d_sink);
    run<BOX_MIX>(n_sm, nb, d_cyc, d_sink);
    run<BOX_MIX2>(n_sm, nb, d_cyc, d_sink);
    run<ATOMS_CF2>(n_sm, nb, d_cyc, d_sink);
    run<LDS64_BCAST>(n_sm, nb, d_cyc, d_sink);
    run<LDS32_BCAST>(n_sm, nb, d_cyc, d_sink);
    run<LDS64_CF>(n_sm, nb, d_cyc, d_sink);
    run<I2FP>(n_sm, nb, d_cyc, d_sink);
    run<MUFU_I2FP>(n_sm, nb, d_cyc, d_sink);
    run<FMUL2>(n_sm, nb, d_cyc, d_sink);
    run<BOX_PACKED>(n_sm, nb, d_cyc, d_sink);
    run<BOX_PACKED_CVT>(n_sm, nb, d_cyc, d_sink);
    run<BOX_PACKED_THRESH>(n_sm, nb, d_cyc, d_sink);
    run<FFMA2_ALU>(n_sm, nb, d_cyc, d_sink);
    run<FFMA2_MUFU>(n_sm, nb, d_cyc, d_sink);
    run<FFMA_ALU>(n_sm, nb, d_cyc, d_sink);
    run<MUFU_ALU>(n_sm, nb, d_cyc, d_sink);
    run<BOX_PACKED_PAIRDIV>(n_sm, nb, d_cyc, d_sink);
    // row f2 at the paper's shape (140-300 epochs per star want few bins: nb = 64 as in C4); smem = S buffers of 64 bins
    run<FOLD_MIX64>(n_sm, 64, d_cyc, d_sink);
    run<FOLD_FIELD_S3>(n_sm, 3 * 64, d_cyc, d_sink);
    run<FOLD_FIELD_S7>(n_sm, 7 * 64, d_cyc, d_sink);
    run<FOLD_FIELD_STARS>(n_sm, 64, d_cyc, d_sink);
    return 0;
}
