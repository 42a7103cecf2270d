// bb_fft8.cuh -- complex64 sub-line FFTs with 8 points per thread (lines of 256 P points, P in {1, 2, 4, 8}).
//
// Same decomposition as bb_fft16.cuh (a line of N = 256 P points = P sub-lines of 256 points, each
// transformed as 16 x 16; the radix-P butterfly that joins them is fused with the pointwise step),
// but a sub-line is held by 32 threads x 8 points, so that an SM runs twice the warps (the phases
// are bound by per-warp latency, profiles/r02_a): every radix-16 is shared by a PAIR of lanes
// (lane ^ 16), each doing a radix-8 over its half and one exchange of 4 values by shfl
// (BASELINE.json north_star item 1: "radix-8/16 butterflies using warp shuffles").
//
// Thread (t, h) of a sub-line, t < 16, h < 2 (h = bit 4 of the lane index).  With
//     n = 16 n1 + n2,  k = k1 + 16 k2,   X[k1 + 16 k2] = sum_n2 w_16^(n2 k2) [ w_256^(n2 k1) sum_n1 x[16 n1 + n2] w_16^(n1 k1) ]
// two register distributions of a 16-point index m over the pair occur:
//     parity : register i of lane h holds m = 2 i + h                (i < 8)
//     split  : register j holds m = 4 h + j, register 4 + j holds m = 4 h + 8 + j   (j < 4)
// A decimation-in-time pair stage takes parity to split, a decimation-in-frequency one split to
// parity; subline8_dit (both stages in time) and subline8_dif (both in frequency) therefore chain
// without any data movement between them: "dit -> pointwise -> dif" maps the parity distribution of
// the sub-line elements (element 32 i + 16 h + t in register i: consecutive lanes, consecutive
// elements) onto itself.
#pragma once
#include "bb_fft16.cuh"

namespace bb {

// a * exp(SIGN 2 pi i M / 32), 0 <= M < 32 (mul_w32 covers M < 16; the rest are its negatives, with
// the sign folded into the constants).
template <int M, int SIGN>
__device__ __forceinline__ cf mul_w32x(cf a) {
    if constexpr (M < 16) {
        return mul_w32<M, SIGN>(a);
    } else if constexpr (M == 16) {
        return make_float2(-a.x, -a.y);
    } else if constexpr (M == 24) {             // * (-SIGN i)
        return SIGN < 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
    } else if constexpr (M == 20 || M == 28) {
        constexpr float rh = -hi_of(cos32d(4)), rl = -lo_of(cos32d(4));
        const u64 axy = pk2(a.x, a.y);
        if constexpr (M == 20)
            return SIGN < 0 ? mul_hilo2(add2(axy, pk2(a.y, -a.x)), rh, rl)
                            : mul_hilo2(add2(axy, pk2(-a.y, a.x)), rh, rl);
        else
            return SIGN < 0 ? mul_hilo2(add2(pk2(-a.x, -a.y), pk2(a.y, -a.x)), rh, rl)
                            : mul_hilo2(add2(pk2(-a.x, -a.y), pk2(-a.y, a.x)), rh, rl);
    } else {
        constexpr double cd = -cos32d(M - 16), sd = SIGN < 0 ? sin32d(M - 16) : -sin32d(M - 16);
        constexpr float c = hi_of(cd), cl = lo_of(cd), s = hi_of(sd), sl = lo_of(sd);
        const u64 axy = pk2(a.x, a.y), ayx = pk2(a.y, a.x);
        u64 t = mul2(ayx, pk2(-sl, sl));
        t = fma2(axy, pk2(cl, cl), t);
        t = fma2(ayx, pk2(-s, s), t);
        return up2(fma2(axy, pk2(c, c), t));
    }
}
// a * exp(SIGN 2 pi i M / 16), 0 <= M < 16
template <int M, int SIGN>
__device__ __forceinline__ cf mul_w16(cf a) { return mul_w32x<2 * M, SIGN>(a); }

__device__ __forceinline__ cf fma2c(float s, cf a, cf b) {      // s a + b, per component
    return up2(fma2(pk2(s, s), pk2(a.x, a.y), pk2(b.x, b.y)));
}
// the value of the other lane of the pair (lane ^ X; X = 16: one pair per sub-line index t of a warp)
template <int X = 16>
__device__ __forceinline__ cf shfl16(cf a) {
    return make_float2(__shfl_xor_sync(0xFFFFFFFFu, a.x, X), __shfl_xor_sync(0xFFFFFFFFu, a.y, X));
}

// Radix-8 DFT, natural order in, out[k] = X[(k + 4 r) mod 8] with r = 0 for s = +1, r = 1 for s = -1
// (s multiplies the odd inputs, i.e. only the last butterfly stage: no extra instructions).
template <int SIGN>
__device__ __forceinline__ void dft8_rot_out(cf (&v)[8], float s) {
    cf a[4], b[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) { a[n] = cadd(v[n], v[n + 4]); b[n] = csub(v[n], v[n + 4]); }
    b[1] = mul_w32<4, SIGN>(b[1]); b[2] = mul_w32<8, SIGN>(b[2]); b[3] = mul_w32<12, SIGN>(b[3]);
    cf c0 = cadd(a[0], a[2]), c1 = cadd(a[1], a[3]), d0 = csub(a[0], a[2]), d1 = mul_w32<8, SIGN>(csub(a[1], a[3]));
    cf e0 = cadd(b[0], b[2]), e1 = cadd(b[1], b[3]), f0 = csub(b[0], b[2]), f1 = mul_w32<8, SIGN>(csub(b[1], b[3]));
    v[0] = fma2c(s, c1, c0); v[4] = fma2c(-s, c1, c0);
    v[2] = fma2c(s, d1, d0); v[6] = fma2c(-s, d1, d0);
    v[1] = fma2c(s, e1, e0); v[5] = fma2c(-s, e1, e0);
    v[3] = fma2c(s, f1, f0); v[7] = fma2c(-s, f1, f0);
}

// Radix-8 DFT of the sequence x[m] = in[(m + 4 r) mod 8] (r as above: lane 1 of a pair holds its
// inputs rotated by four), natural order out: the rotation negates the difference branch.
template <int SIGN>
__device__ __forceinline__ void dft8_rot_in(cf (&v)[8], float s) {
    cf a[4], b[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) { a[n] = cadd(v[n], v[n + 4]); b[n] = csub(v[n], v[n + 4]); }
    constexpr float rh = hi_of(cos32d(4)), rl = lo_of(cos32d(4));
    const float srh = s * rh, srl = s * rl;
    b[0] = make_float2(s * b[0].x, s * b[0].y);
    {   // s * b[1] * (1 + SIGN i) / sqrt2
        const u64 x = pk2(b[1].x, b[1].y);
        b[1] = mul_hilo2(SIGN < 0 ? add2(x, pk2(b[1].y, -b[1].x)) : add2(x, pk2(-b[1].y, b[1].x)), srh, srl);
    }
    b[2] = SIGN < 0 ? make_float2(s * b[2].y, -s * b[2].x) : make_float2(-s * b[2].y, s * b[2].x);
    {   // s * b[3] * (-1 + SIGN i) / sqrt2
        const u64 x = pk2(-b[3].x, -b[3].y);
        b[3] = mul_hilo2(SIGN < 0 ? add2(x, pk2(b[3].y, -b[3].x)) : add2(x, pk2(-b[3].y, b[3].x)), srh, srl);
    }
    cf c0 = cadd(a[0], a[2]), c1 = cadd(a[1], a[3]), d0 = csub(a[0], a[2]), d1 = mul_w32<8, SIGN>(csub(a[1], a[3]));
    cf e0 = cadd(b[0], b[2]), e1 = cadd(b[1], b[3]), f0 = csub(b[0], b[2]), f1 = mul_w32<8, SIGN>(csub(b[1], b[3]));
    v[0] = cadd(c0, c1); v[4] = csub(c0, c1);
    v[2] = cadd(d0, d1); v[6] = csub(d0, d1);
    v[1] = cadd(e0, e1); v[5] = csub(e0, e1);
    v[3] = cadd(f0, f1); v[7] = csub(f0, f1);
}

// 16-point DFT over a lane pair, decimation in time: parity in, split out.
//   h = 0 / 1: which lane of the pair; s = +1 / -1 accordingly.
// X[k] = E0[k] + w^k E1[k], X[k + 8] = E0[k] - w^k E1[k] with E_h the 8-point DFT of lane h's inputs and
// w = exp(SIGN 2 pi i / 16).  Lane 1 produces E1 rotated by four (dft8_rot_out) and twiddled, so that
// both lanes keep registers 0..3 and trade registers 4..7 (lane 1 sends its half negated):
//   out[j] = own[j] - s recv[j],   out[4 + j] = s own[j] + recv[j].
template <int SIGN, int X = 16>
__device__ __forceinline__ void pair16_dit(cf (&v)[8], int h, float s) {
    dft8_rot_out<SIGN>(v, s);
    if (h) {
        v[0] = mul_w16<4, SIGN>(v[0]);  v[1] = mul_w16<5, SIGN>(v[1]);  v[2] = mul_w16<6, SIGN>(v[2]);  v[3] = mul_w16<7, SIGN>(v[3]);
        v[4] = mul_w16<8, SIGN>(v[4]);  v[5] = mul_w16<9, SIGN>(v[5]);  v[6] = mul_w16<10, SIGN>(v[6]); v[7] = mul_w16<11, SIGN>(v[7]);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const cf r = shfl16<X>(v[4 + j]);
        const cf own = v[j];
        v[j] = fma2c(-s, r, own);
        v[4 + j] = fma2c(s, own, r);
    }
}

// 16-point DFT over a lane pair, decimation in frequency: split in, parity out.
//   u[m] = x[m] + x[m + 8], d[m] = (x[m] - x[m + 8]) w^m, m < 8;  X[2k] = DFT8(u)[k], X[2k + 1] = DFT8(d)[k].
// Lane h holds m = 4 h + j: it keeps the half its own output parity needs (lane 0: u, lane 1: the raw
// difference), sends the other, and lane 1 runs its radix-8 on inputs rotated by four (dft8_rot_in).
template <int SIGN, int X = 16>
__device__ __forceinline__ void pair16_dif(cf (&v)[8], int h, float s) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const cf keep = fma2c(s, v[4 + j], v[j]);
        const cf send = fma2c(-s, v[4 + j], v[j]);
        v[j] = keep;
        v[4 + j] = shfl16<X>(send);
    }
    if (h) {   // register i holds the raw difference of m = (i + 4) mod 8
        v[0] = mul_w16<4, SIGN>(v[0]); v[1] = mul_w16<5, SIGN>(v[1]); v[2] = mul_w16<6, SIGN>(v[2]); v[3] = mul_w16<7, SIGN>(v[3]);
        v[5] = mul_w16<1, SIGN>(v[5]); v[6] = mul_w16<2, SIGN>(v[6]); v[7] = mul_w16<3, SIGN>(v[7]);
    }
    dft8_rot_in<SIGN>(v, s);
}

// Where thread (t, h) of a sub-line sits in its shared-memory regions.
struct Lane8 {
    int t, h;
    float s;
};

// One sub-line transform of sign SIGN, decimation in time in both radix-16 stages.
//   in  : v[i] = x[32 i + 16 h + t]                                    (parity over n1, n2 = t)
//   out : v[j] = X[t + 16 (4 h + j)], v[4 + j] = X[t + 16 (4 h + 8 + j)]   (split over k2, k1 = t)
//   tw  : shared, [16][16], tw[k1 * 16 + t] = exp(-2 pi i k1 t / 256)
//   ybuf: shared, this sub-line's transpose region (offset by the column of a column tile); element
//         (k1, n2) at (k1 * 17 + n2) * CW: stores (fixed k1 per half-warp) and loads (fixed n2) are
//         bank-conflict free for 64-bit accesses.
template <int SIGN, int CW, class Sync>
__device__ __forceinline__ void subline8_dit(cf (&v)[8], const cf *__restrict__ tw, cf *ybuf, Lane8 l, Sync sync) {
    pair16_dit<SIGN>(v, l.h, l.s);
    const cf *twp = tw + (4 * l.h) * 16 + l.t;
    cf *yst = ybuf + ((4 * l.h) * 17 + l.t) * CW;
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) {
        const int k1 = (jj & 3) + 8 * (jj >> 2);                  // + 4 h
        yst[k1 * 17 * CW] = cmul_s<SIGN>(v[jj], twp[k1 * 16]);
    }
    sync();
    const cf *yld = ybuf + (l.t * 17 + l.h) * CW;
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = yld[2 * i * CW];
    pair16_dit<SIGN>(v, l.h, l.s);
}

// The same, decimation in frequency in both stages.
//   in  : v[j] = x[t + 16 (4 h + j)], v[4 + j] = x[t + 16 (4 h + 8 + j)]   (split over n1, n2 = t)
//   out : v[k] = X[t + 16 (2 k + h)] = element 32 k + 16 h + t             (parity over k2, k1 = t)
template <int SIGN, int CW, class Sync>
__device__ __forceinline__ void subline8_dif(cf (&v)[8], const cf *__restrict__ tw, cf *ybuf, Lane8 l, Sync sync) {
    pair16_dif<SIGN>(v, l.h, l.s);
    const cf *twp = tw + l.h * 16 + l.t;
    cf *yst = ybuf + (l.h * 17 + l.t) * CW;
#pragma unroll
    for (int k = 0; k < 8; ++k) yst[2 * k * 17 * CW] = cmul_s<SIGN>(v[k], twp[2 * k * 16]);
    sync();
    const cf *yld = ybuf + (l.t * 17 + 4 * l.h) * CW;
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) v[jj] = yld[((jj & 3) + 8 * (jj >> 2)) * CW];
    pair16_dif<SIGN>(v, l.h, l.s);
}

// Radix-8 butterfly over 8 consecutive registers (the class butterfly of 2048-point lines), natural order.
template <int SIGN>
__device__ __forceinline__ void class_dft8(cf *w) {
    cf v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = w[i];
    Dft<8, SIGN>::run(v);
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = v[i];
}

}  // namespace bb
