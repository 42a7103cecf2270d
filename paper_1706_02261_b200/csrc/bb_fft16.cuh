// bb_fft16.cuh -- complex64 line FFTs with 16 points per thread (lines of 256 P points, P in {1, 2, 4}).
//
// A line of N = 256 P points is split by radix-P decimation into P sub-lines ("classes") of
// L = 256 points; a sub-line is held by 16 lanes x 16 points and transformed as 16 x 16
// (DESIGN.md "Line FFT, 16-point threads"):
//     n = 16 n1 + n2,  k = k1 + 16 k2   (all < 16)
//     X[k1 + 16 k2] = sum_n2 w_16^(n2 k2) [ w_256^(n2 k1) sum_n1 x[16 n1 + n2] w_16^(n1 k1) ]
// lane n2 does the inner radix-16 over its registers, multiplies by w_256^(n2 k1) (fp64-built
// table in shared memory), the 16 x 16 matrix is transposed through padded shared memory and
// lane k1 does the outer radix-16.  Input and output have the same distribution: lane t holds
// element t + 16 j in register j.
//
// The radix-P butterfly that joins the classes is NOT part of the sub-line transform: it is
// fused with the pointwise step of the phase (bb_kernels16.cuh), where one thread holds the P
// class values of the same sub-line index.  For a transform of sign s (kernel exp(s 2 pi i nk/N)):
//   decimation in time  (classes on the INPUT,  c = n mod P):
//       X[q + L m] = sum_c [ e(c q / N) F_c[q] ] e(c m / P),        F_c = sub-line transform of x[P n' + c]
//   decimation in frequency (classes on the OUTPUT, c = k mod P):
//       X[P k' + c] = sub-line transform over q of  e(q c / N) sum_m x[q + L m] e(m c / P)
// with e(a) = exp(s 2 pi i a).
#pragma once
#include "bb_fft.cuh"

namespace bb {

constexpr int kL = 256;           // sub-line length

// a * w (SIGN < 0) or a * conj(w) (SIGN > 0): tables hold the forward (negative-exponent) roots.
template <int SIGN>
__device__ __forceinline__ cf cmul_s(cf a, cf w) { return SIGN < 0 ? cmul(a, w) : cmulc(a, w); }

// One sub-line transform of sign SIGN.
//   v    : this lane's 16 points x[t + 16 j]
//   tw   : shared, [16][16], tw[k1*16 + t] = exp(-2 pi i k1 t / 256)
//   ybuf : shared, this sub-line's transpose region (already offset by the column of a column
//          tile); element (k1, n2) lives at (k1*17 + n2)*CW: for 64-bit accesses both the stores
//          (fixed k1, lanes over n2 and the CW columns) and the loads (fixed n2, lanes over k1 and
//          the columns) are bank-conflict free, because 17 CW = CW (mod 16).
//   sync : makes the stores of all 16 lanes of the sub-line visible (half-warp for rows, tile for columns)
template <int SIGN, int CW, class Sync>
__device__ __forceinline__ void subline_fft(cf (&v)[16], const cf *__restrict__ tw, cf *ybuf, int t, Sync sync) {
    Dft<16, SIGN>::run(v);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        cf x = v[k1];
        if (k1 > 0) x = cmul_s<SIGN>(x, tw[k1 * 16 + t]);
        ybuf[(k1 * 17 + t) * CW] = x;
    }
    sync();
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) v[n2] = ybuf[(t * 17 + n2) * CW];
    Dft<16, SIGN>::run(v);
}

// Radix-P butterfly over P consecutive registers of the 16 (P = 1, 2, 4, 8), natural order in and out.
template <int P, int SIGN>
__device__ __forceinline__ void class_dft(cf *w) {
    if constexpr (P == 2) {
        const cf a = cadd(w[0], w[1]);
        w[1] = csub(w[0], w[1]);
        w[0] = a;
    } else if constexpr (P == 4) {
        const cf a = cadd(w[0], w[2]), b = csub(w[0], w[2]);
        const cf c = cadd(w[1], w[3]), d0 = csub(w[1], w[3]);
        const cf d = SIGN < 0 ? make_float2(d0.y, -d0.x) : make_float2(-d0.y, d0.x);   // * (SIGN i)
        w[0] = cadd(a, c);
        w[1] = cadd(b, d);
        w[2] = csub(a, c);
        w[3] = csub(b, d);
    } else if constexpr (P == 8) {
        cf v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = w[i];
        Dft<8, SIGN>::run(v);
#pragma unroll
        for (int i = 0; i < 8; ++i) w[i] = v[i];
    }
}

}  // namespace bb
