// bb_fft.cuh -- in-register complex64 line FFTs for sm_100a.
//
// A line of N = 32*T points is transformed by T threads holding 32 points each, as a
// two-factor Cooley-Tukey split N = 32 x T:
//     n = T*n1 + n2  (n1 < 32, n2 < T),   k = k1 + 32*k2  (k1 < 32, k2 < T)
//     X[k1 + 32 k2] = sum_n2 [ w_N^(n2 k1) * ( sum_n1 x[T n1 + n2] w_32^(n1 k1) ) ] w_T^(n2 k2)
// thread n2 computes the inner radix-32 DFT over its 32 registers, multiplies by the
// twiddle w_N^(n2 k1) (fp64-built table, read from shared memory), the 32 x T matrix is
// transposed through padded shared memory, and thread t then does 32/T radix-T DFTs over
// n2 for k1 = t + T*m.  The result lands in the SAME distribution as the input
// (thread t holds X[t + T*j], j < 32), so transform -> pointwise -> transform chains stay in
// registers.  Radix kernels are fully unrolled radix-2 decimation-in-frequency recursions
// with compile-time twiddles (correctly rounded from double).
#pragma once
#include <cuda_runtime.h>

namespace bb {

typedef float2 cf;

// Complex add / subtract as ONE packed instruction (FADD2, sm_100): same lane throughput as two FADDs
// but half the issue slots, and the butterflies are two thirds additions.  Same rounding (rn per lane).
__device__ __forceinline__ cf cadd(cf a, cf b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<cf *>(&r);
}
__device__ __forceinline__ cf csub(cf a, cf b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<cf *>(&r);
}
// Packed-pair plumbing: ptxas folds the pair construction into operand selectors (scalar broadcast
// R.F32, swapped halves R.F32x2.LO_HI, and a sign per half: -R.F32x2.LO_HI.NP), so these cost no instructions.
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk2(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ cf up2(u64 v) { cf r; asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
// (A, B) * (rh + rl) per lane, one rounding of t*rh + t*rl each: two packed instructions
__device__ __forceinline__ cf mul_hilo2(u64 ab, float rh, float rl) {
    return up2(fma2(ab, pk2(rh, rh), mul2(ab, pk2(rl, rl))));
}

// a * w as FMUL2 + FFMA2: (x c, y c) + (y, x) * (-s, s); the swapped and half-negated operand is an
// operand selector of the instruction, not an instruction.
__device__ __forceinline__ cf cmul(cf a, cf w) {
    return up2(fma2(pk2(a.y, a.x), pk2(-w.y, w.y), mul2(pk2(a.x, a.y), pk2(w.x, w.x))));
}
// a * conj(w)
__device__ __forceinline__ cf cmulc(cf a, cf w) {
    return up2(fma2(pk2(a.y, a.x), pk2(w.y, -w.y), mul2(pk2(a.x, a.y), pk2(w.x, w.x))));
}

// cos(2 pi m / 32), m = 0..16, in double; the kernels use it as a two-float constant
// hi = (float)c, lo = (float)(c - hi).
__device__ __forceinline__ constexpr double cos32d(int m) {
    constexpr double C[17] = {
        1.0,
        0.98078528040323044912618223613424,
        0.92387953251128675612818318939679,
        0.83146961230254523707878837761791,
        0.70710678118654752440084436210485,
        0.55557023301960222474283081394853,
        0.38268343236508977172845998403040,
        0.19509032201612826784828486847702,
        0.0,
        -0.19509032201612826784828486847702,
        -0.38268343236508977172845998403040,
        -0.55557023301960222474283081394853,
        -0.70710678118654752440084436210485,
        -0.83146961230254523707878837761791,
        -0.92387953251128675612818318939679,
        -0.98078528040323044912618223613424,
        -1.0};
    return C[m];
}
__device__ __forceinline__ constexpr double sin32d(int m) {   // sin(2 pi m/32) = cos(2 pi (m-8)/32), m in [0,16]
    return cos32d(m >= 8 ? m - 8 : 8 - m);
}
__device__ __forceinline__ constexpr float hi_of(double c) { return (float)c; }
__device__ __forceinline__ constexpr float lo_of(double c) { return (float)(c - (double)(float)c); }


// a * exp(SIGN * 2 pi i * M / 32),  0 <= M < 16.
// The constants are two-float values and the low parts enter INSIDE the fused multiply-add
// chain, so each product is an unbiased rounding of the exact one.  With plain float32
// constants every 32nd root of unity happens to round to |w| < 1 (by 0.7e-8 .. 2.9e-8); the
// same shrink factor would then hit the field at every step and the error of a propagation
// would grow linearly with the number of steps.
template <int M, int SIGN>
__device__ __forceinline__ cf mul_w32(cf a) {
    if constexpr (M == 0) {
        return a;
    } else if constexpr (M == 8) {              // * (SIGN i)
        return SIGN < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
    } else if constexpr (M == 4 || M == 12) {   // * (+-1 + SIGN i)/sqrt2
        constexpr float rh = hi_of(cos32d(4)), rl = lo_of(cos32d(4));
        // (p, q) = (x + y, y - x) as one packed add of (x, y) and (y, -x)
        const u64 axy = pk2(a.x, a.y);
        if constexpr (M == 4)
            return SIGN < 0 ? mul_hilo2(add2(axy, pk2(a.y, -a.x)), rh, rl)        // ( p,  q)
                            : mul_hilo2(add2(axy, pk2(-a.y, a.x)), rh, rl);       // (-q,  p)
        else
            return SIGN < 0 ? mul_hilo2(add2(pk2(-a.x, -a.y), pk2(a.y, -a.x)), rh, rl)   // ( q, -p)
                            : mul_hilo2(add2(pk2(-a.x, -a.y), pk2(-a.y, a.x)), rh, rl);  // (-p, -q)
    } else {
        // a * (c + i s), c = ch + cl, s = sh + sl: four packed instructions, low parts first
        constexpr double cd = cos32d(M), sd = SIGN < 0 ? -sin32d(M) : sin32d(M);
        constexpr float c = hi_of(cd), cl = lo_of(cd), s = hi_of(sd), sl = lo_of(sd);
        const u64 axy = pk2(a.x, a.y), ayx = pk2(a.y, a.x);
        u64 t = mul2(ayx, pk2(-sl, sl));
        t = fma2(axy, pk2(cl, cl), t);
        t = fma2(ayx, pk2(-s, s), t);
        return up2(fma2(axy, pk2(c, c), t));
    }
}

// Radix-R DFT over registers, natural order in and out:
//   v[k] <- sum_n v[n] exp(SIGN 2 pi i n k / R)
template <int R, int SIGN>
struct Dft {
    static __device__ __forceinline__ void run(cf (&v)[R]) {
        constexpr int H = R / 2;
        cf a[H], b[H];
#pragma unroll
        for (int n = 0; n < H; ++n) {
            a[n] = cadd(v[n], v[n + H]);
            b[n] = csub(v[n], v[n + H]);
        }
        twiddle<0>(b);
        Dft<H, SIGN>::run(a);
        Dft<H, SIGN>::run(b);
#pragma unroll
        for (int k = 0; k < H; ++k) {
            v[2 * k] = a[k];
            v[2 * k + 1] = b[k];
        }
    }
    template <int n>
    static __device__ __forceinline__ void twiddle(cf (&b)[R / 2]) {
        if constexpr (n < R / 2) {
            b[n] = mul_w32<n*(32 / R), SIGN>(b[n]);
            twiddle<n + 1>(b);
        }
    }
};
template <int SIGN>
struct Dft<2, SIGN> {
    static __device__ __forceinline__ void run(cf (&v)[2]) {
        cf a = cadd(v[0], v[1]);
        v[1] = csub(v[0], v[1]);
        v[0] = a;
    }
};
template <int SIGN>
struct Dft<1, SIGN> {
    static __device__ __forceinline__ void run(cf (&)[1]) {}
};

// Shared-memory geometry of the 32 x T transpose (float2 units); paddings found by brute
// force to make both the stores and the loads bank-conflict free for 64-bit accesses.
//   row mapping   : lane = g*T + t, one region per line g of a warp
//   column mapping: r = c + CW*t inside a tile of CW columns, one region per column c
template <int T> struct RowGeom {
    static constexpr int S = T + 1;                                   // stride between k1 rows
    static constexpr int RS = 32 * S + (T < 16 ? T : 0);              // stride between lines
    static constexpr int WARP = T == 1 ? 0 : (32 / T) * RS;           // float2 per warp (T = 1: no transpose)
};
template <int T, int CW> struct ColGeom {
    static constexpr int S = (CW == 16) ? T : T + 1;
    static constexpr int RS = 32 * S + (CW == 16 ? 1 : (CW == 8 ? 2 : (T == 2 ? 2 : 4)));
    static constexpr int TILE = T == 1 ? 0 : CW * RS;                 // float2 per tile slot
};

// Team synchronisation of the transposes: a row line lives in one warp, a column tile spans the CTA.
struct SyncSel {
    bool warp;
    __device__ __forceinline__ void operator()() const {
        if (warp) __syncwarp();
        else __syncthreads();
    }
};

// One forward line FFT (see file header).  v: this thread's 32 points x[t + T*j].
//   tw   : shared, [32][T], tw[k1*T + t] = exp(-2 pi i k1 t / N)
//   ybuf : shared, base of this thread's line region; S = stride between k1 rows
// The inverse transform is conj . forward . conj (done by the caller), so that one copy of this
// code serves both directions.  For T = 32 the two radix-32 stages are a rolled loop over the
// same butterfly code.
template <int T, int S, class Sync>
__device__ __forceinline__ void line_fft_fwd(cf (&v)[32], const cf *__restrict__ tw, cf *ybuf, int t, Sync sync) {
    if constexpr (T == 1) {
        Dft<32, -1>::run(v);
    } else if constexpr (T == 32) {
#pragma unroll 1
        for (int stage = 0; stage < 2; ++stage) {
            Dft<32, -1>::run(v);
            if (stage == 0) {
#pragma unroll
                for (int k1 = 0; k1 < 32; ++k1) {
                    cf x = v[k1];
                    if (k1 > 0) x = cmul(x, tw[k1 * T + t]);
                    ybuf[k1 * S + t] = x;
                }
                sync();
#pragma unroll
                for (int n2 = 0; n2 < 32; ++n2) v[n2] = ybuf[t * S + n2];
                sync();
            }
        }
    } else {
        Dft<32, -1>::run(v);
#pragma unroll
        for (int k1 = 0; k1 < 32; ++k1) {
            cf x = v[k1];
            if (k1 > 0) x = cmul(x, tw[k1 * T + t]);
            ybuf[k1 * S + t] = x;
        }
        sync();
        constexpr int G = 32 / T;
#pragma unroll
        for (int m = 0; m < G; ++m) {
            cf w[T];
#pragma unroll
            for (int n2 = 0; n2 < T; ++n2) w[n2] = ybuf[(t + T * m) * S + n2];
            Dft<T, -1>::run(w);
#pragma unroll
            for (int k2 = 0; k2 < T; ++k2) v[m + G * k2] = w[k2];
        }
        sync();
    }
}

}  // namespace bb
