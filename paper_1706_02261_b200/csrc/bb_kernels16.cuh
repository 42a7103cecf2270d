// bb_kernels16.cuh -- the BPM step kernel with 16 points per thread (Nx, Ny in {256, 512, 1024, 2048}; single fields and batches).
//
// Same two-phase structure as bb_kernels.cuh:
//   column phase C_j : FFT_y  -> x H_j                          -> IFFT_y
//   row phase    R_j : IFFT_x -> x exp(i phi(dn[j-1])), |u|^2   -> FFT_x
// but a line of N = 256 P points is split into P sub-lines of 256 points (bb_fft16.cuh) held
// by 16 lanes x 16 points each, so an SM runs 16 warps at <= 128 registers instead of 8 at
// ~180, and the radix-P butterfly that joins the sub-lines is fused with the pointwise step:
//
//   load classes -> P sub-line transforms -> exchange -> [twiddle, radix-P, POINTWISE, radix-P,
//   twiddle] -> exchange -> P sub-line transforms -> store classes
//
// "exchange" regroups, through shared memory, the team of 16 P threads that owns a line from
// "thread = (class, lane), 16 indices of one class" to "thread = (group, lane), 16/P indices
// of every class".  Row phase: classes are kx mod P, and between the phases the field is kept
// kx-class-major in memory (kx = P k' + c at column c N/P + k'), so that every sub-line is
// contiguous; the propagator table is built with the same column permutation.  Column phase:
// classes are y mod P (interleaved rows), natural order at both ends.
#pragma once
#include "bb_kernels.cuh"
#include "bb_fft16.cuh"

namespace bb {

constexpr int kThreads16 = 512;

template <int PX, int PY>
struct Smem16 {
    static constexpr int kTw = 256;                                   // sub-line twiddles [16][16]
    static constexpr int kTwc = (PX - 1) * kL + (PY - 1) * kL;          // class twiddles, x then y
    static constexpr int kY = (kThreads16 / 16) * 16 * 17;              // sub-line transposes; the class exchange
                                                                        // (kThreads16 * 16) reuses the same region
    static constexpr int kPw = kThreads16 * 16;                         // pointwise factors: one buffer for the
                                                                        // propagator values, one for the screen
    static constexpr size_t bytes = (size_t)(kTw + kTwc + kY + 2 * kPw) * sizeof(cf) + 16 + 8 * 8;
};

struct Phase16 {
    bool is_row;
    bool first, second;    // first / second transform of the phase runs
    int kind;              // 0 none, 1 phase screen of a dn slice (+ intensity), 2 propagator table
    const void *src;
    float pa;
    long long slice;       // kind 1: element offset of the intensity slice
};

__device__ __forceinline__ Phase16 decode_phase16(const KParams &P, int p) {
    Phase16 d;
    d.kind = 0; d.src = nullptr; d.pa = 0.f; d.slice = 0;
    d.is_row = (p & 1) == 0;
    if (d.is_row) {
        d.first = p >= 2;
        d.second = (p >> 1) < P.Nz_total;
        const int j = row_step(P, p >> 1);
        if (j >= 0) {
            // (homogeneous medium, KParams::noscreen: dn is a null pointer that is never read -- the staging
            // functions take dn = 0 -- and d.src only tells the slices apart)
            d.kind = 1;
            d.slice = (long long)(j - P.j_base) * ((long long)P.Nx * P.Ny);
            d.src = P.dn + d.slice;
            d.pa = P.phase_a[j];
        }
    } else {
        d.first = d.second = true;
        d.kind = 2;
        d.src = P.htab[col_step(P, p >> 1)];
    }
    return d;
}

// Thread roles inside the team that owns one line (row phase) or one tile of CW columns (column phase).
template <int P, int CW>
struct Team16 {
    static constexpr int TEAM = 16 * P * CW;           // threads
    static constexpr int NTEAM = kThreads16 / TEAM;    // teams per CTA
    static constexpr int JP = 16 / P;                  // sub-line indices per thread after the exchange
    int team, col, t, c;
    __device__ __forceinline__ Team16() {
        const int r = threadIdx.x % TEAM;
        team = threadIdx.x / TEAM;
        col = r % CW;
        t = (r / CW) % 16;
        c = r / (16 * CW);
    }
    __device__ __forceinline__ void sync() const {
        if constexpr (TEAM == 16) __syncwarp(0xFFFFu << (16 * (team & 1)));
        else if constexpr (TEAM == 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(TEAM) : "memory");
    }
    // sub-line index of slot jp after the exchange, and line index (pixel / frequency) of slot (jp, m)
    __device__ __forceinline__ int q(int jp) const { return t + 16 * (P * jp + c); }
};

// Columns that can hold light.  The propagator is zero for kx^2 >= k^2 (bb.h step 2, evanescent
// cut), so on an oversampled grid (dx < lambda / 2n) a band of kx columns is exactly zero after
// every column phase: such columns are neither computed, stored nor loaded.  F = largest |DFT bin|
// that may be non-zero (from the host, conservative).  Bookkeeping is per tile of `cw` adjacent
// memory columns; in the kx-class-major layout class c holds bins P k' + c, whose live columns are
// a low run k' <= (F - c) / P and a high run k' >= ceil((N - F - c) / P).
template <int P>
struct LiveCols {
    int nlo[P], nhi[P], ntc;           // live tiles at the low / high end of each class, tiles per class
    __device__ __forceinline__ LiveCols(int F, int N, int cw_log2) {   // tiles of 1 << cw_log2 columns
        const int L = N / P, cw = 1 << cw_log2;
        ntc = L >> cw_log2;
#pragma unroll
        for (int c = 0; c < P; ++c) {
            int lo_cols = F >= c ? (F - c) / P + 1 : 0;
            if (lo_cols > L) lo_cols = L;
            int hs = (N - F - c + P - 1) / P;
            if (hs > L) hs = L;
            int a = (lo_cols + cw - 1) >> cw_log2, b = ntc - (hs >> cw_log2);
            if (a + b >= ntc) { a = ntc; b = 0; }
            nlo[c] = a; nhi[c] = b;
        }
    }
    __device__ __forceinline__ int total() const {
        int n = 0;
#pragma unroll
        for (int c = 0; c < P; ++c) n += nlo[c] + nhi[c];
        return n;
    }
    // m-th live tile -> tile index in memory order
    __device__ __forceinline__ int tile(int m) const {
        int u = 0;
#pragma unroll
        for (int c = 0; c < P; ++c) {
            const int n = nlo[c] + nhi[c];
            if (m >= 0 && m < n) u = c * ntc + (m < nlo[c] ? m : ntc - n + m);
            m -= n;
        }
        return u;
    }
};

// Bit i set: sub-line element e0 + 16 i (e0 < 16) of kx class c sits in a live tile of 1 << cw_log2
// columns (cw_log2 <= 4).  Same rule as LiveCols, for one class, in closed form: the live tiles are
// tau < lo or tau >= hi with tau = (e0 + 16 i) >> cw_log2 = (i << (4 - cw_log2)) + (e0 >> cw_log2).
template <int P>
__device__ __forceinline__ unsigned live_mask16(int F, int N, int c, int e0, int cw_log2) {
    const int L = N / P, cw = 1 << cw_log2;
    int lo_cols = F >= c ? (F - c) / P + 1 : 0;
    if (lo_cols > L) lo_cols = L;
    int hs = (N - F - c + P - 1) / P;
    if (hs > L) hs = L;
    int lo = (lo_cols + cw - 1) >> cw_log2, hi = hs >> cw_log2;
    if (lo >= hi) return 0xFFFFu;
    const int sh = 4 - cw_log2, t2 = e0 >> cw_log2, r = (1 << sh) - 1;
    int nl = (lo - t2 + r) >> sh, nh = (hi - t2 + r) >> sh;        // i < nl or i >= nh
    nl = nl < 0 ? 0 : (nl > 16 ? 16 : nl);
    nh = nh < 0 ? 0 : (nh > 16 ? 16 : nh);
    return (((1u << nl) - 1u) | ~((1u << nh) - 1u)) & 0xFFFFu;
}

// What a thread derives from the live band F of a phase (unit range of the CTA, first unit of the
// team, load mask): recomputed only when F changes, i.e. when the reference index does -- every
// instruction of a phase prologue is paid by all 16 warps with nothing to overlap it.
struct UnitCache {
    int F = -1, a0 = 0, a1 = 0, u0 = 0;
    unsigned lmask = 0xFFFFu;
    unsigned tma_parity = 0;           // phase bit of the team's TMA barrier
};

// ---- TMA / mbarrier plumbing (column tiles of the single-field kernel) ----
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// false: gave up (a hang would take the box down; the caller raises the watchdog flag)
__device__ __forceinline__ bool mbar_wait(unsigned long long *bar, unsigned parity) {
    for (unsigned spins = 0; spins < (1u << 22); ++spins) {
        unsigned ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (ok) return true;
    }
    return false;
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3,
                                            unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

struct HalfWarpSync {
    unsigned mask;
    __device__ __forceinline__ void operator()() const { __syncwarp(mask); }
};
// The CW * 16 threads that share the transposes of one class of a column tile (whole warps).
template <int THREADS>
struct ClassSync {
    int id;
    __device__ __forceinline__ void operator()() const {
        asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(THREADS) : "memory");
    }
};

// sin and cos of the phase-screen argument (bb.h step 4).  Arguments are k0 dz (n - n_ref), a
// fraction of a radian for any sample a BPM step is valid for: three-term Cody-Waite reduction by
// pi/2 and degree-7/8 polynomials on [-pi/4, pi/4] (weighted least-squares fits, max abs error
// 4.5e-8 / 7.4e-8 in float32, i.e. half an ulp of 1), without the large-argument path of sincosf
// that made the staging 28 % of a row phase (profiles/r01_b).  Huge arguments take the library path.
__device__ __forceinline__ void screen_sincos(float a, float &sn, float &cs) {
    if (fabsf(a) > 4096.f) { sincosf(a, &sn, &cs); return; }
    const float k = rintf(a * 6.366197467e-01f);
    float r = fmaf(k, -1.570796371e+00f, a);
    r = fmaf(k, 4.371138829e-08f, r);
    r = fmaf(k, 1.776356839e-15f, r);
    const int q = (int)k;
    const float r2 = r * r;
    float sp = fmaf(-1.9513932562e-04f, r2, 8.3321482563e-03f);
    sp = fmaf(sp, r2, -1.6666654339e-01f);
    const float s0 = fmaf(r * r2, sp, r);
    float cp = fmaf(2.4435851735e-05f, r2, -1.3887341487e-03f);
    cp = fmaf(cp, r2, 4.1666646237e-02f);
    const float c0 = fmaf(r2 * r2, cp, fmaf(-0.5f, r2, 1.f));
    const float s1 = (q & 1) ? c0 : s0, c1 = (q & 1) ? s0 : c0;
    sn = (q & 2) ? -s1 : s1;
    cs = ((q + 1) & 2) ? -c1 : c1;
}

// The same for arguments already known to lie in [-pi/4, pi/4] (the usual case: |k0 dz dn| << 1).
__device__ __forceinline__ void screen_sincos_small(float r, float &sn, float &cs) {
    const float r2 = r * r;
    float sp = fmaf(-1.9513932562e-04f, r2, 8.3321482563e-03f);
    sp = fmaf(sp, r2, -1.6666654339e-01f);
    sn = fmaf(r * r2, sp, r);
    float cp = fmaf(2.4435851735e-05f, r2, -1.3887341487e-03f);
    cp = fmaf(cp, r2, 4.1666646237e-02f);
    cs = fmaf(r2 * r2, cp, fmaf(-0.5f, r2, 1.f));
}

// (cos r, sin r) for r in [-pi/4, pi/4]: the two Horner chains of screen_sincos_small as packed
// instructions (same operations per lane, hence the same bits), for code with registers to spare.
__device__ __forceinline__ cf screen_cossin_small_packed(float r) {
    const float r2 = r * r;
    u64 p = fma2(pk2(r2, r2), pk2(2.4435851735e-05f, -1.9513932562e-04f), pk2(-1.3887341487e-03f, 8.3321482563e-03f));
    p = fma2(p, pk2(r2, r2), pk2(4.1666646237e-02f, -1.6666654339e-01f));
    const u64 m = mul2(pk2(r2, r), pk2(r2, r2));                 // (r2 r2, r r2)
    return up2(fma2(m, p, pk2(fmaf(-0.5f, r2, 1.f), r)));
}

// Pointwise factors of the unit the thread works on, slot (jp, m) -> pw[(jp*P + m) * kThreads16]:
// kind 1: exp(i (pb dn + pa)) at pixel n = q(jp) + 256 m of row `unit` of a dn slice (bb.h step 4);
// kind 2: table value H[n][column] of column tile `unit` (bb.h step 2).  Runs off the critical
// path where it can (while a grid barrier is pending).
template <int P, int CW, bool ROW, int NX>
__device__ __forceinline__ void fill_pw16(int kind, const void *src, int unit, float pa, float pb, cf *pw, bool noscreen) {
    const Team16<P, CW> tm;
    constexpr int JP = 16 / P;
    if (kind == 1) {
        const float *dnp = reinterpret_cast<const float *>(src) + (long long)unit * NX;
        float x[16];
#pragma unroll
        for (int jp = 0; jp < JP; ++jp)
#pragma unroll
            for (int m = 0; m < P; ++m) x[jp * P + m] = noscreen ? 0.f : __ldcs(dnp + tm.q(jp) + kL * m);
        float amax = 0.f;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            x[i] = fmaf(pb, x[i], pa);
            amax = fmaxf(amax, fabsf(x[i]));
        }
        if (__all_sync(__activemask(), amax <= 0.78539816f)) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                float s, c;
                screen_sincos_small(x[i], s, c);
                pw[i * kThreads16] = make_float2(c, s);
            }
        } else {
#pragma unroll 2
            for (int i = 0; i < 16; ++i) {
                float s, c;
                screen_sincos(x[i], s, c);
                pw[i * kThreads16] = make_float2(c, s);
            }
        }
    } else {
        const cf *hp = reinterpret_cast<const cf *>(src) + (long long)unit * CW + tm.col;
#pragma unroll
        for (int jp = 0; jp < JP; ++jp)
#pragma unroll
            for (int m = 0; m < P; ++m)
                pw[(jp * P + m) * kThreads16] = __ldg(hp + (long long)(tm.q(jp) + kL * m) * NX);
    }
}

// Batch kernel: screen factors of ALL rows this CTA owns, pw[rl * NX + n] = exp(i (pb dn + pa)) at
// pixel n of row a0 + rl, staged by the whole CTA (coalesced dn reads) and shared by the teams that
// apply them to the B fields.
template <int NX, int NY>
__device__ __forceinline__ void stage_rows_screen(const KParams &K, const Phase16 &d, cf *pw) {
    const int a0 = (int)((unsigned)NY * blockIdx.x / gridDim.x);
    const int a1 = (int)((unsigned)NY * (blockIdx.x + 1) / gridDim.x);
    const int total = (a1 - a0) * NX;
    const float *dnp = reinterpret_cast<const float *>(d.src) + (long long)a0 * NX;
#pragma unroll 4
    for (int idx = threadIdx.x; idx < total; idx += kThreads16) {
        const float a = fmaf(K.phase_b, K.noscreen ? 0.f : __ldcs(dnp + idx), d.pa);
        float s, c;
        if (__all_sync(__activemask(), fabsf(a) <= 0.78539816f)) screen_sincos_small(a, s, c);
        else screen_sincos(a, s, c);
        pw[idx] = make_float2(c, s);
    }
}

// Single-field kernel, column phase: a CTA that owns fewer column tiles than it has column teams (the
// usual case on an oversampled grid, where the evanescent band is pruned: 144 live tiles on 148 SMs at
// 1024^2) has idle warps.  They compute the screen factors exp(i (pb dn + pa)) of the CTA's rows for
// the NEXT row phase into the thread-private columns of the row teams (slot (jp, m) of row thread
// (team rl, class c, lane t) <- pixel n = t + 16 (PX jp + c) + 256 m of row r0 + rl), so that this
// work leaves the critical path between two phases (profiles/r02: 1.4 us behind every row phase).
template <int PX, int NX, int NY, int TEAMC>
__device__ __forceinline__ void stage_screen_by_idle_warps(const KParams &K, const Phase16 &dS, cf *sm_pwS) {
    typedef Team16<PX, 1> TR;
    constexpr int PER = (NX + TEAMC - 1) / TEAMC;              // pixels of a row per staging thread
    constexpr int RCH = 8;                                     // rows in flight (all loads issued before the first use)
    const int r0 = (int)((unsigned)NY * blockIdx.x / gridDim.x);
    const int r1 = (int)((unsigned)NY * (blockIdx.x + 1) / gridDim.x);
    const int rows = min(r1 - r0, TR::NTEAM);
    const int s = (int)threadIdx.x - (kThreads16 - TEAMC);     // the last column team stages
    const float *dnp = reinterpret_cast<const float *>(dS.src) + (long long)r0 * NX + s;
    const float pa = dS.pa, pb = K.phase_b;
#pragma unroll 1
    for (int rb = 0; rb < rows; rb += RCH) {
        float x[RCH][PER];
#pragma unroll
        for (int rl = 0; rl < RCH; ++rl)
#pragma unroll
            for (int k = 0; k < PER; ++k)
                x[rl][k] = (rb + rl < rows && s + k * TEAMC < NX && !K.noscreen) ? __ldcs(dnp + (rb + rl) * NX + k * TEAMC) : 0.f;
        // ONE decision for the whole chunk (small arguments: the compact packed path), so that the code
        // the warp walks through stays short: a vote and both paths per value made the staging
        // instruction-fetch bound (5 us for 28 values per thread)
        float amax = 0.f;
#pragma unroll
        for (int rl = 0; rl < RCH; ++rl)
#pragma unroll
            for (int k = 0; k < PER; ++k) {
                x[rl][k] = fmaf(pb, x[rl][k], pa);
                amax = fmaxf(amax, fabsf(x[rl][k]));
            }
        const bool small = __all_sync(__activemask(), amax <= 0.78539816f);
        if (small) {
#pragma unroll
            for (int rl = 0; rl < RCH; ++rl) {
                if (rb + rl < rows) {
#pragma unroll
                    for (int k = 0; k < PER; ++k) {
                        const int n = s + k * TEAMC;
                        if (n < NX) {
                            const int m = n >> 8, q = n & 255, t = q & 15, z = q >> 4, c = z % PX, jp = z / PX;
                            sm_pwS[(jp * PX + m) * kThreads16 + (rb + rl) * TR::TEAM + c * 16 + t] = screen_cossin_small_packed(x[rl][k]);
                        }
                    }
                }
            }
        } else {
#pragma unroll 1
            for (int i = 0; i < RCH * PER; ++i) {
                const int rl = i / PER, k = i % PER, n = s + k * TEAMC;
                if (rb + rl < rows && n < NX) {
                    const int m = n >> 8, q = n & 255, t = q & 15, z = q >> 4, c = z % PX, jp = z / PX;
                    float sn, cs;
                    float a = 0.f;
#pragma unroll
                    for (int u = 0; u < RCH * PER; ++u) a = (u == i) ? x[u / PER][u % PER] : a;     // registers, not a local array
                    screen_sincos(a, sn, cs);
                    sm_pwS[(jp * PX + m) * kThreads16 + (rb + rl) * TR::TEAM + c * 16 + t] = make_float2(cs, sn);
                }
            }
        }
    }
}

// ----------------------------------------------------------------------------------------
// One phase over the lines (rows, or tiles of CW columns) this CTA owns.
//   ROW : P = PX, CW = 1, signs (+1, -1);  column: P = PY, CW = 8 or 4, signs (-1, +1).
// ----------------------------------------------------------------------------------------
template <int P, int CW, bool ROW, int NX, int NY, bool BATCH>
__device__ __forceinline__ void run_phase16(const KParams &K, const Phase16 &d, const cf *sm_tw, const cf *sm_twc,
                                            cf *sm_y, cf *sm_pw, PwTag &tag, UnitCache &uc, int Fin, int cwc,
                                            unsigned long long *sm_mbar = nullptr, int pstage = -1,
                                            cf *sm_pwS = nullptr, PwTag *tagS = nullptr) {
    typedef Team16<P, CW> TM;
    constexpr int S1 = ROW ? +1 : -1, S2 = -S1;
    constexpr int JP = TM::JP;
    constexpr long long NS = ROW ? 1 : NX;               // element stride of the line index
    constexpr long long CS = ROW ? kL : NX;              // class stride: class-major (rows) / interleaved (columns)
    constexpr long long IS = ROW ? 1 : (long long)P * NX;   // stride inside a class
    const TM tm;
    // Column phase of a single field: the tile request goes out before anything else is computed (the
    // team's first tile is known from the previous step unless the live band changed): the L2 -> shared
    // memory copy is ~1 us of pure latency at the head of the phase.
    bool tma_issued = false;
    if constexpr (!ROW && !BATCH) {
        if (K.use_tma && uc.F == Fin && uc.a0 + tm.team < uc.a1) {
            if (threadIdx.x % TM::TEAM == 0) {
                cf *stage0 = sm_y + tm.team * (TM::TEAM * 17);
                asm volatile("fence.proxy.async;" ::: "memory");
                mbar_expect_tx(sm_mbar + tm.team, (unsigned)(P * kL * CW * sizeof(cf)));
#pragma unroll
                for (int cc = 0; cc < P; ++cc) tma_load_4d(stage0 + cc * kL * CW, &K.tmap, uc.u0 * CW, cc, 0, 0, sm_mbar + tm.team);
            }
            tma_issued = true;
        }
    }
    // rows: all of them; columns: the live tiles of this step (Fin), spread evenly over the CTAs
    constexpr int CWL = CW == 8 ? 3 : (CW == 4 ? 2 : 0);
    typedef LiveCols<ROW ? 1 : (NX / kL)> LV;
    if (uc.F != Fin) {
        const LV lv(Fin, NX, CWL);
        const int NU0 = ROW ? NY : lv.total();
        uc.a0 = (int)((unsigned)NU0 * blockIdx.x / gridDim.x);              // NU <= 1024: fits 32 bits
        uc.a1 = (int)((unsigned)NU0 * (blockIdx.x + 1) / gridDim.x);
        uc.u0 = ROW ? uc.a0 + tm.team : lv.tile(uc.a0 + tm.team);
        // row phase: which of the thread's 16 sub-line elements sit in live column tiles on input
        // (what the previous column phase wrote; the rest is stale and stands for zeros)
        if constexpr (ROW) uc.lmask = live_mask16<P>(Fin, NX, tm.c, tm.t, cwc == 4 ? 2 : 3);
        uc.F = Fin;
    }
    const int a0 = uc.a0, a1 = uc.a1;
    const unsigned lmask = uc.lmask;
    if constexpr (!ROW && !BATCH) {
        // idle column teams stage the screen factors of the next row phase (see stage_screen_by_idle_warps)
        // pstage: the row phase after this column phase (it applies dn slice pstage / 2 - 1), or -1
        const int busy = min(a1 - a0, TM::NTEAM);
        const int jstage = pstage >= 0 ? row_step(K, pstage >> 1) : -1;
        const void *src_stage = jstage >= 0 ? K.dn + (long long)(jstage - K.j_base) * ((long long)NX * NY) : nullptr;
        if (src_stage != nullptr && busy < TM::NTEAM && tagS->src != src_stage) {
            if (tm.team == TM::NTEAM - 1) stage_screen_by_idle_warps<NX / kL, NX, NY, TM::TEAM>(K, decode_phase16(K, pstage), sm_pwS);
            typedef Team16<NX / kL, 1> TR;
            const int tr = (int)threadIdx.x / TR::TEAM;
            const int r0 = (int)((unsigned)NY * blockIdx.x / gridDim.x), r1 = (int)((unsigned)NY * (blockIdx.x + 1) / gridDim.x);
            if (tr < TR::NTEAM && r0 + tr < r1) { tagS->src = src_stage; tagS->pix0 = r0 + tr; }
        }
    }
    const int NU = ROW ? NY : (BATCH ? LV(Fin, NX, CWL).total() : 0);
    cf *ybuf = sm_y + ((threadIdx.x / (16 * CW)) * (16 * 17 * CW)) + tm.col;        // one region per (team, class)
    cf *xbuf = sm_y + tm.team * (TM::TEAM * 17) + tm.col;                            // same memory, team's part
    cf *pw = sm_pw + threadIdx.x;
    const bool want_I = d.kind == 1 && K.inten != nullptr;
    const bool accumulate = (K.flags & 1u) != 0;
    // batch kernel: units are (line, field) pairs, fields fastest, so that the teams of a CTA share
    // the pointwise factors of a line; the summed intensity of a row is accumulated in shared
    // memory (acc, floats, in the buffer the propagator values use during column phases)
    const int B = BATCH ? K.B : 1;
    const long long npx = (long long)NX * NY;
    const bool summed = BATCH && ROW && want_I && !(K.flags & 2u) && K.B > 1;
    float *acc = reinterpret_cast<float *>(sm_pw - Smem16<NX / kL, NY / kL>::kPw);   // = the H buffer (ROW: sm_pw is the screen buffer)
    if constexpr (BATCH && ROW) {
        if (d.kind == 1 && tag.src != d.src) {                 // CTA-uniform: not staged during the barrier
            stage_rows_screen<NX, NY>(K, d, sm_pw);
            tag.src = d.src;
            __syncthreads();
        }
        if (summed) {
            for (int idx = threadIdx.x; idx < (a1 - a0) * NX; idx += kThreads16) acc[idx] = 0.f;
            __syncthreads();
        }
    }
    const HalfWarpSync hsync{0xFFFFu << (16 * ((threadIdx.x >> 4) & 1))};
    // hardware barriers: 0 = CTA, 1 .. NTEAM = teams, above = (team, class) groups of a column tile
    // (one class: the class group is the team)
    const ClassSync<16 * CW> tsync{P == 1 ? 1 + tm.team : 1 + TM::NTEAM + (int)threadIdx.x / (16 * CW)};
    static_assert(ROW || ((16 * CW) % 32 == 0 && (P == 1 ? TM::NTEAM : TM::NTEAM + kThreads16 / (16 * CW)) <= 15), "barrier ids");

    const int k0 = BATCH ? (ROW ? a0 * B : (int)(((long long)NU * B * blockIdx.x) / gridDim.x)) : a0;
    const int k1 = BATCH ? (ROW ? a1 * B : (int)(((long long)NU * B * (blockIdx.x + 1)) / gridDim.x)) : a1;
#pragma unroll 1
    for (int k = k0 + tm.team; k < k1; k += TM::NTEAM) {
        const int m = BATCH ? k / B : k, b = BATCH ? k - m * B : 0;
        const int u = ROW ? m : (!BATCH && k == k0 + tm.team ? uc.u0 : LV(Fin, NX, CWL).tile(m));
        if constexpr (BATCH && ROW) {
            pw = sm_pw + (m - a0) * NX;                         // the row's factors, indexed by pixel
        } else if (d.kind != 0 && (tag.src != d.src || tag.pix0 != u)) {
            fill_pw16<P, CW, ROW, NX>(d.kind, d.src, u, d.pa, K.phase_b, pw, K.noscreen != 0);
            tag.src = d.src; tag.pix0 = u;
        }
        cf *line = K.field + b * npx + (ROW ? (long long)u * NX : (long long)u * CW + tm.col);
        cf v[16];
        bool loaded = false;
        if constexpr (!ROW) {
            if (K.use_tma) {
                // One thread asks the TMA unit for the P y-classes of the tile ([256][CW] each, into the
                // team's part of the transpose region); the 16 CW strided 8 CW-byte row segments per warp
                // load instruction, which kept the LSU busy for 0.5 us, become conflict-free LDS.
                cf *stage = sm_y + tm.team * (TM::TEAM * 17);
                unsigned long long *bar = sm_mbar + tm.team;
                if (threadIdx.x % TM::TEAM == 0 && (BATCH || !tma_issued)) {
                    // the tiles were written by other CTAs through the generic proxy (st.global, before the grid
                    // barrier) and the landing zone by this CTA: order both before the async-proxy copy.  The
                    // full proxy fence is needed once per phase (it costs ~0.1 us); later tiles only have to order
                    // this CTA's own shared-memory accesses.
                    if (k == k0 + tm.team) asm volatile("fence.proxy.async;" ::: "memory");
                    else asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(bar, (unsigned)(P * kL * CW * sizeof(cf)));
#pragma unroll
                    for (int cc = 0; cc < P; ++cc) tma_load_4d(stage + cc * kL * CW, &K.tmap, u * CW, cc, 0, b, bar);
                }
                if constexpr (!BATCH) tma_issued = false;   // (only the first tile of a phase is requested early)
                if (!mbar_wait(bar, uc.tma_parity)) {       // the copy never arrived: flag it and leave the phase; the grid
                    atomicExch(K.status, 2);                // barrier's watchdog sees the flag and ends the kernel
                    return;
                }
                uc.tma_parity ^= 1u;
#pragma unroll
                for (int i = 0; i < 16; ++i) v[i] = stage[(tm.c * kL + tm.t + 16 * i) * CW + tm.col];
                tm.sync();                              // staged tile read: the region goes back to the transposes
                loaded = true;
            }
        }
        if (d.first) {
            if (!loaded) {
                const cf *src = line + tm.c * CS + tm.t * IS;
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    v[i] = make_float2(0.f, 0.f);
                    if (!ROW || ((lmask >> i) & 1u)) v[i] = ld_cg(src + 16 * IS * i);
                }
            }
            if constexpr (ROW) subline_fft<S1, CW>(v, sm_tw, ybuf, tm.t, hsync);
            else subline_fft<S1, CW>(v, sm_tw, ybuf, tm.t, tsync);
            if constexpr (P > 1) {
                // exchange: (class, 16 indices) -> (group, 16/P indices of every class)
                tm.sync();                                  // the team's transposes have been read
#pragma unroll
                for (int j = 0; j < 16; ++j) xbuf[((tm.c * 16 + j) * 16 + tm.t) * CW] = v[j];
                tm.sync();
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int cc = 0; cc < P; ++cc)
                        v[jp * P + cc] = xbuf[((cc * 16 + P * jp + tm.c) * 16 + tm.t) * CW];
#pragma unroll
                for (int jp = 0; jp < JP; ++jp) {
#pragma unroll
                    for (int cc = 1; cc < P; ++cc)
                        v[jp * P + cc] = cmul_s<S1>(v[jp * P + cc], sm_twc[(cc - 1) * kL + tm.q(jp)]);
                    class_dft<P, S1>(&v[jp * P]);
                }
            }
        } else {
#pragma unroll
            for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                for (int m = 0; m < P; ++m) v[jp * P + m] = ld_cg(line + (tm.q(jp) + kL * m) * NS);
        }
        // v[jp*P + m] is element n = q(jp) + 256 m of the line, in its natural (x- or ky-) order
        if (d.kind == 1) {
            // u = value * screen (bb.h step 4), intensity (step 5)
            if constexpr (BATCH) {
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int mm = 0; mm < P; ++mm) v[jp * P + mm] = cmul(v[jp * P + mm], pw[tm.q(jp) + kL * mm]);
            } else {
#pragma unroll
                for (int i = 0; i < 16; ++i) v[i] = cmul(v[i], pw[i * kThreads16]);
            }
            if (summed) {
                float *ar = acc + (m - a0) * NX;
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int mm = 0; mm < P; ++mm) {
                        const cf w = v[jp * P + mm];
                        atomicAdd(ar + tm.q(jp) + kL * mm, fmaf(w.x, w.x, w.y * w.y));
                    }
            } else if (want_I) {
                float *ip = K.inten + d.slice + (long long)u * NX
                            + ((K.flags & 2u) ? (long long)b * K.inten_bstride : 0);
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int mm = 0; mm < P; ++mm) {
                        const cf w = v[jp * P + mm];
                        float I = fmaf(w.x, w.x, w.y * w.y);
                        float *a = ip + tm.q(jp) + kL * mm;
                        if (accumulate) I += *a;
                        __stcg(a, I);
                    }
            }
        } else if (d.kind == 2) {
            // U * H (bb.h step 2)
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = cmul(v[i], pw[i * kThreads16]);
        }
        if (d.second) {
            if constexpr (P > 1) {
#pragma unroll
                for (int jp = 0; jp < JP; ++jp) {
                    class_dft<P, S2>(&v[jp * P]);
#pragma unroll
                    for (int cc = 1; cc < P; ++cc)
                        v[jp * P + cc] = cmul_s<S2>(v[jp * P + cc], sm_twc[(cc - 1) * kL + tm.q(jp)]);
                }
                // (no barrier here: a thread writes exactly the slots it read in the first exchange, and nobody
                // else touches them in between)
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int cc = 0; cc < P; ++cc)
                        xbuf[((cc * 16 + P * jp + tm.c) * 16 + tm.t) * CW] = v[jp * P + cc];
                tm.sync();
#pragma unroll
                for (int j = 0; j < 16; ++j) v[j] = xbuf[((tm.c * 16 + j) * 16 + tm.t) * CW];
            }
            tm.sync();                                      // region free again for the transposes
            if constexpr (ROW) subline_fft<S2, CW>(v, sm_tw, ybuf, tm.t, hsync);
            else subline_fft<S2, CW>(v, sm_tw, ybuf, tm.t, tsync);
            // (a TMA store of the tile, the mirror image of its load, was slower: the team waits for its completion)
            cf *dst = line + tm.c * CS + tm.t * IS;
#pragma unroll
            for (int i = 0; i < 16; ++i) st_cg(dst + 16 * IS * i, v[i]);     // dead columns too: predicated
                                                                              // stores cost more than they save
        } else {
#pragma unroll
            for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                for (int m = 0; m < P; ++m) st_cg(line + (tm.q(jp) + kL * m) * NS, v[jp * P + m]);
        }
        tm.sync();                                          // buffers free for the team's next unit
    }
    if constexpr (BATCH && ROW) {
        if (summed) {
            // I[j] (+)= sum over the fields (bb.h step 5): the CTA's rows are contiguous in the slice
            __syncthreads();
            float *ip = K.inten + d.slice + (long long)a0 * NX;
            for (int idx = threadIdx.x; idx < (a1 - a0) * NX; idx += kThreads16) {
                float I = acc[idx];
                if (accumulate) I += ip[idx];
                __stcs(ip + idx, I);
            }
        }
    }
}

// Stage the pointwise factors of phase `d` for the unit this thread will work on, unless the
// buffer already holds them.  Called while a grid barrier is pending.
template <int P, int CW, bool ROW, int NX, int NY, bool BATCH>
__device__ __forceinline__ void prefill_phase16(const KParams &K, const Phase16 &d, cf *sm_pw, PwTag &tag, int Fin) {
    typedef Team16<P, CW> TM;
    if (d.kind == 0) return;
    if constexpr (BATCH && ROW) {
        if (tag.src != d.src) {
            stage_rows_screen<NX, NY>(K, d, sm_pw);
            tag.src = d.src;
        }
        return;
    }
    const TM tm;
    const LiveCols<ROW ? 1 : (NX / kL)> lv(Fin, NX, CW == 8 ? 3 : (CW == 4 ? 2 : 0));
    const int NU = ROW ? NY : lv.total();
    const int a0 = (int)((unsigned)NU * blockIdx.x / gridDim.x);              // NU <= 1024: fits 32 bits
    const int a1 = (int)((unsigned)NU * (blockIdx.x + 1) / gridDim.x);
    const int B = BATCH ? K.B : 1;
    const int k0 = BATCH ? (int)(((long long)NU * B * blockIdx.x) / gridDim.x) : a0;
    const int k1 = BATCH ? (int)(((long long)NU * B * (blockIdx.x + 1)) / gridDim.x) : a1;
    const int k = k0 + tm.team;
    if (k >= k1) return;
    const int m = BATCH ? k / B : k;
    const int u = ROW ? m : lv.tile(m);
    if (tag.src == d.src && tag.pix0 == u) return;
    fill_pw16<P, CW, ROW, NX>(d.kind, d.src, u, d.pa, K.phase_b, sm_pw + threadIdx.x, K.noscreen != 0);
    tag.src = d.src; tag.pix0 = u;
}

// CWC: columns per column tile (8, or 4 when few columns are live); BATCH: several fields (KParams::B)
template <int PX, int PY, int CWC, bool BATCH>
__global__ void __launch_bounds__(kThreads16, 1) bpm16_kernel(const __grid_constant__ KParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    using L = Smem16<PX, PY>;
    constexpr int NX = kL * PX, NY = kL * PY;
    cf *sm_tw = reinterpret_cast<cf *>(smem_raw);
    cf *sm_twcx = sm_tw + L::kTw;
    cf *sm_twcy = sm_twcx + (PX - 1) * kL;
    cf *sm_y = sm_twcy + (PY - 1) * kL;
    cf *sm_pwH = sm_y + L::kY;          // propagator values of this CTA's column tiles: stay put while the
                                        // reference index (the table) does not change
    cf *sm_pwS = sm_pwH + L::kPw;       // screen factors of this CTA's rows for the NEXT row phase
    int *sm_abort = reinterpret_cast<int *>(sm_pwS + L::kPw);
    unsigned long long *sm_mbar = reinterpret_cast<unsigned long long *>(sm_abort + 2);   // one TMA barrier per column team
    if (threadIdx.x < 8) mbar_init(sm_mbar + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");

    for (int i = threadIdx.x; i < L::kTw; i += kThreads16) sm_tw[i] = P.tw256[i];
    for (int i = threadIdx.x; i < (PX - 1) * kL; i += kThreads16) sm_twcx[i] = P.twcx[i];
    for (int i = threadIdx.x; i < (PY - 1) * kL; i += kThreads16) sm_twcy[i] = P.twcy[i];
    __syncthreads();

    PwTag tagH = {nullptr, -1}, tagS = {nullptr, -1};
    UnitCache ucR, ucC;
    // largest live |kx bin| of the step whose column phase wrote the field a phase reads (row phase)
    // or whose tiles it computes (column phase); fetched one phase ahead so that the global load is not on the critical path
    auto live_in = [&](int p) {
        const bool row = (p & 1) == 0;
        return row ? ((p >> 1) >= 1 ? P.fmax[col_step(P, (p >> 1) - 1)] : NX / 2) : P.fmax[col_step(P, p >> 1)];
    };
    int Fa_next = live_in(P.p0);
    Phase16 d_next = decode_phase16(P, P.p0);
    const int r0 = (int)((unsigned)NY * blockIdx.x / gridDim.x);          // rows of this CTA (row phases)
    const int r1 = (int)((unsigned)NY * (blockIdx.x + 1) / gridDim.x);
    unsigned nbar = 0;
    // optional timeline (bb_probe_trace): per phase and CTA, clock64 at phase start / work done /
    // arrived / prefilled / released, and the global timer at release
    long long *tr = P.trace ? P.trace + ((long long)(P.p0 - P.trace_p0) * gridDim.x + blockIdx.x) * 6 : nullptr;
    const bool tracer = tr != nullptr && threadIdx.x == 0;
#pragma unroll 1
    for (int p = P.p0; p < P.p1; ++p) {
        const Phase16 d = d_next;              // decoded while the previous barrier was pending
        if (tracer) tr[0] = clock64();
        if (d.is_row && p + 2 < P.p1) {
            // the dn rows this CTA turns into screen factors at the end of this phase (for the row
            // phase after next): start them on their way from HBM to L2 now, one bulk prefetch per row
            const int jn = row_step(P, (p >> 1) + 1);
            if ((int)threadIdx.x < r1 - r0 && jn >= 0 && !P.noscreen) {
                const float *row = P.dn + (long long)(jn - P.j_base) * ((long long)NX * NY)
                                   + (long long)(r0 + threadIdx.x) * NX;
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(row), "r"(NX * 4) : "memory");
            }
        }
        // largest live |kx bin| of the step whose column phase wrote / will read the field
        const int Fa = Fa_next;
        if (d.is_row) {
            run_phase16<PX, 1, true, NX, NY, BATCH>(P, d, sm_tw, sm_twcx, sm_y, sm_pwS, tagS, ucR, Fa, CWC);
        } else {
            run_phase16<PY, CWC, false, NX, NY, BATCH>(P, d, sm_tw, sm_twcy, sm_y, sm_pwH, tagH, ucC, Fa, CWC, sm_mbar,
                                                       (!BATCH && p + 1 < P.p1) ? p + 1 : -1, sm_pwS, &tagS);
        }
        if (tracer) tr[1] = clock64();
        if (BATCH && d.is_row && d.kind == 1 && P.inten != nullptr && !(P.flags & 2u) && P.B > 1)
            tagH.src = nullptr;                // the intensity sums used the propagator buffer
        if (p + 1 < P.p1) {
            ++nbar;
            grid_arrive(P.bar);
            if (tracer) tr[2] = clock64();
            Fa_next = live_in(p + 1);
            d_next = decode_phase16(P, p + 1);   // its global loads (table pointer, phase offset) overlap the barrier
            // While the barrier is pending, stage what does not depend on the field.  After a row
            // phase: the propagator values of the coming column phase (only when the table changed)
            // and the screen factors of the NEXT row phase (its dn slice is known), so that the
            // sin/cos work has a whole barrier + column phase of slack.  After a column phase:
            // the screen factors, if they are not there yet (first row phase of a launch).
            if (d.is_row) {
                const int Fn = Fa_next;
                prefill_phase16<PY, CWC, false, NX, NY, BATCH>(P, d_next, sm_pwH, tagH, Fn);
                // screen factors of the row phase after next: here, unless the coming column phase has
                // idle warps for them (same live band as the last column phase, which had an idle team)
                const bool col_stages = !BATCH && ucC.F == Fn && (ucC.a1 - ucC.a0) < Team16<PY, CWC>::NTEAM;
                if (p + 2 < P.p1 && !col_stages) prefill_phase16<PX, 1, true, NX, NY, BATCH>(P, decode_phase16(P, p + 2), sm_pwS, tagS, 0);
            } else {
                prefill_phase16<PX, 1, true, NX, NY, BATCH>(P, d_next, sm_pwS, tagS, 0);
            }
            if (tracer) tr[3] = clock64();
            if (grid_wait(P.bar, nbar * gridDim.x, P.status, sm_abort)) return;
            if (tracer) {
                tr[4] = clock64();
                long long g;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g));
                tr[5] = g;
                tr += 6 * gridDim.x;
            }
        }
    }
}

}  // namespace bb
