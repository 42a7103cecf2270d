// bb_kernels16.cuh -- the BPM step kernel with 16 points per thread (Nx, Ny in {256, 512, 1024}, B = 1).
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
constexpr int kCW16 = 8;                       // columns per column tile: 64-byte row segments

template <int PX, int PY>
struct Smem16 {
    static constexpr int kTw = 256;                                   // sub-line twiddles [16][16]
    static constexpr int kTwc = (PX - 1) * kL + (PY - 1) * kL;          // class twiddles, x then y
    static constexpr int kY = (kThreads16 / 16) * 16 * 17;              // sub-line transposes
    static constexpr int kX = kThreads16 * 16;                          // class exchange
    static constexpr int kPw = kThreads16 * 16;                         // pointwise factors
    static constexpr size_t bytes = (size_t)(kTw + kTwc + kY + kX + kPw) * sizeof(cf) + 16;
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
        if (d.first) {
            const int j = (p >> 1) - 1;
            d.kind = 1;
            d.slice = (long long)(j - P.j_base) * ((long long)P.Nx * P.Ny);
            d.src = P.dn + d.slice;
            d.pa = P.phase_a[j];
        }
    } else {
        d.first = d.second = true;
        d.kind = 2;
        d.src = P.htab[p >> 1];
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

struct HalfWarpSync {
    unsigned mask;
    __device__ __forceinline__ void operator()() const { __syncwarp(mask); }
};
template <class T>
struct TeamSync {
    const T &tm;
    __device__ __forceinline__ void operator()() const { tm.sync(); }
};

// Pointwise factors of the unit the thread works on, slot (jp, m) -> pw[(jp*P + m) * kThreads16]:
// kind 1: exp(i (pb dn + pa)) at pixel n = q(jp) + 256 m of row `unit` of a dn slice (bb.h step 4);
// kind 2: table value H[n][column] of column tile `unit` (bb.h step 2).  Runs off the critical
// path where it can (while a grid barrier is pending).
template <int P, int CW, bool ROW, int NX>
__device__ __forceinline__ void fill_pw16(int kind, const void *src, int unit, float pa, float pb, cf *pw) {
    const Team16<P, CW> tm;
    constexpr int JP = 16 / P;
    if (kind == 1) {
        const float *dnp = reinterpret_cast<const float *>(src) + (long long)unit * NX;
        float x[16];
#pragma unroll
        for (int jp = 0; jp < JP; ++jp)
#pragma unroll
            for (int m = 0; m < P; ++m) x[jp * P + m] = __ldcs(dnp + tm.q(jp) + kL * m);
#pragma unroll 4
        for (int i = 0; i < 16; ++i) {
            float s, c;
            sincosf(fmaf(pb, x[i], pa), &s, &c);
            pw[i * kThreads16] = make_float2(c, s);
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

// ----------------------------------------------------------------------------------------
// One phase over the lines (rows, or tiles of CW columns) this CTA owns.
//   ROW : P = PX, CW = 1, signs (+1, -1);  column: P = PY, CW = kCW16, signs (-1, +1).
// ----------------------------------------------------------------------------------------
template <int P, int CW, bool ROW, int NX, int NY>
__device__ __forceinline__ void run_phase16(const KParams &K, const Phase16 &d, const cf *sm_tw, const cf *sm_twc,
                                            cf *sm_y, cf *sm_x, cf *sm_pw, PwTag &tag) {
    typedef Team16<P, CW> TM;
    constexpr int S1 = ROW ? +1 : -1, S2 = -S1;
    constexpr int JP = TM::JP;
    constexpr long long NS = ROW ? 1 : NX;               // element stride of the line index
    constexpr long long CS = ROW ? kL : NX;              // class stride: class-major (rows) / interleaved (columns)
    constexpr long long IS = ROW ? 1 : (long long)P * NX;   // stride inside a class
    constexpr int NU = ROW ? NY : NX / CW;
    const TM tm;
    const int a0 = (int)(((long long)NU * blockIdx.x) / gridDim.x);
    const int a1 = (int)(((long long)NU * (blockIdx.x + 1)) / gridDim.x);
    cf *ybuf = sm_y + ((threadIdx.x / (16 * CW)) * (16 * 17 * CW)) + tm.col;        // one region per (team, class)
    cf *xbuf = sm_x + tm.team * (TM::TEAM * 16) + tm.col;
    cf *pw = sm_pw + threadIdx.x;
    const bool want_I = d.kind == 1 && K.inten != nullptr;
    const bool accumulate = (K.flags & 1u) != 0;
    const HalfWarpSync hsync{0xFFFFu << (16 * ((threadIdx.x >> 4) & 1))};
    const TeamSync<TM> tsync{tm};

#pragma unroll 1
    for (int u = a0 + tm.team; u < a1; u += TM::NTEAM) {
        if (d.kind != 0 && (tag.src != d.src || tag.pix0 != u)) {
            fill_pw16<P, CW, ROW, NX>(d.kind, d.src, u, d.pa, K.phase_b, pw);
            tag.src = d.src; tag.pix0 = u;
        }
        cf *line = K.field + (ROW ? (long long)u * NX : (long long)u * CW + tm.col);
        cf v[16];
        if (d.first) {
            const cf *src = line + tm.c * CS + tm.t * IS;
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = ld_cg(src + 16 * IS * i);
            if constexpr (ROW) subline_fft<S1, CW>(v, sm_tw, ybuf, tm.t, hsync);
            else subline_fft<S1, CW>(v, sm_tw, ybuf, tm.t, tsync);
            if constexpr (P > 1) {
                // exchange: (class, 16 indices) -> (group, 16/P indices of every class)
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
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = cmul(v[i], pw[i * kThreads16]);
            if (want_I) {
                float *ip = K.inten + d.slice + (long long)u * NX;
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int m = 0; m < P; ++m) {
                        const cf w = v[jp * P + m];
                        float I = fmaf(w.x, w.x, w.y * w.y);
                        float *a = ip + tm.q(jp) + kL * m;
                        if (accumulate) I += *a;
                        __stcs(a, I);
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
                tm.sync();                                  // every read of the first exchange is done
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int cc = 0; cc < P; ++cc)
                        xbuf[((cc * 16 + P * jp + tm.c) * 16 + tm.t) * CW] = v[jp * P + cc];
                tm.sync();
#pragma unroll
                for (int j = 0; j < 16; ++j) v[j] = xbuf[((tm.c * 16 + j) * 16 + tm.t) * CW];
            }
            if constexpr (P == 1) tm.sync();                // transpose region: reads of the first transform are done
            if constexpr (ROW) subline_fft<S2, CW>(v, sm_tw, ybuf, tm.t, hsync);
            else subline_fft<S2, CW>(v, sm_tw, ybuf, tm.t, tsync);
            cf *dst = line + tm.c * CS + tm.t * IS;
#pragma unroll
            for (int i = 0; i < 16; ++i) st_cg(dst + 16 * IS * i, v[i]);
        } else {
#pragma unroll
            for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                for (int m = 0; m < P; ++m) st_cg(line + (tm.q(jp) + kL * m) * NS, v[jp * P + m]);
        }
        tm.sync();                                          // buffers free for the team's next unit
    }
}

template <int P, int CW, bool ROW, int NX, int NY>
__device__ __forceinline__ void prefill_phase16(const KParams &K, const Phase16 &d, cf *sm_pw, PwTag &tag) {
    typedef Team16<P, CW> TM;
    if (d.kind == 0) return;
    constexpr int NU = ROW ? NY : NX / CW;
    const TM tm;
    const int a0 = (int)(((long long)NU * blockIdx.x) / gridDim.x);
    const int a1 = (int)(((long long)NU * (blockIdx.x + 1)) / gridDim.x);
    const int u = a0 + tm.team;
    if (u >= a1 || (tag.src == d.src && tag.pix0 == u)) return;
    fill_pw16<P, CW, ROW, NX>(d.kind, d.src, u, d.pa, K.phase_b, sm_pw + threadIdx.x);
    tag.src = d.src; tag.pix0 = u;
}

template <int PX, int PY>
__global__ void __launch_bounds__(kThreads16, 1) bpm16_kernel(const KParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using L = Smem16<PX, PY>;
    constexpr int NX = kL * PX, NY = kL * PY;
    cf *sm_tw = reinterpret_cast<cf *>(smem_raw);
    cf *sm_twcx = sm_tw + L::kTw;
    cf *sm_twcy = sm_twcx + (PX - 1) * kL;
    cf *sm_y = sm_twcy + (PY - 1) * kL;
    cf *sm_x = sm_y + L::kY;
    cf *sm_pw = sm_x + L::kX;
    int *sm_abort = reinterpret_cast<int *>(sm_pw + L::kPw);

    for (int i = threadIdx.x; i < L::kTw; i += kThreads16) sm_tw[i] = P.tw256[i];
    for (int i = threadIdx.x; i < (PX - 1) * kL; i += kThreads16) sm_twcx[i] = P.twcx[i];
    for (int i = threadIdx.x; i < (PY - 1) * kL; i += kThreads16) sm_twcy[i] = P.twcy[i];
    __syncthreads();

    PwTag tag = {nullptr, -1};
    unsigned nbar = 0;
#pragma unroll 1
    for (int p = P.p0; p < P.p1; ++p) {
        const Phase16 d = decode_phase16(P, p);
        if (d.is_row) run_phase16<PX, 1, true, NX, NY>(P, d, sm_tw, sm_twcx, sm_y, sm_x, sm_pw, tag);
        else run_phase16<PY, kCW16, false, NX, NY>(P, d, sm_tw, sm_twcy, sm_y, sm_x, sm_pw, tag);
        if (p + 1 < P.p1) {
            ++nbar;
            grid_arrive(P.bar);
            const Phase16 dn = decode_phase16(P, p + 1);
            if (dn.is_row) prefill_phase16<PX, 1, true, NX, NY>(P, dn, sm_pw, tag);
            else prefill_phase16<PY, kCW16, false, NX, NY>(P, dn, sm_pw, tag);
            if (grid_wait(P.bar, nbar * gridDim.x, P.status, sm_abort)) return;
        }
    }
}

}  // namespace bb
