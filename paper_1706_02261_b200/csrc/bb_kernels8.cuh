// bb_kernels8.cuh -- the BPM step kernel with 8 points per thread (Nx, Ny in {256, 512, 1024, 2048}; single
// fields and batches).
//
// Same two-phase structure as bb_kernels.cuh:
//   column phase C_j : FFT_y  -> x H_j                          -> IFFT_y
//   row phase    R_j : IFFT_x -> x exp(i phi(dn[j-1])), |u|^2   -> FFT_x
// and the same decomposition of a line of N = 256 P points into P sub-lines ("classes") as
// bb_kernels16.cuh, with the radix-P butterfly that joins the classes fused with the pointwise step:
//
//   load classes -> P sub-line transforms -> exchange -> [twiddle, radix-P, POINTWISE, radix-P,
//   twiddle] -> exchange -> P sub-line transforms -> store classes
//
// but a sub-line is held by 32 threads x 8 points (bb_fft8.cuh: every radix-16 is shared by a pair of
// lanes through one shfl exchange), so a CTA has 1024 threads at <= 64 registers and an SM runs 28
// warps in a row phase of a 1024^2 grid instead of 14: the phases are bound by the latency of each
// warp's own instruction stream (profiles/r02_a), not by a throughput.
//
// Row phase: classes are kx mod P, and between the phases the field is kept kx-class-major in memory
// (kx = P k' + c at column c N/P + k'); the propagator table is built with the same column
// permutation.  Column phase: classes are y mod P (interleaved rows), natural order at both ends.
#pragma once
#include "bb_kernels16.cuh"
#include "bb_fft8.cuh"

namespace bb {

constexpr int kThreads8 = 1024;
constexpr int kSlots8 = 8;            // points per thread

template <int PX, int PY>
struct Smem8 {
    static constexpr int kTw = 256;                                   // sub-line twiddles [16][16]
    static constexpr int kTwc = (PX - 1) * kL + (PY - 1) * kL;        // class twiddles, x then y
    static constexpr int kY = (kThreads8 / 32) * 16 * 17;             // sub-line transposes; the class exchange and the
                                                                      // TMA landing zone of a team reuse the team's part
    static constexpr int kPw = kThreads8 * kSlots8;                   // pointwise factors: propagator values / screen
    static constexpr size_t bytes = (size_t)(kTw + kTwc + kY + 2 * kPw) * sizeof(cf) + 16 + 8 * 8;
};

// Thread roles inside the team that owns one line (row phase, CW = 1) or one tile of CW columns.
//   r = thread index in the team = 32 CW c + 32 w + lane;  lane = col + CW tl + 16 h;  t = (16 / CW) w + tl
//   after the class exchange the thread holds, for jp < 8 / P, sub-line index q(jp) = rr + 32 P jp of
//   every class (rr = r / CW).
template <int P, int CW>
struct Team8 {
    static constexpr int TEAM = 32 * P * CW;            // threads
    static constexpr int NTEAM_ALL = kThreads8 / TEAM;
    static constexpr int NTEAM = (TEAM > 32 && NTEAM_ALL > 14) ? 14 : NTEAM_ALL;   // teams that work (hardware barrier ids 1..14)
    static constexpr int JP = kSlots8 / P;
    static constexpr int QS = 32 * P;                   // stride of q between the slots jp
    int team, col, c, rr;
    Lane8 l;
    __device__ __forceinline__ Team8() {
        const int r = threadIdx.x % TEAM, lane = threadIdx.x & 31;
        team = threadIdx.x / TEAM;
        col = lane % CW;
        c = r / (32 * CW);
        rr = r / CW;
        l.h = lane >> 4;
        l.t = (16 / CW) * ((r / 32) % CW) + (lane / CW) % (16 / CW);
        l.s = l.h ? -1.f : 1.f;
    }
    __device__ __forceinline__ void sync() const {
        if constexpr (TEAM == 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(TEAM) : "memory");
    }
    __device__ __forceinline__ int q(int jp) const { return rr + QS * jp; }
    // line element (pixel / frequency) held in register `slot` at the pointwise step
    //   P > 1 (after the class exchange and the radix-P butterfly): slot = jp P + m -> q(jp) + 256 m
    //   P = 1 (no exchange; the split distribution of bb_fft8.cuh):  t + 16 (4 h + (slot & 3) + 8 (slot >> 2))
    __device__ __forceinline__ int pix(int slot) const {
        return P > 1 ? q(slot / P) + kL * (slot % P) : l.t + 16 * (4 * l.h + (slot & 3) + 8 * (slot >> 2));
    }
};

struct WarpSync {
    __device__ __forceinline__ void operator()() const { __syncwarp(); }
};
// The CW warps that share the transposes of one class of a column tile.
template <int THREADS>
struct GroupSync {
    int id;
    __device__ __forceinline__ void operator()() const {
        if constexpr (THREADS == 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(THREADS) : "memory");
    }
};

// Radix-P butterfly over P consecutive registers, natural order in and out (P = 1, 2, 4, 8).
template <int P, int SIGN>
__device__ __forceinline__ void class_dft_any(cf *w) {
    if constexpr (P == 8) class_dft8<SIGN>(w);
    else class_dft<P, SIGN>(w);
}

// Pointwise factors of the unit the thread works on, slot (jp, m) -> pw[(jp*P + m) * kThreads8]:
// kind 1: exp(i (pb dn + pa)) at pixel n = q(jp) + 256 m of row `unit` of a dn slice (bb.h step 4);
// kind 2: table value H[n][column] of column tile `unit` (bb.h step 2).
template <int P, int CW, bool ROW, int NX>
__device__ __forceinline__ void fill_pw8(int kind, const void *src, int unit, float pa, float pb, cf *pw, bool noscreen) {
    const Team8<P, CW> tm;
    if (kind == 1) {
        const float *dnp = reinterpret_cast<const float *>(src) + (long long)unit * NX;
        float x[kSlots8];
#pragma unroll
        for (int i = 0; i < kSlots8; ++i) x[i] = noscreen ? 0.f : __ldcs(dnp + tm.pix(i));
        float amax = 0.f;
#pragma unroll
        for (int i = 0; i < kSlots8; ++i) {
            x[i] = fmaf(pb, x[i], pa);
            amax = fmaxf(amax, fabsf(x[i]));
        }
        if (__all_sync(__activemask(), amax <= 0.78539816f)) {
#pragma unroll
            for (int i = 0; i < kSlots8; ++i) {
                float s, c;
                screen_sincos_small(x[i], s, c);
                pw[i * kThreads8] = make_float2(c, s);
            }
        } else {
#pragma unroll 2
            for (int i = 0; i < kSlots8; ++i) {
                float s, c;
                screen_sincos(x[i], s, c);
                pw[i * kThreads8] = make_float2(c, s);
            }
        }
    } else {
        const cf *hp = reinterpret_cast<const cf *>(src) + (long long)unit * CW + tm.col;
#pragma unroll
        for (int i = 0; i < kSlots8; ++i) pw[i * kThreads8] = __ldg(hp + (long long)tm.pix(i) * NX);
    }
}

// Batch kernel: screen factors of ALL rows this CTA owns, pw[rl * NX + n] = exp(i (pb dn + pa)) at
// pixel n of row a0 + rl, staged by the whole CTA and shared by the teams that apply them to the B fields.
template <int NX, int NY>
__device__ __forceinline__ void stage_rows_screen8(const KParams &K, const Phase16 &d, cf *pw) {
    const int a0 = (int)((unsigned)NY * blockIdx.x / gridDim.x);
    const int a1 = (int)((unsigned)NY * (blockIdx.x + 1) / gridDim.x);
    const int total = (a1 - a0) * NX;
    const float *dnp = reinterpret_cast<const float *>(d.src) + (long long)a0 * NX;
#pragma unroll 4
    for (int idx = threadIdx.x; idx < total; idx += kThreads8) {
        const float a = fmaf(K.phase_b, K.noscreen ? 0.f : __ldcs(dnp + idx), d.pa);
        float s, c;
        if (__all_sync(__activemask(), fabsf(a) <= 0.78539816f)) screen_sincos_small(a, s, c);
        else screen_sincos(a, s, c);
        pw[idx] = make_float2(c, s);
    }
}

// ----------------------------------------------------------------------------------------
// One phase over the lines (rows, or tiles of CW columns) this CTA owns.
//   ROW : P = PX, CW = 1, signs (+1, -1);  column: P = PY, CW = 8 or 4, signs (-1, +1).
// ----------------------------------------------------------------------------------------
template <int P, int CW, bool ROW, int NX, int NY, bool BATCH>
__device__ __forceinline__ void run_phase8(const KParams &K, const Phase16 &d, const cf *sm_tw, const cf *sm_twc,
                                           cf *sm_y, cf *sm_pw, PwTag &tag, UnitCache &uc, int Fin, int cwc,
                                           unsigned long long *sm_mbar = nullptr, float scale = 1.f) {
    typedef Team8<P, CW> TM;
    constexpr int S1 = ROW ? +1 : -1, S2 = -S1;
    constexpr int JP = TM::JP;
    constexpr long long NS = ROW ? 1 : NX;               // element stride of the line index
    constexpr long long CS = ROW ? kL : NX;              // class stride: class-major (rows) / interleaved (columns)
    constexpr long long IS = ROW ? 1 : (long long)P * NX;   // stride inside a class
    // transform programs (bb_fft2, bb_multiplex_*) keep kx in natural order: class c, index k' at P k' + c
    const long long CSr = (ROW && K.xnat) ? 1 : CS, ISr = (ROW && K.xnat) ? P : IS;
    const TM tm;
    if (tm.team >= TM::NTEAM) return;
    constexpr int CWL = CW == 8 ? 3 : (CW == 4 ? 2 : 0);
    typedef LiveCols<ROW ? 1 : (NX / kL)> LV;
    if (uc.F != Fin) {
        const LV lv(Fin, NX, CWL);
        const int NU0 = ROW ? NY : lv.total();
        uc.a0 = (int)((unsigned)NU0 * blockIdx.x / gridDim.x);
        uc.a1 = (int)((unsigned)NU0 * (blockIdx.x + 1) / gridDim.x);
        uc.u0 = ROW ? uc.a0 + tm.team : lv.tile(uc.a0 + tm.team);
        // row phase: which of the 16 sub-line elements t + 16 i sit in live column tiles on input
        // (what the previous column phase wrote; the rest is stale and stands for zeros)
        if constexpr (ROW) uc.lmask = live_mask16<P>(Fin, NX, tm.c, tm.l.t, cwc == 4 ? 2 : 3);
        uc.F = Fin;
    }
    const int a0 = uc.a0, a1 = uc.a1;
    const unsigned lmask = uc.lmask >> tm.l.h;           // bit 2 i: element 32 i + 16 h + t
    const int NU = ROW ? NY : (BATCH ? LV(Fin, NX, CWL).total() : 0);
    cf *ybuf = sm_y + (threadIdx.x / (32 * CW)) * (16 * 17 * CW) + tm.col;        // one region per (team, class)
    cf *xbuf = sm_y + tm.team * (TM::TEAM / 32) * (16 * 17) + tm.col;             // same memory, the team's part
    cf *pw = sm_pw + threadIdx.x;
    const bool want_I = d.kind == 1 && K.inten != nullptr;
    const bool accumulate = (K.flags & 1u) != 0;
    const int B = BATCH ? K.B : 1;
    const long long npx = (long long)NX * NY;
    const bool summed = BATCH && ROW && want_I && !(K.flags & 2u) && K.B > 1;
    float *acc = reinterpret_cast<float *>(sm_pw - Smem8<NX / kL, NY / kL>::kPw);   // = the H buffer (ROW: sm_pw is the screen buffer)
    if constexpr (BATCH && ROW) {
        // CTA-uniform branches, but only the working teams are here: hardware barrier 15 over them
        constexpr int NW = TM::NTEAM * TM::TEAM;
        if (d.kind == 1 && tag.src != d.src) {                 // not staged during the barrier
            asm volatile("bar.sync 15, %0;" ::"n"(NW) : "memory");
            for (int idx = threadIdx.x; idx < (a1 - a0) * NX; idx += NW) {
                const float a = fmaf(K.phase_b, K.noscreen ? 0.f : __ldcs(reinterpret_cast<const float *>(d.src) + (long long)a0 * NX + idx), d.pa);
                float s, c;
                screen_sincos(a, s, c);
                sm_pw[idx] = make_float2(c, s);
            }
            tag.src = d.src;
            asm volatile("bar.sync 15, %0;" ::"n"(NW) : "memory");
        }
        if (summed) {
            for (int idx = threadIdx.x; idx < (a1 - a0) * NX; idx += NW) acc[idx] = 0.f;
            asm volatile("bar.sync 15, %0;" ::"n"(NW) : "memory");
        }
    }
    const WarpSync wsync;
    // hardware barriers: 0 = CTA, 1 .. NTEAM = teams, above = (team, class) groups of a column tile
    const GroupSync<32 * CW> gsync{P == 1 ? 1 + tm.team : 1 + TM::NTEAM + (int)threadIdx.x / (32 * CW)};
    static_assert(ROW || (P == 1 ? TM::NTEAM : TM::NTEAM + kThreads8 / (32 * CW)) <= 15, "barrier ids");

    const int k0 = BATCH ? (ROW ? a0 * B : (int)(((long long)NU * B * blockIdx.x) / gridDim.x)) : a0;
    const int k1 = BATCH ? (ROW ? a1 * B : (int)(((long long)NU * B * (blockIdx.x + 1)) / gridDim.x)) : a1;
#pragma unroll 1
    for (int k = k0 + tm.team; k < k1; k += TM::NTEAM) {
        const int m = BATCH ? k / B : k, b = BATCH ? k - m * B : 0;
        const int u = ROW ? m : (!BATCH && k == k0 + tm.team ? uc.u0 : LV(Fin, NX, CWL).tile(m));
        if constexpr (BATCH && ROW) {
            pw = sm_pw + (m - a0) * NX;                         // the row's factors, indexed by pixel
        } else if (d.kind != 0 && (tag.src != d.src || tag.pix0 != u)) {
            fill_pw8<P, CW, ROW, NX>(d.kind, d.src, u, d.pa, K.phase_b, pw, K.noscreen != 0);
            tag.src = d.src; tag.pix0 = u;
        }
        cf *line = K.field + b * npx + (ROW ? (long long)u * NX : (long long)u * CW + tm.col);
        cf v[kSlots8];
        bool loaded = false;
        if constexpr (!ROW) {
            if (K.use_tma) {
                // One thread asks the TMA unit for the P y-classes of the tile ([256][CW] each, into the
                // team's part of the transpose region); the threads then read their points with LDS.
                cf *stage = sm_y + tm.team * (TM::TEAM / 32) * (16 * 17);
                unsigned long long *bar = sm_mbar + tm.team;
                if (threadIdx.x % TM::TEAM == 0) {
                    // the tiles were written by other CTAs through the generic proxy (st.global) and the landing
                    // zone by this CTA: order both before the async-proxy copy (full fence once per phase)
                    if (k == k0 + tm.team) asm volatile("fence.proxy.async;" ::: "memory");
                    else asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(bar, (unsigned)(P * kL * CW * sizeof(cf)));
#pragma unroll
                    for (int cc = 0; cc < P; ++cc) tma_load_4d(stage + cc * kL * CW, &K.tmap, u * CW, cc, 0, b, bar);
                }
                if (!mbar_wait(bar, uc.tma_parity)) {       // the copy never arrived: flag it and leave the phase; the grid
                    atomicExch(K.status, 2);                // barrier's watchdog sees the flag and ends the kernel
                    return;
                }
                uc.tma_parity ^= 1u;
#pragma unroll
                for (int i = 0; i < kSlots8; ++i) v[i] = stage[(tm.c * kL + 32 * i + 16 * tm.l.h + tm.l.t) * CW + tm.col];
                tm.sync();                              // staged tile read: the region goes back to the transposes
                loaded = true;
            }
        }
        if (d.first) {
            if (!loaded) {
                const cf *src = line + tm.c * CSr + (16 * tm.l.h + tm.l.t) * ISr;
#pragma unroll
                for (int i = 0; i < kSlots8; ++i) {
                    v[i] = make_float2(0.f, 0.f);
                    if (!ROW || ((lmask >> (2 * i)) & 1u)) v[i] = ld_cg(src + 32 * ISr * i);
                }
            }
            if constexpr (ROW) subline8_dit<S1, CW>(v, sm_tw, ybuf, tm.l, wsync);
            else subline8_dit<S1, CW>(v, sm_tw, ybuf, tm.l, gsync);
            // v[j] = F_c[t + 16 (4 h + j)], v[4 + j] = F_c[t + 16 (4 h + 8 + j)]
            if constexpr (P > 1) {
                // exchange: (class, 8 indices) -> (group, 8/P indices of every class)
                tm.sync();                                  // the team's transposes have been read
                cf *xw = xbuf + (tm.c * kL + tm.l.t + 64 * tm.l.h) * CW;
#pragma unroll
                for (int jj = 0; jj < 8; ++jj) xw[(16 * (jj & 3) + 128 * (jj >> 2)) * CW] = v[jj];
                tm.sync();
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int cc = 0; cc < P; ++cc) v[jp * P + cc] = xbuf[(cc * kL + tm.q(jp)) * CW];
#pragma unroll
                for (int jp = 0; jp < JP; ++jp) {
#pragma unroll
                    for (int cc = 1; cc < P; ++cc)
                        v[jp * P + cc] = cmul_s<S1>(v[jp * P + cc], sm_twc[(cc - 1) * kL + tm.q(jp)]);
                    class_dft_any<P, S1>(&v[jp * P]);
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < kSlots8; ++i) v[i] = ld_cg(line + (long long)tm.pix(i) * NS);
        }
        // P > 1: v[jp*P + m] is element n = q(jp) + 256 m of the line, in its natural (x- or ky-) order;
        // P = 1: v[jj] is element n = t + 16 (4 h + (jj & 3) + 8 (jj >> 2))
        auto pix = [&](int slot) { return tm.pix(slot); };
        if (d.kind == 1) {
            // u = value * screen (bb.h step 4), intensity (step 5)
            if constexpr (BATCH) {
#pragma unroll
                for (int i = 0; i < kSlots8; ++i) v[i] = cmul(v[i], pw[pix(i)]);
            } else {
#pragma unroll
                for (int i = 0; i < kSlots8; ++i) v[i] = cmul(v[i], pw[i * kThreads8]);
            }
            if (summed) {
                float *ar = acc + (m - a0) * NX;
#pragma unroll
                for (int i = 0; i < kSlots8; ++i) atomicAdd(ar + pix(i), fmaf(v[i].x, v[i].x, v[i].y * v[i].y));
            } else if (want_I) {
                float *ip = K.inten + d.slice + (long long)u * NX
                            + ((K.flags & 2u) ? (long long)b * K.inten_bstride : 0);
#pragma unroll
                for (int i = 0; i < kSlots8; ++i) {
                    float I = fmaf(v[i].x, v[i].x, v[i].y * v[i].y);
                    float *a = ip + pix(i);
                    if (accumulate) I += *a;
                    __stcg(a, I);
                }
            }
        } else if (d.kind == 2) {
            // U * H (bb.h step 2)
#pragma unroll
            for (int i = 0; i < kSlots8; ++i) v[i] = cmul(v[i], pw[i * kThreads8]);
        }
        if (scale != 1.f) {
#pragma unroll
            for (int i = 0; i < kSlots8; ++i) v[i] = make_float2(v[i].x * scale, v[i].y * scale);
        }
        if (d.second) {
            if constexpr (P > 1) {
#pragma unroll
                for (int jp = 0; jp < JP; ++jp) {
                    class_dft_any<P, S2>(&v[jp * P]);
#pragma unroll
                    for (int cc = 1; cc < P; ++cc)
                        v[jp * P + cc] = cmul_s<S2>(v[jp * P + cc], sm_twc[(cc - 1) * kL + tm.q(jp)]);
                }
                // (no barrier here: a thread writes exactly the slots it read in the first exchange, and nobody
                // else touches them in between)
#pragma unroll
                for (int jp = 0; jp < JP; ++jp)
#pragma unroll
                    for (int cc = 0; cc < P; ++cc) xbuf[(cc * kL + tm.q(jp)) * CW] = v[jp * P + cc];
                tm.sync();
                const cf *xr = xbuf + (tm.c * kL + tm.l.t + 64 * tm.l.h) * CW;
#pragma unroll
                for (int jj = 0; jj < 8; ++jj) v[jj] = xr[(16 * (jj & 3) + 128 * (jj >> 2)) * CW];
            }
            tm.sync();                                      // region free again for the transposes
            if constexpr (ROW) subline8_dif<S2, CW>(v, sm_tw, ybuf, tm.l, wsync);
            else subline8_dif<S2, CW>(v, sm_tw, ybuf, tm.l, gsync);
            cf *dst = line + tm.c * CSr + (16 * tm.l.h + tm.l.t) * ISr;
#pragma unroll
            for (int i = 0; i < kSlots8; ++i) st_cg(dst + 32 * ISr * i, v[i]);
        } else {
#pragma unroll
            for (int i = 0; i < kSlots8; ++i) st_cg(line + (long long)pix(i) * NS, v[i]);
        }
        tm.sync();                                          // buffers free for the team's next unit
    }
    if constexpr (BATCH && ROW) {
        if (summed) {
            // I[j] (+)= sum over the fields (bb.h step 5): the CTA's rows are contiguous in the slice
            constexpr int NW = TM::NTEAM * TM::TEAM;
            asm volatile("bar.sync 15, %0;" ::"n"(NW) : "memory");
            float *ip = K.inten + d.slice + (long long)a0 * NX;
            for (int idx = threadIdx.x; idx < (a1 - a0) * NX; idx += NW) {
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
__device__ __forceinline__ void prefill_phase8(const KParams &K, const Phase16 &d, cf *sm_pw, PwTag &tag, int Fin) {
    typedef Team8<P, CW> TM;
    if (d.kind == 0) return;
    if constexpr (BATCH && ROW) {
        if (tag.src != d.src) {
            stage_rows_screen8<NX, NY>(K, d, sm_pw);
            tag.src = d.src;
        }
        return;
    }
    const TM tm;
    if (tm.team >= TM::NTEAM) return;
    const LiveCols<ROW ? 1 : (NX / kL)> lv(Fin, NX, CW == 8 ? 3 : (CW == 4 ? 2 : 0));
    const int NU = ROW ? NY : lv.total();
    const int a0 = (int)((unsigned)NU * blockIdx.x / gridDim.x);
    const int a1 = (int)((unsigned)NU * (blockIdx.x + 1) / gridDim.x);
    const int B = BATCH ? K.B : 1;
    const int k0 = BATCH ? (int)(((long long)NU * B * blockIdx.x) / gridDim.x) : a0;
    const int k1 = BATCH ? (int)(((long long)NU * B * (blockIdx.x + 1)) / gridDim.x) : a1;
    const int k = k0 + tm.team;
    if (k >= k1) return;
    const int m = BATCH ? k / B : k;
    const int u = ROW ? m : lv.tile(m);
    if (tag.src == d.src && tag.pix0 == u) return;
    fill_pw8<P, CW, ROW, NX>(d.kind, d.src, u, d.pa, K.phase_b, sm_pw + threadIdx.x, K.noscreen != 0);
    tag.src = d.src; tag.pix0 = u;
}

// CWC: columns per column tile (8, or 4 when few columns are live); BATCH: several fields (KParams::B)
template <int PX, int PY, int CWC, bool BATCH>
__global__ void __launch_bounds__(kThreads8, 1) bpm8_kernel(const __grid_constant__ KParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    using L = Smem8<PX, PY>;
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

    for (int i = threadIdx.x; i < L::kTw; i += kThreads8) sm_tw[i] = P.tw256[i];
    for (int i = threadIdx.x; i < (PX - 1) * kL; i += kThreads8) sm_twcx[i] = P.twcx[i];
    for (int i = threadIdx.x; i < (PY - 1) * kL; i += kThreads8) sm_twcy[i] = P.twcy[i];
    __syncthreads();

    PwTag tagH = {nullptr, -1}, tagS = {nullptr, -1};
    UnitCache ucR, ucC;
    auto live_in = [&](int p) {
        if (P.mode == 1) return NX / 2;                       // transform programs: every column is live
        const bool row = (p & 1) == 0;
        return row ? ((p >> 1) >= 1 ? P.fmax[col_step(P, (p >> 1) - 1)] : NX / 2) : P.fmax[col_step(P, p >> 1)];
    };
    // mode 1 (bb_fft2, bb_multiplex_*): phase p is the line transform KParams::prog[p] describes
    auto decode = [&](int p) {
        if (P.mode == 0) return decode_phase16(P, p);
        Phase16 d;
        d.kind = 0; d.src = nullptr; d.pa = 0.f; d.slice = 0;
        d.is_row = P.prog[p].is_row != 0;
        d.first = d.is_row ? P.prog[p].inv != 0 : P.prog[p].fwd != 0;
        d.second = d.is_row ? P.prog[p].fwd != 0 : P.prog[p].inv != 0;
        return d;
    };
    int Fa_next = live_in(P.p0);
    Phase16 d_next = decode(P.p0);
    const int r0 = (int)((unsigned)NY * blockIdx.x / gridDim.x);          // rows of this CTA (row phases)
    const int r1 = (int)((unsigned)NY * (blockIdx.x + 1) / gridDim.x);
    unsigned nbar = 0;
    long long *tr = P.trace ? P.trace + ((long long)(P.p0 - P.trace_p0) * gridDim.x + blockIdx.x) * 6 : nullptr;
    const bool tracer = tr != nullptr && threadIdx.x == 0;
#pragma unroll 1
    for (int p = P.p0; p < P.p1; ++p) {
        const Phase16 d = d_next;              // decoded while the previous barrier was pending
        if (tracer) tr[0] = clock64();
        if (d.is_row && p + 2 < P.p1 && P.mode == 0) {
            // the dn rows this CTA turns into screen factors at the end of this phase (for the row
            // phase after next): start them on their way from HBM to L2 now, one bulk prefetch per row
            const int jn = row_step(P, (p >> 1) + 1);
            if ((int)threadIdx.x < r1 - r0 && jn >= 0 && !P.noscreen) {
                const float *row = P.dn + (long long)(jn - P.j_base) * ((long long)NX * NY)
                                   + (long long)(r0 + threadIdx.x) * NX;
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(row), "r"(NX * 4) : "memory");
            }
        }
        const int Fa = Fa_next;
        const float scale = P.mode == 1 ? P.prog[p].scale : 1.f;
        if (d.is_row) run_phase8<PX, 1, true, NX, NY, BATCH>(P, d, sm_tw, sm_twcx, sm_y, sm_pwS, tagS, ucR, Fa, CWC, nullptr, scale);
        else run_phase8<PY, CWC, false, NX, NY, BATCH>(P, d, sm_tw, sm_twcy, sm_y, sm_pwH, tagH, ucC, Fa, CWC, sm_mbar, scale);
        if (tracer) tr[1] = clock64();
        if (BATCH && d.is_row && d.kind == 1 && P.inten != nullptr && !(P.flags & 2u) && P.B > 1)
            tagH.src = nullptr;                // the intensity sums used the propagator buffer
        if (p + 1 < P.p1) {
            ++nbar;
            grid_arrive(P.bar);
            if (tracer) tr[2] = clock64();
            Fa_next = live_in(p + 1);
            d_next = decode(p + 1);   // its global loads (table pointer, phase offset) overlap the barrier
            if (P.mode == 1) {
            } else if (d.is_row) {
                const int Fn = Fa_next;
                prefill_phase8<PY, CWC, false, NX, NY, BATCH>(P, d_next, sm_pwH, tagH, Fn);
                if (p + 2 < P.p1) prefill_phase8<PX, 1, true, NX, NY, BATCH>(P, decode_phase16(P, p + 2), sm_pwS, tagS, 0);
            } else {
                prefill_phase8<PX, 1, true, NX, NY, BATCH>(P, d_next, sm_pwS, tagS, 0);
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
