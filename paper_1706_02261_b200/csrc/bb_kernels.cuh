// bb_kernels.cuh -- the BPM step kernel (row phase, column phase, persistent driver).
//
// One BPM step (bb.h; BASELINE.json:north_star sentence 2) is split into two phases that
// each keep a whole line in registers, so the field crosses L2 twice per step:
//   column phase  C_j :  FFT_y  ->  x H_j  ->  IFFT_y               (k-space pointwise op)
//   row phase     R_j :  IFFT_x ->  x exp(i phi(dn[j-1])) -> |u|^2 -> FFT_x   (x-space op)
// The sequence for Nz steps is  R_0(FFT_x only), C_0, R_1, C_1, ..., C_{Nz-1}, R_Nz(no FFT_x).
// Phases are separated by a grid-wide barrier inside ONE persistent cooperative kernel
// (or by kernel boundaries in the per-phase diagnostic mode).  See DESIGN.md "Kernels".
//
// Code size is a first-order concern: a phase runs every instruction once, so the kernel
// is instruction-fetch bound unless its hot path fits the 32 KB instruction cache
// (profiles/r01_a_*).  Hence ONE copy of the line FFT serves rows and columns (run-time
// thread mapping) and both directions (inverse = conj . forward . conj), the two
// transforms of a phase are a rolled loop, and the pointwise factors of a phase (phase
// screen or propagator values) are staged in a thread-private shared-memory column
// -- filled while the grid barrier before the phase is pending.
#pragma once
#include <cuda.h>
#include "bb_fft.cuh"

namespace bb {

constexpr int kThreads = 256;          // threads per CTA
constexpr int kWarps = kThreads / 32;
constexpr unsigned kSpinLimit = 1u << 24;   // grid-barrier watchdog (polls), ~ seconds

struct PhaseProg {   // generic (non-BPM) phase: used by bb_fft2 and bb_multiplex_psf
    int is_row;
    int inv;         // inverse line FFT first
    int fwd;         // forward line FFT last
    float scale;     // multiply the result (1 = none)
};

struct KParams {
    cf *field;                 // [B][Ny][Nx]
    const float *dn;           // slice j_base of the dn volume
    float *inten;              // slice j_base of the intensity volume, or nullptr
    long long inten_bstride;   // elements between fields of a per-field intensity volume
    const cf *const *htab;     // device [Nz_total]: propagator table of step j
    const float *phase_a;      // device [Nz_total]: k0 dz (n0 - n_ref[j])
    float phase_b;             // k0 dz
    int Nx, Ny, B;
    int BW;                    // warps of a CTA that split the batch in the row phase (power of 2 <= 8)
    int Nz_total;              // row phase r does the forward FFT_x iff r < Nz_total
    int j_base;
    int p0, p1;                // phases [p0, p1) run in this launch
    int mode;                  // 0: BPM phase sequence, 1: prog[]
    PhaseProg prog[2];
    const cf *twx, *twy;       // global twiddle tables [32][T]
    const cf *tw256, *twcx, *twcy;   // 16-point-thread kernel: sub-line twiddles [16][16], class twiddles [P-1][256]
    unsigned *bar;             // grid barrier counter (zeroed before the launch)
    int *status;               // device flag: != 0 -> watchdog tripped
    unsigned flags;            // BB_ACCUMULATE = 1, BB_INTENSITY_PER_FIELD = 2
    int backward;              // BB_BACKWARD: steps run from Nz_total - 1 down to 0 (tables and phase offsets are
                               // conjugated by the host: dz -> -dz)
    int noscreen;              // BB_HOMOGENEOUS: no phase screen (dn is not read), intensity only
    int xnat;                  // 8-point-thread kernel, transform programs: rows are in natural kx order in memory
    const int *fmax;           // device [Nz_total]: largest |kx DFT bin| the propagator of step j lets through (conservative)
    int cw4;                   // 16-point-thread kernel: column tiles of 4 columns instead of 8
    int use_tma;               // 16-point-thread kernel: column tiles are fetched by TMA through `tmap`
    long long *trace;          // bb_probe_trace: [phase - trace_p0][CTA][6] time stamps, or nullptr
    int trace_p0;
    // fields as a 4-D tensor (column, y mod PY, y div PY, field) of 8-byte elements, box = (CW, 1, 256, 1):
    // one TMA request brings one y-class of a column tile, [256][CW] row-major, into shared memory
    alignas(64) CUtensorMap tmap;
};

// Which z-step a phase belongs to.  Forward: row phase r applies the screen of step r - 1 (r >= 1), column
// phase r the propagator of step r.  Backward (time reversal, Fig. 2c): a step is "x conj screen,
// FFT2, x conj H, IFFT2", so row phase r applies the screen of step Nz - 1 - r (r < Nz) BEFORE the
// transform pair that column phase r completes with the table of the same step.
__device__ __forceinline__ int row_step(const KParams &P, int r) {
    return P.backward ? (r < P.Nz_total ? P.Nz_total - 1 - r : -1) : r - 1;
}
__device__ __forceinline__ int col_step(const KParams &P, int r) { return P.backward ? P.Nz_total - 1 - r : r; }

__device__ __forceinline__ cf ld_cg(const cf *p) { return __ldcg(p); }
__device__ __forceinline__ void st_cg(cf *p, cf v) { __stcg(p, v); }

// What one phase does, decoded from the phase index.
struct PhaseDesc {
    bool is_row;
    bool first;        // transform 0 of the phase runs  (row: IFFT_x, column: FFT_y)
    bool second;       // transform 1 of the phase runs  (row: FFT_x,  column: IFFT_y)
    int kind;          // pointwise factor between the two: 0 none, 1 phase screen of dn slice, 2 table,
                       // 3 no factor but the intensity is recorded (homogeneous medium)
    float scale;
    const void *src;   // kind 1: dn slice (float), kind 2: propagator table (cf)
    float pa;          // kind 1: phase offset k0 dz (n0 - n_ref[j])
    long long slice;   // kind 1: element offset of the intensity slice
    bool in_cj;        // the field in memory is the conjugate of the value (see decode_phase)
    bool out_cj;       // leave the conjugate in memory
};

__device__ __forceinline__ PhaseDesc decode_phase(const KParams &P, int p) {
    PhaseDesc d;
    d.kind = 0; d.scale = 1.f; d.src = nullptr; d.pa = 0.f; d.slice = 0;
    d.in_cj = d.out_cj = false;
    if (P.mode == 0) {
        // Between a column phase and the row phase after it the field is held CONJUGATED in
        // memory: the inverse transforms are conj . forward . conj, so IFFT_y leaves the
        // conjugate in registers and IFFT_x wants it as input -- no sign flips on the hot path.
        d.is_row = (p & 1) == 0;
        d.in_cj = d.is_row && p >= 2;
        d.out_cj = !d.is_row;
        if (d.is_row) {
            d.first = p >= 2;
            d.second = (p >> 1) < P.Nz_total;
            const int j = row_step(P, p >> 1);
            if (j >= 0) {
                d.slice = (long long)(j - P.j_base) * ((long long)P.Nx * P.Ny);
                if (P.noscreen) {
                    d.kind = 3;
                } else {
                    d.kind = 1;
                    d.src = P.dn + d.slice;
                    d.pa = P.phase_a[j];
                }
            }
        } else {
            d.first = true; d.second = true;
            d.kind = 2;
            d.src = P.htab[col_step(P, p >> 1)];
        }
    } else {
        const PhaseProg &g = P.prog[p];
        d.is_row = g.is_row != 0;
        d.first = d.is_row ? g.inv != 0 : g.fwd != 0;
        d.second = d.is_row ? g.fwd != 0 : g.inv != 0;
        d.scale = g.scale;
    }
    return d;
}

// ----------------------------------------------------------------------------------------
// Thread mapping of a phase.  Row phase: a warp owns G = 32/T consecutive rows ("row
// group") of one field, lane = g*T + t; the warps of a CTA are split RW x BW (RW row groups
// at a time, BW warps striding over the batch).  Column phase: a tile is CW adjacent
// columns x all rows of one field, handled by CW*T threads (thread r: column c = r % CW,
// FFT lane t = r / CW), so every global access of a warp is whole 8*CW-byte row segments and
// no transposed copy of the field ever exists.  Either way thread (line, t) holds elements
// x[t + T i], i < 32, at  pix0 + i*estride  of its field.
// ----------------------------------------------------------------------------------------
struct Unit {
    bool valid;
    bool first_of_group, last_of_group;   // row phase: first / last batch iteration of a row group
    int b;
    long long pix0;
};

template <int T, int CW>
struct Mapping {
    static constexpr int G = 32 / T;
    static constexpr int NT = CW * T;            // threads per column tile
    static constexpr int NS = kThreads / NT;     // column tiles in flight per CTA
    bool is_row;
    int t, n_iter, B, Nx;
    long long estride;
    cf *ybuf;
    int a0, a1, sub, nb, bw, BW, RW, gc;

    __device__ __forceinline__ Mapping(const KParams &P, bool is_row_, cf *sm_y) {
        const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
        is_row = is_row_; B = P.B; Nx = P.Nx;
        if (is_row) {
            gc = lane / T; t = lane % T;
            BW = P.BW; RW = kWarps / BW;
            sub = warp / BW; bw = warp % BW;
            const int NRG = P.Ny / G;
            a0 = (int)(((long long)NRG * blockIdx.x) / gridDim.x);
            a1 = (int)(((long long)NRG * (blockIdx.x + 1)) / gridDim.x);
            nb = (B + BW - 1) / BW;
            n_iter = ((a1 - a0 + RW - 1) / RW) * nb;
            estride = T;
            ybuf = sm_y + warp * RowGeom<T>::WARP + gc * RowGeom<T>::RS;
        } else {
            const int r = tid % NT;
            sub = tid / NT; gc = r % CW; t = r / CW;
            BW = 1; RW = 1; bw = 0; nb = 1;
            const int NU = (P.Nx / CW) * B;
            a0 = (int)(((long long)NU * blockIdx.x) / gridDim.x);
            a1 = (int)(((long long)NU * (blockIdx.x + 1)) / gridDim.x);
            n_iter = (a1 - a0 + NS - 1) / NS;
            estride = (long long)T * P.Nx;
            ybuf = sm_y + sub * ColGeom<T, CW>::TILE + gc * ColGeom<T, CW>::RS;
        }
    }
    __device__ __forceinline__ Unit unit(int k) const {
        Unit u;
        if (is_row) {
            const int it = k / nb, bi = k - it * nb;
            const int rg = a0 + it * RW + sub;
            u.b = bw + bi * BW;
            u.valid = rg < a1 && u.b < B;
            u.first_of_group = bi == 0;
            u.last_of_group = bi == nb - 1;
            u.pix0 = (long long)(rg * G + gc) * Nx + t;
        } else {
            const int uu = a0 + k * NS + sub;
            const int ct = uu / B;
            u.b = uu - ct * B;
            u.valid = uu < a1;
            u.first_of_group = u.last_of_group = false;
            u.pix0 = (long long)t * Nx + (long long)ct * CW + gc;
        }
        return u;
    }
};

// Which pointwise factors the thread's shared-memory column currently holds.
struct PwTag { const void *src; long long pix0; };

// Fill the thread-private column pw[i * kThreads], i < 32, with the pointwise factors of the
// thread's elements:  exp(i (pb dn + pa))  at pix0 + T i of a dn slice (row mapping; bb.h step 4),
// or the table values H at pix0 + T NX i (column mapping; bb.h step 2).  A real function (one
// copy, two call sites): it runs off the critical path, while a grid barrier is pending.
template <int T, int NX>
__device__ __noinline__ void fill_pw(int kind, const void *src, long long pix0, float pa, float pb, cf *pw) {
    if (kind == 1) {
        const float *dnp = reinterpret_cast<const float *>(src) + pix0;
        float x[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) x[i] = __ldcs(dnp + T * i);
#pragma unroll
        for (int i = 0; i < 32; ++i) pw[i * kThreads].x = x[i];
#pragma unroll 2
        for (int i = 0; i < 32; ++i) {
            float s, c;
            sincosf(fmaf(pb, pw[i * kThreads].x, pa), &s, &c);
            pw[i * kThreads] = make_float2(c, s);
        }
    } else {
        const cf *hp = reinterpret_cast<const cf *>(src) + pix0;
        cf h[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) h[i] = __ldg(hp + (long long)(T * NX) * i);
#pragma unroll
        for (int i = 0; i < 32; ++i) pw[i * kThreads] = h[i];
    }
}

// ----------------------------------------------------------------------------------------
// One phase over the lines this CTA owns.  MODE 0: row or column mapping chosen at run time
// (square grids: one copy of everything), 1: row mapping only, 2: column mapping only.
// Loads, stores and the pointwise step are written per mapping (compile-time strides, so the
// addresses are immediates); the line FFT between them is shared.
// ----------------------------------------------------------------------------------------
template <int T, int CW, int NX, int MODE>
__device__ __forceinline__ void run_phase(const KParams &P, const PhaseDesc &d, const cf *sm_tw, cf *sm_y,
                                          cf *sm_pw, float *sm_acc, PwTag &tag) {
    static_assert(RowGeom<T>::S == T + 1 && ColGeom<T, CW>::S == T + 1, "one k1-row stride for both mappings");
    constexpr long long CS = (long long)T * NX;               // element stride of the column mapping
    const bool is_row = MODE == 0 ? d.is_row : MODE == 1;
    const Mapping<T, CW> m(P, is_row, sm_y);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long npx = (long long)P.Nx * P.Ny;
    const bool want_I = (d.kind == 1 || d.kind == 3) && P.inten != nullptr;
    const bool per_field = (P.flags & 2u) != 0;
    const bool accumulate = (P.flags & 1u) != 0;
    const bool summed = want_I && !per_field && P.B > 1;      // CTA-uniform
    const bool cta_has_work = m.a1 > m.a0;
    cf *pw = sm_pw + tid;
    float *acc = sm_acc + warp * 1024;
    const SyncSel sync{is_row};

#pragma unroll 1
    for (int k = 0; k < m.n_iter; ++k) {
        const Unit u = m.unit(k);
        if (summed && u.first_of_group) {
#pragma unroll
            for (int i = 0; i < 32; ++i) acc[i * 32 + lane] = 0.f;
        }
        // the column transposes synchronise the whole CTA, so there every thread walks through
        if (is_row ? u.valid : cta_has_work) {
            if (u.valid && (d.kind == 1 || d.kind == 2) && (tag.src != d.src || tag.pix0 != u.pix0)) {
                fill_pw<T, NX>(d.kind, d.src, u.pix0, d.pa, P.phase_b, pw);
                tag.src = d.src; tag.pix0 = u.pix0;
            }
            cf *line = P.field + (long long)u.b * npx + u.pix0;
            cf v[32];
            if (is_row) {
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] = ld_cg(line + T * i);
            } else {
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] = u.valid ? ld_cg(line + CS * i) : make_float2(0.f, 0.f);
            }
            bool cj = d.in_cj;                                 // v holds the conjugate of the value
#pragma unroll 1
            for (int pass = 0; pass < 2; ++pass) {
                if (pass == 0 ? d.first : d.second) {
                    const bool inverse = is_row ? pass == 0 : pass == 1;
                    if (inverse != cj) {
#pragma unroll
                        for (int i = 0; i < 32; ++i) v[i].y = -v[i].y;
                    }
                    line_fft_fwd<T, T + 1>(v, sm_tw, m.ybuf, m.t, sync);
                    cj = inverse;
                }
                if (pass == 0 && d.kind != 0) {
                    if (is_row) {
                        // u = value * screen, from the conjugate the inverse transform leaves (bb.h step 4)
                        if (d.kind == 3 ? cj : !cj) {
#pragma unroll
                            for (int i = 0; i < 32; ++i) v[i].y = -v[i].y;
                        }
                        cj = false;
                        if (d.kind != 3) {
#pragma unroll
                            for (int i = 0; i < 32; ++i) v[i] = cmulc(pw[i * kThreads], v[i]);
                        }
                        if (want_I) {
                            if (summed) {
#pragma unroll
                                for (int i = 0; i < 32; ++i)
                                    acc[i * 32 + lane] += fmaf(v[i].x, v[i].x, v[i].y * v[i].y);
                            } else {
                                float *ip = P.inten + d.slice + u.pix0
                                            + (per_field ? (long long)u.b * P.inten_bstride : 0);
                                if (accumulate) {
#pragma unroll
                                    for (int i = 0; i < 32; ++i)
                                        __stcs(ip + T * i, fmaf(v[i].x, v[i].x, v[i].y * v[i].y) + ip[T * i]);
                                } else {
#pragma unroll
                                    for (int i = 0; i < 32; ++i)
                                        __stcs(ip + T * i, fmaf(v[i].x, v[i].x, v[i].y * v[i].y));
                                }
                            }
                        }
                    } else {
                        // U * H, left conjugated for the inverse transform that follows (bb.h step 2)
                        if (cj) {
#pragma unroll
                            for (int i = 0; i < 32; ++i) v[i].y = -v[i].y;
                        }
                        cj = true;
#pragma unroll
                        for (int i = 0; i < 32; ++i) {
                            const cf h = pw[i * kThreads];
                            v[i] = make_float2(fmaf(v[i].x, h.x, -(v[i].y * h.y)), fmaf(-v[i].x, h.y, -(v[i].y * h.x)));
                        }
                    }
                }
            }
            if (cj != d.out_cj || d.scale != 1.f) {
                const float sx = d.scale, sy = cj != d.out_cj ? -d.scale : d.scale;
#pragma unroll
                for (int i = 0; i < 32; ++i) { v[i].x *= sx; v[i].y *= sy; }
            }
            if (is_row) {
#pragma unroll
                for (int i = 0; i < 32; ++i) st_cg(line + T * i, v[i]);
            } else if (u.valid) {
#pragma unroll
                for (int i = 0; i < 32; ++i) st_cg(line + CS * i, v[i]);
            }
        }
        if (summed && u.last_of_group) {
            __syncthreads();
            if (m.bw == 0 && u.valid) {
                float *ip = P.inten + d.slice + u.pix0;
#pragma unroll 4
                for (int i = 0; i < 32; ++i) {
                    float I = 0.f;
#pragma unroll 1
                    for (int q = 0; q < m.BW; ++q) I += acc[q * 1024 + i * 32 + lane];
                    if (accumulate) I += ip[T * i];
                    __stcs(ip + T * i, I);
                }
            }
            __syncthreads();
        }
    }
}

// While the grid barrier before phase `d` is pending: stage the pointwise factors of the
// thread's first unit of that phase (they do not depend on the field).
template <int T, int CW, int NX, int MODE>
__device__ __forceinline__ void prefill_phase(const KParams &P, const PhaseDesc &d, cf *sm_y, cf *sm_pw, PwTag &tag) {
    if (d.kind != 1 && d.kind != 2) return;
    const Mapping<T, CW> m(P, MODE == 0 ? d.is_row : MODE == 1, sm_y);
    if (m.n_iter < 1) return;
    const Unit u = m.unit(0);
    if (!u.valid || (tag.src == d.src && tag.pix0 == u.pix0)) return;
    fill_pw<T, NX>(d.kind, d.src, u.pix0, d.pa, P.phase_b, sm_pw + threadIdx.x);
    tag.src = d.src; tag.pix0 = u.pix0;
}

// ----------------------------------------------------------------------------------------
// Grid barrier, split in two so that independent work runs while it is pending: every CTA
// arrives with a release (all its stores ordered before by the block barrier), and polls
// with an acquire.  `target` = arrivals expected since the counter was zeroed.  A watchdog
// turns a would-be hang into an error flag.
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ void grid_arrive(unsigned *bar) {
    __syncthreads();
    if (threadIdx.x == 0)
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
}
// (measured alternatives, both slower on an empty phase loop, 1.55 us per barrier as written: polling with
// relaxed loads plus one acquire fence 1.75 us; every thread fencing its own stores and a relaxed add 1.87 us)
__device__ __forceinline__ bool grid_wait(unsigned *bar, unsigned target, int *status, int *sm_abort) {
    if (threadIdx.x == 0) {
        unsigned spins = 0;
        int abort_ = 0;
        for (;;) {
            unsigned v;
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
            if (v >= target) break;
            if (((++spins) & 1023u) == 0) {
                if (*(volatile int *)status != 0) { abort_ = 1; break; }
                if (spins >= kSpinLimit) { atomicExch(status, 1); abort_ = 1; break; }
            }
        }
        *sm_abort = abort_;
    }
    __syncthreads();
    return *sm_abort != 0;
}

template <int TX, int TY, int CW>
struct SmemLayout {
    static constexpr int kTw = 32 * TX + 32 * TY;                                   // cf
    static constexpr int kRowY = kWarps * RowGeom<TX>::WARP;
    static constexpr int kColY = (kThreads / (CW * TY)) * ColGeom<TY, CW>::TILE;
    static constexpr int kY = kRowY > kColY ? kRowY : kColY;
    static constexpr int kPw = 32 * kThreads;
    static constexpr int kAcc = kWarps * 1024;                                      // floats
    static constexpr size_t bytes = (size_t)(kTw + kY + kPw) * sizeof(cf) + (size_t)kAcc * sizeof(float) + 16;
};

template <int TX, int TY, int CW>
__global__ void __launch_bounds__(kThreads, 1) bpm_kernel(const KParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    using L = SmemLayout<TX, TY, CW>;
    cf *sm_twx = reinterpret_cast<cf *>(smem_raw);
    cf *sm_twy = sm_twx + 32 * TX;
    cf *sm_y = sm_twy + 32 * TY;
    cf *sm_pw = sm_y + L::kY;
    float *sm_acc = reinterpret_cast<float *>(sm_pw + L::kPw);
    int *sm_abort = reinterpret_cast<int *>(sm_acc + L::kAcc);

    for (int i = threadIdx.x; i < 32 * TX; i += kThreads) sm_twx[i] = P.twx[i];
    for (int i = threadIdx.x; i < 32 * TY; i += kThreads) sm_twy[i] = P.twy[i];
    __syncthreads();

    PwTag tag = {nullptr, -1};
    unsigned nbar = 0;
#pragma unroll 1
    for (int p = P.p0; p < P.p1; ++p) {
        const PhaseDesc d = decode_phase(P, p);
        if constexpr (TX == TY) {
            run_phase<TX, CW, 32 * TX, 0>(P, d, sm_twx, sm_y, sm_pw, sm_acc, tag);
        } else {
            if (d.is_row) run_phase<TX, CW, 32 * TX, 1>(P, d, sm_twx, sm_y, sm_pw, sm_acc, tag);
            else run_phase<TY, CW, 32 * TX, 2>(P, d, sm_twy, sm_y, sm_pw, sm_acc, tag);
        }
        if (p + 1 < P.p1) {
            ++nbar;
            grid_arrive(P.bar);
            const PhaseDesc dn = decode_phase(P, p + 1);
            if constexpr (TX == TY) {
                prefill_phase<TX, CW, 32 * TX, 0>(P, dn, sm_y, sm_pw, tag);
            } else {
                if (dn.is_row) prefill_phase<TX, CW, 32 * TX, 1>(P, dn, sm_y, sm_pw, tag);
                else prefill_phase<TY, CW, 32 * TX, 2>(P, dn, sm_y, sm_pw, tag);
            }
            if (grid_wait(P.bar, nbar * gridDim.x, P.status, sm_abort)) return;
        }
    }
}

}  // namespace bb
