// bb_kernels.cuh -- the BPM step kernels (row phase, column phase, persistent driver).
//
// One BPM step (bb.h; BASELINE.json:north_star sentence 2) is split into two phases that
// each keep a whole line in registers, so the field crosses L2 twice per step:
//   column phase  C_j :  FFT_y  ->  x H_j  ->  IFFT_y               (k-space pointwise op)
//   row phase     R_j :  IFFT_x ->  x exp(i phi(dn[j-1])) -> |u|^2 -> FFT_x   (x-space op)
// The sequence for Nz steps is  R_0(FFT_x only), C_0, R_1, C_1, ..., C_{Nz-1}, R_Nz(no FFT_x).
// Phases are separated by a grid-wide barrier inside ONE persistent cooperative kernel
// (or by kernel boundaries in the per-phase diagnostic mode).  See DESIGN.md "Kernels".
#pragma once
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
    unsigned *bar;             // grid barrier counter (zeroed before the launch)
    int *status;               // device flag: != 0 -> watchdog tripped
    unsigned flags;            // BB_ACCUMULATE = 1, BB_INTENSITY_PER_FIELD = 2
};

__device__ __forceinline__ cf ld_cg(const cf *p) { return __ldcg(p); }
__device__ __forceinline__ void st_cg(cf *p, cf v) { __stcg(p, v); }

// ----------------------------------------------------------------------------------------
// Grid barrier: every CTA arrives with a release (fence + atomic add) and polls with an
// acquire.  `target` = arrivals expected since the counter was zeroed.  A watchdog turns a
// would-be hang into an error flag.
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ bool grid_barrier(unsigned *bar, unsigned target, int *status, int *sm_abort) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
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
        __threadfence();
        *sm_abort = abort_;
    }
    __syncthreads();
    return *sm_abort != 0;
}

// ----------------------------------------------------------------------------------------
// Row phase.  A warp owns G = 32/TX consecutive rows ("row group") of one field; the warps
// of a CTA are split RW x BW: RW row groups at a time, BW warps striding over the batch.
// ----------------------------------------------------------------------------------------
template <int TX>
__device__ __forceinline__ void row_phase(const KParams &P, bool inv, bool screen, bool fwd, float scale,
                                          int j, const cf *sm_tw, cf *sm_y, float *sm_acc) {
    constexpr int G = 32 / TX;
    using RG = RowGeom<TX>;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / TX, t = lane % TX;
    const int BW = P.BW, RW = kWarps / BW;
    const int rw = warp / BW, bw = warp % BW;
    const int NRG = P.Ny / G;
    const int rg0 = (int)(((long long)NRG * blockIdx.x) / gridDim.x);
    const int rg1 = (int)(((long long)NRG * (blockIdx.x + 1)) / gridDim.x);
    const int passes = (rg1 - rg0 + RW - 1) / RW;
    cf *ybuf = sm_y + warp * RG::WARP + g * RG::RS;
    const size_t npx = (size_t)P.Nx * P.Ny;
    const bool want_I = screen && P.inten != nullptr;
    const bool per_field = (P.flags & 2u) != 0;
    const bool accumulate = (P.flags & 1u) != 0;
    const bool summed = want_I && !per_field && P.B > 1;      // CTA-uniform
    const float pa = screen ? P.phase_a[j] : 0.f;
    const float pb = P.phase_b;
    float *acc = sm_acc + warp * 1024;

    for (int it = 0; it < passes; ++it) {
        const int rg = rg0 + it * RW + rw;
        const bool valid = rg < rg1;                           // warp-uniform
        const int y = rg * G + g;
        const size_t off = (size_t)y * P.Nx + t;
        float dnv[32];
        if (screen && valid) {
            const float *dnp = P.dn + (size_t)(j - P.j_base) * npx + off;
#pragma unroll
            for (int i = 0; i < 32; ++i) dnv[i] = __ldcs(dnp + TX * i);
        }
        if (summed) {
#pragma unroll
            for (int i = 0; i < 32; ++i) acc[i * 32 + lane] = 0.f;
        }
        if (valid) {
            for (int b = bw; b < P.B; b += BW) {
                cf *line = P.field + (size_t)b * npx + off;
                cf v[32];
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] = ld_cg(line + TX * i);
                if (inv) line_fft<TX, +1, RG::S>(v, sm_tw, ybuf, t, SyncWarp());
                if (screen) {
#pragma unroll
                    for (int i = 0; i < 32; ++i) {
                        float s, c;
                        sincosf(fmaf(pb, dnv[i], pa), &s, &c);
                        v[i] = cmul(v[i], make_float2(c, s));
                    }
                    if (want_I) {
                        if (summed) {
#pragma unroll
                            for (int i = 0; i < 32; ++i)
                                acc[i * 32 + lane] += fmaf(v[i].x, v[i].x, v[i].y * v[i].y);
                        } else {
                            float *ip = P.inten + (size_t)(j - P.j_base) * npx + off
                                        + (per_field ? (size_t)b * (size_t)P.inten_bstride : 0);
#pragma unroll
                            for (int i = 0; i < 32; ++i) {
                                float I = fmaf(v[i].x, v[i].x, v[i].y * v[i].y);
                                if (accumulate) I += ip[TX * i];
                                __stcs(ip + TX * i, I);
                            }
                        }
                    }
                }
                if (fwd) line_fft<TX, -1, RG::S>(v, sm_tw, ybuf, t, SyncWarp());
                if (scale != 1.f) {
#pragma unroll
                    for (int i = 0; i < 32; ++i) { v[i].x *= scale; v[i].y *= scale; }
                }
#pragma unroll
                for (int i = 0; i < 32; ++i) st_cg(line + TX * i, v[i]);
            }
        }
        if (summed) {
            __syncthreads();
            if (bw == 0 && valid) {
                float *ip = P.inten + (size_t)(j - P.j_base) * npx + off;
#pragma unroll
                for (int i = 0; i < 32; ++i) {
                    float I = 0.f;
                    for (int q = 0; q < BW; ++q) I += acc[q * 1024 + i * 32 + lane];
                    if (accumulate) I += ip[TX * i];
                    __stcs(ip + TX * i, I);
                }
            }
            __syncthreads();
        }
    }
}

// ----------------------------------------------------------------------------------------
// Column phase.  A tile is CW adjacent columns x all Ny rows of one field, handled by
// CW*TY threads (thread r: column c = r % CW, FFT lane t = r / CW) so that every global
// access of a warp is whole 32*CW/... byte row segments -- no transposed copy of the field
// ever exists.  The propagator values a thread needs sit at exactly the (y, c) positions it
// loads, so its slice of the table is cached in a thread-private shared-memory column and
// reloaded only when the tile or the table changes (n_ref changes once per slab).
// ----------------------------------------------------------------------------------------
template <int TY, int CW>
__device__ __forceinline__ void col_phase(const KParams &P, bool fwd, const cf *tab, bool inv, float scale,
                                          const cf *sm_tw, cf *sm_y, cf *sm_h,
                                          int &tag_ct, const cf *&tag_tab) {
    constexpr int NT = CW * TY;            // threads per tile
    constexpr int NS = kThreads / NT;      // tiles in flight per CTA
    using CG = ColGeom<TY, CW>;
    const int tid = threadIdx.x;
    const int sl = tid / NT, r = tid % NT;
    const int c = r % CW, t = r / CW;
    const int NU = (P.Nx / CW) * P.B;
    const int u0 = (int)(((long long)NU * blockIdx.x) / gridDim.x);
    const int u1 = (int)(((long long)NU * (blockIdx.x + 1)) / gridDim.x);
    const int passes = (u1 - u0 + NS - 1) / NS;
    cf *ybuf = sm_y + sl * CG::TILE + c * CG::RS;
    cf *hs = sm_h + tid;
    const size_t npx = (size_t)P.Nx * P.Ny;

    for (int it = 0; it < passes; ++it) {
        const int u = u0 + it * NS + sl;
        const bool valid = u < u1;
        const int ct = u / P.B, b = u - ct * P.B;
        const size_t off = (size_t)t * P.Nx + (size_t)ct * CW + c;
        cf *col = P.field + (size_t)b * npx + off;
        const size_t ystride = (size_t)TY * P.Nx;
        cf v[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] = valid ? ld_cg(col + ystride * i) : make_float2(0.f, 0.f);
        if (tab != nullptr && valid && (tag_ct != ct || tag_tab != tab)) {
            const cf *hp = tab + off;
#pragma unroll
            for (int i = 0; i < 32; ++i) hs[i * kThreads] = __ldg(hp + ystride * i);
            tag_ct = ct;
            tag_tab = tab;
        }
        if (fwd) line_fft<TY, -1, CG::S>(v, sm_tw, ybuf, t, SyncBlock());
        if (tab != nullptr) {
#pragma unroll
            for (int i = 0; i < 32; ++i) v[i] = cmul(v[i], hs[i * kThreads]);
        }
        if (inv) line_fft<TY, +1, CG::S>(v, sm_tw, ybuf, t, SyncBlock());
        if (scale != 1.f) {
#pragma unroll
            for (int i = 0; i < 32; ++i) { v[i].x *= scale; v[i].y *= scale; }
        }
        if (valid) {
#pragma unroll
            for (int i = 0; i < 32; ++i) st_cg(col + ystride * i, v[i]);
        }
    }
}

template <int TX, int TY, int CW>
struct SmemLayout {
    static constexpr int kTw = 32 * TX + 32 * TY;                                   // cf
    static constexpr int kRowY = kWarps * RowGeom<TX>::WARP;
    static constexpr int kColY = (kThreads / (CW * TY)) * ColGeom<TY, CW>::TILE;
    static constexpr int kY = kRowY > kColY ? kRowY : kColY;
    static constexpr int kH = 32 * kThreads;
    static constexpr int kAcc = kWarps * 1024;                                      // floats
    static constexpr size_t bytes = (size_t)(kTw + kY + kH) * sizeof(cf) + (size_t)kAcc * sizeof(float) + 16;
};

template <int TX, int TY, int CW>
__global__ void __launch_bounds__(kThreads, 1) bpm_kernel(const KParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using L = SmemLayout<TX, TY, CW>;
    cf *sm_twx = reinterpret_cast<cf *>(smem_raw);
    cf *sm_twy = sm_twx + 32 * TX;
    cf *sm_y = sm_twy + 32 * TY;
    cf *sm_h = sm_y + L::kY;
    float *sm_acc = reinterpret_cast<float *>(sm_h + L::kH);
    int *sm_abort = reinterpret_cast<int *>(sm_acc + L::kAcc);

    for (int i = threadIdx.x; i < 32 * TX; i += kThreads) sm_twx[i] = P.twx[i];
    for (int i = threadIdx.x; i < 32 * TY; i += kThreads) sm_twy[i] = P.twy[i];
    __syncthreads();

    int tag_ct = -1;
    const cf *tag_tab = nullptr;
    unsigned nbar = 0;
    for (int p = P.p0; p < P.p1; ++p) {
        bool is_row, inv, fwd;
        float scale = 1.f;
        if (P.mode == 0) {
            is_row = (p & 1) == 0;
            inv = is_row ? (p >= 2) : true;
            fwd = is_row ? ((p >> 1) < P.Nz_total) : true;
        } else {
            const PhaseProg &g = P.prog[p];
            is_row = g.is_row != 0; inv = g.inv != 0; fwd = g.fwd != 0; scale = g.scale;
        }
        if (is_row) {
            const bool screen = (P.mode == 0) && inv;
            row_phase<TX>(P, inv, screen, fwd, scale, (p >> 1) - 1, sm_twx, sm_y, sm_acc);
        } else {
            const cf *tab = (P.mode == 0) ? P.htab[p >> 1] : nullptr;
            col_phase<TY, CW>(P, fwd, tab, inv, scale, sm_twy, sm_y, sm_h, tag_ct, tag_tab);
        }
        if (p + 1 < P.p1) {
            ++nbar;
            if (grid_barrier(P.bar, nbar * gridDim.x, P.status, sm_abort)) return;
        }
    }
}

}  // namespace bb
