// bb_kernelsc.cuh -- the BPM step kernel for small grids (Nx, Ny in {128, 256}): one thread-block
// cluster per field, the field resident in the cluster's DISTRIBUTED SHARED MEMORY for the whole
// propagation ("C1/C2 ... on-chip variant").
//
// Same two-phase structure as the grid kernels:
//   row phase    R_j : IFFT_x -> x exp(i phi(dn[j-1])), |u|^2   -> FFT_x        (CTA c owns rows  [c R, (c+1) R))
//   column phase C_j : FFT_y  -> x H_j                          -> IFFT_y       (CTA d owns kx in [d W, (d+1) W))
// with R = Ny / CS, W = Nx / CS for a cluster of CS CTAs.  What differs is where the field lives between
// the phases and what separates them:
//   * every thread holds ONE 8-point segment of one line per phase (Nx Ny / (8 CS) threads per CTA), so a
//     phase is load -> transform -> pointwise -> transform -> send, with no loop;
//   * the field is held in tiles: element (y, kx) sits in the CTA that owns it for the coming phase, in tile
//     "block index along the other axis", at [y mod R][kx mod W] (row stride W + 1: reading a row and
//     reading a column of a tile are both bank-conflict free).  A phase writes its result back IN PLACE
//     (every thread to the positions it read) and the CTA then sends tile t of its buffer to CTA t with
//     one bulk copy (cp.async.bulk shared::cta -> shared::cluster), which counts its bytes on an mbarrier of
//     the receiver: a CTA starts a phase when all CS tiles have landed.  No barrier separates the phases --
//     the exchange is all-to-all, so "my tiles have arrived" implies that every CTA has finished the phase
//     before, has read its buffer and has sent from it, which is what reusing the buffers needs.
//     (BULK = false keeps the plain form for comparison: st.shared::cluster from registers into the owners'
//     buffers and barrier.cluster.arrive.release / wait.acquire between the phases -- the release has to wait
//     for the remote stores AND the intensity stores to drain, 0.5-0.8 us per phase.)
//   * the two grid barriers per step (1.55 us each through L2, profiles/r02_whatif.md) are gone; the only
//     global traffic of a step is the dn slice in, the intensity slice out and, when n_ref changes, the
//     propagator values of the CTA's columns;
//   * pointwise factors are thread-private: the thread that applies H[ky][kx] / the screen of pixel
//     (y, x) is the same in every step, so the values live in a private column of shared memory
//     (propagator: until the table changes; screen: computed while the cluster barrier is pending
//     from dn values loaded before the column phase).
// The first phase of a launch reads the field from global memory and the last one writes it back (in
// the layout the grid kernels use between launches: rows in natural kx order), so chunked runs
// (bb_propagate_host) and BB_LAUNCH_PER_PHASE work unchanged.
//
// Line transforms on 8-point threads (bb_fft8.cuh): 256 points = one warp (16 x 16 over lane pairs,
// subline8_dit / subline8_dif); 128 points = half a warp (16 x 8: a radix-16 over the lane pair
// (l, l ^ 8), twiddle, 16 x 8 transpose through shared memory, a radix-8 in registers; input and
// output both have element 16 i + l in register i of lane l).
#pragma once
#include "bb_kernels8.cuh"

namespace bb {

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ unsigned dsmem_addr(const void *local, unsigned rank) {
    unsigned a = (unsigned)__cvta_generic_to_shared(local), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_dsmem(unsigned addr, cf v) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
// bulk copy of `bytes` (multiple of 16) from this CTA's shared memory into another CTA's; the bytes are counted on
// the mbarrier `mbar` of the RECEIVING CTA (both destination addresses from dsmem_addr)
__device__ __forceinline__ void bulk_to_cta(unsigned dst, const void *src_local, unsigned bytes, unsigned mbar) {
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "r"((unsigned)__cvta_generic_to_shared(src_local)), "r"(bytes), "r"(mbar) : "memory");
}

// A line of N points on N / PT threads x PT points.
//   elem(i): line element in register i before `first` and after `second` (what is loaded / sent)
//   pix(s) : line element in register s between the two (where the pointwise factor applies)
template <int N, int PT> struct LineC;

template <> struct LineC<256, 8> {
    static constexpr int TL = 32;            // threads per line
    static constexpr int YB = 16 * 17;       // transpose region of a line (cf)
    static constexpr int TW = 256;           // twiddle table entries
    Lane8 l;
    int ll;
    __device__ __forceinline__ explicit LineC(int ll_) : ll(ll_) { l.h = ll_ >> 4; l.t = ll_ & 15; l.s = l.h ? -1.f : 1.f; }
    __device__ __forceinline__ int elem(int i) const { return 32 * i + ll; }
    __device__ __forceinline__ int pix(int s) const { return l.t + 16 * (4 * l.h + (s & 3) + 8 * (s >> 2)); }
    template <int SIGN> __device__ __forceinline__ void first(cf (&v)[8], const cf *tw, cf *yb) const { subline8_dit<SIGN, 1>(v, tw, yb, l, WarpSync()); }
    template <int SIGN> __device__ __forceinline__ void second(cf (&v)[8], const cf *tw, cf *yb) const { subline8_dif<SIGN, 1>(v, tw, yb, l, WarpSync()); }
    // tw[k1 * 16 + t] = exp(-2 pi i k1 t / 256)
    static __device__ __forceinline__ void fill_tw(cf *tw, int tid, int nt) {
        for (int i = tid; i < TW; i += nt) {
            double s, c;
            sincospi(-2.0 * (double)((i >> 4) * (i & 15)) / 256.0, &s, &c);
            tw[i] = make_float2((float)c, (float)s);
        }
    }
};

template <> struct LineC<128, 8> {
    static constexpr int TL = 16;
    static constexpr int YB = 16 * 10;       // [k1][n2] with row stride 10: conflict-free 64-bit stores and 128-bit loads
    static constexpr int TW = 128;
    int ll, h, n2;
    float s;
    __device__ __forceinline__ explicit LineC(int ll_) : ll(ll_), h(ll_ >> 3), n2(ll_ & 7) { s = h ? -1.f : 1.f; }
    __device__ __forceinline__ int elem(int i) const { return 16 * i + ll; }
    __device__ __forceinline__ int pix(int i) const { return 16 * i + ll; }
    // n = 8 n1 + n2, k = k1 + 16 k2:  X[k1 + 16 k2] = sum_n2 w_8^(n2 k2) [ w_128^(n2 k1) sum_n1 x[8 n1 + n2] w_16^(n1 k1) ]
    // lane pair (n2, h = 0 / 1) does the radix-16 over n1 = 2 i + h; lane k1 does the radix-8 over n2.
    template <int SIGN> __device__ __forceinline__ void xf(cf (&v)[8], const cf *tw, cf *yb) const {
        pair16_dit<SIGN, 8>(v, h, s);
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) {
            const int k1 = 4 * h + (jj & 3) + 8 * (jj >> 2);
            yb[k1 * 10 + n2] = cmul_s<SIGN>(v[jj], tw[k1 * 8 + n2]);
        }
        __syncwarp();
        const float4 *src = reinterpret_cast<const float4 *>(yb + ll * 10);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float4 a = src[q];
            v[2 * q] = make_float2(a.x, a.y);
            v[2 * q + 1] = make_float2(a.z, a.w);
        }
        Dft<8, SIGN>::run(v);
    }
    template <int SIGN> __device__ __forceinline__ void first(cf (&v)[8], const cf *tw, cf *yb) const { xf<SIGN>(v, tw, yb); }
    template <int SIGN> __device__ __forceinline__ void second(cf (&v)[8], const cf *tw, cf *yb) const { xf<SIGN>(v, tw, yb); }
    // tw[k1 * 8 + n2] = exp(-2 pi i k1 n2 / 128)
    static __device__ __forceinline__ void fill_tw(cf *tw, int tid, int nt) {
        for (int i = tid; i < TW; i += nt) {
            double s, c;
            sincospi(-2.0 * (double)((i >> 3) * (i & 7)) / 128.0, &s, &c);
            tw[i] = make_float2((float)c, (float)s);
        }
    }
};

// 256 points on 16 lanes x 16 points (bb_fft16.cuh: radix-16 in registers, 16 x 16 transpose, radix-16): 0.6 x the
// instructions of the 8-point form per point, half the warps.  Lane t holds element t + 16 j in register j throughout.
template <> struct LineC<256, 16> {
    static constexpr int TL = 16;
    static constexpr int YB = 16 * 17;
    static constexpr int TW = 256;
    int t;
    unsigned mask;
    __device__ __forceinline__ explicit LineC(int ll_) : t(ll_), mask(0xFFFFu << (16 * ((threadIdx.x >> 4) & 1))) {}
    __device__ __forceinline__ int elem(int j) const { return t + 16 * j; }
    __device__ __forceinline__ int pix(int j) const { return t + 16 * j; }
    template <int SIGN> __device__ __forceinline__ void first(cf (&v)[16], const cf *tw, cf *yb) const { subline_fft<SIGN, 1>(v, tw, yb, t, HalfWarpSync{mask}); }
    template <int SIGN> __device__ __forceinline__ void second(cf (&v)[16], const cf *tw, cf *yb) const { subline_fft<SIGN, 1>(v, tw, yb, t, HalfWarpSync{mask}); }
    static __device__ __forceinline__ void fill_tw(cf *tw, int tid, int nt) { LineC<256, 8>::fill_tw(tw, tid, nt); }
};

template <int NX, int NY, int CS, int PT>
struct SmemC {
    static constexpr int R = NY / CS, W = NX / CS;       // rows / columns a CTA owns
    static constexpr int NT = NX * NY / (PT * CS);       // threads of a CTA: one PT-point segment each
    static constexpr int TS = W + 1;                     // row stride inside a tile
    // 16 consecutive kx of a row span two tiles when W = 8: their distance must be 8 (mod 16) elements
    static constexpr int TILE = R * TS + ((W == 8 && R == 16) ? 8 : 0);
    static constexpr int BUF = CS * TILE;                // one tile per CTA of the cluster
    static constexpr int kTwX = LineC<NX, PT>::TW, kTwY = LineC<NY, PT>::TW;
    static constexpr int kYX = R * LineC<NX, PT>::YB, kYY = W * LineC<NY, PT>::YB;
    static constexpr int kY = kYX > kYY ? kYX : kYY;     // line transposes (rows and columns take turns)
    static constexpr int kPw = NT * PT;                  // private pointwise factors, [slot][thread]
    static constexpr size_t bytes = (size_t)(kTwX + kTwY + kY + 2 * BUF + 2 * kPw) * sizeof(cf) + 16;   // + two mbarriers
    static constexpr bool fits = NT <= 1024 && bytes <= 227 * 1024;
};

// exp(i (pb x + pa)) for the 8 dn values of a thread -> its private column of screen factors (bb.h step 4)
template <int NT, int PT>
__device__ __forceinline__ void screen_to_pw(float (&x)[PT], float pa, float pb, cf *pw) {
    float amax = 0.f;
#pragma unroll
    for (int i = 0; i < PT; ++i) {
        x[i] = fmaf(pb, x[i], pa);
        amax = fmaxf(amax, fabsf(x[i]));
    }
    if (__all_sync(0xFFFFFFFFu, amax <= 0.78539816f)) {
#pragma unroll
        for (int i = 0; i < PT; ++i) {
            float s, c;
            screen_sincos_small(x[i], s, c);
            pw[i * NT] = make_float2(c, s);
        }
    } else {
#pragma unroll      // (a rolled loop would index x[] dynamically and put the thread's dn values in local memory)
        for (int i = 0; i < PT; ++i) {
            float s, c;
            screen_sincos(x[i], s, c);
            pw[i * NT] = make_float2(c, s);
        }
    }
}


// One launch = phases [p0, p1) of the propagation of field blockIdx.x / CS by one cluster of CS CTAs.
template <int NX, int NY, int CS, int MODE, int PT>
__global__ void __launch_bounds__(SmemC<NX, NY, CS, PT>::NT, 1) bpmc_kernel(const __grid_constant__ KParams P) {
    using L = SmemC<NX, NY, CS, PT>;
    using LX = LineC<NX, PT>;
    using LY = LineC<NY, PT>;
    constexpr int NT = L::NT, R = L::R, W = L::W, TS = L::TS, TILE = L::TILE;
    constexpr bool BULK = MODE == 1;                         // 0: remote stores + cluster barriers
    constexpr unsigned kTileBytes = TILE * sizeof(cf), kBufBytes = L::BUF * sizeof(cf);   // tiles travel with their padding
    static_assert(kTileBytes % 16 == 0, "bulk copies move multiples of 16 bytes");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cf *sm_twx = reinterpret_cast<cf *>(smem_raw);
    cf *sm_twy = sm_twx + L::kTwX;
    cf *sm_y = sm_twy + L::kTwY;
    cf *rowbuf = sm_y + L::kY;           // my rows, tile d = the columns CTA d owns          (input of a row phase)
    cf *colbuf = rowbuf + L::BUF;        // my columns, tile c = the rows CTA c owns          (input of a column phase)
    cf *sm_pwH = colbuf + L::BUF;        // propagator values of my column segment, [slot][thread]
    cf *sm_pwS = sm_pwH + L::kPw;        // screen factors of my row segment for the coming row phase
    unsigned long long *sm_mbar = reinterpret_cast<unsigned long long *>(sm_pwS + L::kPw);   // [0] rowbuf, [1] colbuf: all tiles in
    const int tid = threadIdx.x;
    const unsigned rank = cluster_ctarank();
    const int b = blockIdx.x / CS;

    if (BULK && tid == 0) {
        mbar_init(sm_mbar, 1);
        mbar_init(sm_mbar + 1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_expect_tx(sm_mbar, kBufBytes);          // armed for the first exchange into either buffer
        mbar_expect_tx(sm_mbar + 1, kBufBytes);
    }
    LX::fill_tw(sm_twx, tid, NT);
    LY::fill_tw(sm_twy, tid, NT);
    __syncthreads();
    // nobody writes into a CTA that has not started (or whose mbarriers do not exist yet)
    cluster_arrive();
    cluster_wait();

    // row role: segment llx of row yl;  column role: segment lly of column kxl
    const int yl = tid / LX::TL, kxl = tid / LY::TL;
    const LX lx(tid % LX::TL);
    const LY ly(tid % LY::TL);
    const int y = (int)rank * R + yl, kx = (int)rank * W + kxl;
    cf *ybx = sm_y + yl * LX::YB, *yby = sm_y + kxl * LY::YB;
    cf *field = P.field + (long long)b * ((long long)NX * NY);
    cf *pwH = sm_pwH + tid, *pwS = sm_pwS + tid;
    const void *tagH = nullptr, *tagS = nullptr;
    const bool accumulate = (P.flags & 1u) != 0;
    // intensity summed over a batch (bb.h step 5): the host has zeroed the slices (or they hold what BB_ACCUMULATE adds to)
    const bool summed = P.B > 1 && !(P.flags & 2u);
    unsigned par_row = 0, par_col = 0;

    // the thread's propagator values H[ky = pix(s)][kx] (bb.h step 2) -> private column
    auto load_H = [&](const void *src) {
        const cf *hp = reinterpret_cast<const cf *>(src) + kx;
#pragma unroll
        for (int i = 0; i < PT; ++i) pwH[i * NT] = __ldg(hp + (long long)ly.pix(i) * NX);
        tagH = src;
    };
    auto load_dn = [&](const Phase16 &d, float (&x)[PT]) {
        const float *dnp = reinterpret_cast<const float *>(d.src) + (long long)y * NX;
#pragma unroll
        for (int i = 0; i < PT; ++i) x[i] = P.noscreen ? 0.f : __ldcs(dnp + lx.pix(i));
    };
    // bb_probe_trace: [phase][CTA][6] = phase start, transforms done, result sent, factors staged, next phase may start
    // (SM clock), the same instant on the global timer (ns)
    long long *tr = P.trace ? P.trace + ((long long)(P.p0 - P.trace_p0) * gridDim.x + blockIdx.x) * 6 : nullptr;
    const bool tracer = tr != nullptr && tid == 0;

    // BULK: all tiles of `buf` have landed.  A thread whose wait gives up flags it (bb_device_status reports it) and
    // remembers it in `gave_up`; it does NOT leave on its own -- the other warps of the CTA may have seen the tiles and
    // would wait for it at the next CTA barrier for ever.  The CTA leaves together at that barrier (send_tiles).
    bool gave_up = false;
    auto tiles_in = [&](int which, unsigned &parity) {
        if (!mbar_wait(sm_mbar + which, parity)) {
            atomicExch(P.status, 2);
            gave_up = true;
        }
        parity ^= 1u;
        if (tid == 0) mbar_expect_tx(sm_mbar + which, kBufBytes);     // armed again long before the next tiles can come
    };
    // BULK: the result is back in `own` (in place); tile t goes to CTA t's `theirs`, slot `rank`.
    // false: some thread of this CTA gave up waiting for tiles (the same answer in every thread) -- nothing is sent.
    auto send_tiles = [&](cf *own, cf *theirs, int which) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // my writes, before the copy engine reads them
        if (__syncthreads_or(gave_up)) return false;
        // one copy per tile, spread over the warps (a warp issues its copies one after the other: ~30 ns each from
        // different lanes, ~70 ns each from a loop in one lane)
        constexpr int NW = NT / 32, TPW = (CS + NW - 1) / NW;
        const int t = (tid >> 5) * TPW + (tid & 31);
        if ((tid & 31) < TPW && t < CS)
            bulk_to_cta(dsmem_addr(theirs + rank * TILE, (unsigned)t), own + t * TILE, kTileBytes,
                        dsmem_addr(sm_mbar + which, (unsigned)t));
        return true;
    };

    Phase16 d = decode_phase16(P, P.p0);
#pragma unroll 1
    for (int p = P.p0; p < P.p1; ++p) {
        const bool from_g = p == P.p0, to_g = p + 1 == P.p1;
        if (tracer) tr[0] = clock64();
        Phase16 dnx = d;
        if (!to_g) dnx = decode_phase16(P, p + 1);
        cf v[PT];
        float xn[PT];
        bool stage_next = false;
        if (d.is_row) {
            if (d.kind == 1 && tagS != d.src) {          // not staged during the previous phase
                load_dn(d, xn);
                screen_to_pw<NT, PT>(xn, d.pa, P.phase_b, pwS);
                tagS = d.src;
            }
            if (from_g) {
                const cf *src = field + (long long)y * NX;
#pragma unroll
                for (int i = 0; i < PT; ++i) v[i] = ld_cg(src + (d.first ? lx.elem(i) : lx.pix(i)));
            } else {
#pragma unroll
                for (int i = 0; i < PT; ++i) {
                    const int k = lx.elem(i);
                    v[i] = rowbuf[(k / W) * TILE + yl * TS + (k % W)];
                }
            }
            if (d.first) {
                lx.template first<+1>(v, sm_twx, ybx);
                __syncwarp();
            }
            if (d.kind == 1) {
                // u = value * screen (bb.h step 4), intensity (step 5)
#pragma unroll
                for (int i = 0; i < PT; ++i) v[i] = cmul(v[i], pwS[i * NT]);
                if (P.inten != nullptr) {
                    float *ip = P.inten + d.slice + (long long)y * NX + ((P.flags & 2u) ? (long long)b * P.inten_bstride : 0);
#pragma unroll
                    for (int i = 0; i < PT; ++i) {
                        float I = fmaf(v[i].x, v[i].x, v[i].y * v[i].y);
                        float *a = ip + lx.pix(i);
                        if (summed) {
                            atomicAdd(a, I);             // one cluster per field: the sum over the batch is made in L2
                        } else {
                            if (accumulate) I += *a;
                            __stcs(a, I);
                        }
                    }
                }
            }
            if (d.second) lx.template second<-1>(v, sm_twx, ybx);
            if (tracer) tr[1] = clock64();
            if (to_g) {
                cf *dst = field + (long long)y * NX;
#pragma unroll
                for (int i = 0; i < PT; ++i) st_cg(dst + (d.second ? lx.elem(i) : lx.pix(i)), v[i]);
            } else if constexpr (BULK) {
#pragma unroll
                for (int i = 0; i < PT; ++i) {
                    const int k = lx.elem(i);
                    rowbuf[(k / W) * TILE + yl * TS + (k % W)] = v[i];
                }
                if (!send_tiles(rowbuf, colbuf, 1)) break;       // CTA-uniform (the CTA still meets the others below)
            } else {
#pragma unroll
                for (int i = 0; i < PT; ++i) {
                    const int k = lx.elem(i);
                    st_dsmem(dsmem_addr(colbuf + rank * TILE + yl * TS + (k % W), (unsigned)(k / W)), v[i]);
                }
            }
        } else {
            stage_next = !to_g && dnx.kind == 1 && tagS != dnx.src;
            if (stage_next) load_dn(dnx, xn);            // on their way while the column phase runs
            if (tagH != d.src) load_H(d.src);            // first column phase of a launch
            if (from_g) {
                const cf *src = field + kx;
#pragma unroll
                for (int i = 0; i < PT; ++i) v[i] = ld_cg(src + (long long)ly.elem(i) * NX);
            } else {
#pragma unroll
                for (int i = 0; i < PT; ++i) {
                    const int k = ly.elem(i);
                    v[i] = colbuf[(k / R) * TILE + (k % R) * TS + kxl];
                }
            }
            ly.template first<-1>(v, sm_twy, yby);
            __syncwarp();
            // U * H (bb.h step 2)
#pragma unroll
            for (int i = 0; i < PT; ++i) v[i] = cmul(v[i], pwH[i * NT]);
            ly.template second<+1>(v, sm_twy, yby);
            if (tracer) tr[1] = clock64();
            if (to_g) {
                cf *dst = field + kx;
#pragma unroll
                for (int i = 0; i < PT; ++i) st_cg(dst + (long long)ly.elem(i) * NX, v[i]);
            } else if constexpr (BULK) {
#pragma unroll
                for (int i = 0; i < PT; ++i) {
                    const int k = ly.elem(i);
                    colbuf[(k / R) * TILE + (k % R) * TS + kxl] = v[i];
                }
                if (!send_tiles(colbuf, rowbuf, 0)) break;
            } else {
#pragma unroll
                for (int i = 0; i < PT; ++i) {
                    const int k = ly.elem(i);
                    st_dsmem(dsmem_addr(rowbuf + rank * TILE + (k % R) * TS + kxl, (unsigned)(k / R)), v[i]);
                }
            }
        }
        if (!to_g) {
            if (tracer) tr[2] = clock64();
            if constexpr (MODE == 0) cluster_arrive();
            // while the exchange is under way: the pointwise factors of the next phase
            if (d.is_row) {
                if (tagH != dnx.src) load_H(dnx.src);
            } else if (stage_next) {
                screen_to_pw<NT, PT>(xn, dnx.pa, P.phase_b, pwS);
                tagS = dnx.src;
            }
            if (tracer) tr[3] = clock64();
            if constexpr (BULK) {
                if (dnx.is_row) tiles_in(0, par_row); else tiles_in(1, par_col);
            } else {
                cluster_wait();
            }
            if (tracer) {
                tr[4] = clock64();
                long long g;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g));
                tr[5] = g;
                tr += 6 * gridDim.x;
            }
            d = dnx;
        }
    }
    // no CTA leaves while its shared memory may still be the source or the target of a copy
    if (BULK && P.p1 - P.p0 > 1) {
        cluster_arrive();
        cluster_wait();
    }
}

}  // namespace bb
