// bb_aux_kernels.cuh -- kernels off the per-slice loop: propagator table (fp64), multiplexed
// point-source spectrum, per-slice sums of dn for the adapted reference index.
#pragma once
#include <cuda_runtime.h>

namespace bb {

// DFT bin -> signed frequency index (bb.h: kx[p] = 2 pi (p < N/2 ? p : p - N) / (N d)).
__device__ __forceinline__ int freq_index(int p, int n) { return (p < n / 2) ? p : p - n; }

// H[q][p] = (s > 0) ? exp(i dz sqrt(s)) * inv_norm : 0,  s = k^2 - kx^2 - ky^2   (bb.h; reading A2).
// Everything in double, no fused multiply-adds in s (the cut-off test is a decision).
// perm > 1: column p holds DFT bin perm * (p mod Nx/perm) + p / (Nx/perm), the kx-class-major order in
// which the 16-point-thread kernel keeps the field between its phases (bb_kernels16.cuh).
__global__ void propagator_table_kernel(float2 *__restrict__ H, int Nx, int Ny, double dx, double dz,
                                        double k, double inv_norm, int perm) {
    const double two_pi = 6.283185307179586476925286766559;
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    int q = blockIdx.y;
    if (p >= Nx) return;
    const int Lc = Nx / perm;
    const int bin = perm * (p % Lc) + p / Lc;
    double kx = __ddiv_rn(__dmul_rn(two_pi, (double)freq_index(bin, Nx)), __dmul_rn((double)Nx, dx));
    double ky = __ddiv_rn(__dmul_rn(two_pi, (double)freq_index(q, Ny)), __dmul_rn((double)Ny, dx));
    double s = __dsub_rn(__dsub_rn(__dmul_rn(k, k), __dmul_rn(kx, kx)), __dmul_rn(ky, ky));
    float2 h = make_float2(0.f, 0.f);
    if (s > 0.0) {
        double sn, cs;
        sincos(__dmul_rn(dz, sqrt(s)), &sn, &cs);
        h.x = (float)(cs * inv_norm);
        h.y = (float)(sn * inv_norm);
    }
    H[(size_t)q * Nx + p] = h;
}

// Emitter data prepared for the spectrum kernel: fractional positions in units of the
// field width (double, so that the phase ramp can be range-reduced exactly), phase, amplitude.
struct EmitterPrep { double ax, ay; float phase, amp; };

__global__ void emitter_prep_kernel(const float *__restrict__ pos, const float *__restrict__ phase,
                                    const float *__restrict__ amp, int M, int Nx, int Ny, double dx,
                                    EmitterPrep *__restrict__ out) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    double X = (double)pos[2 * e] + (double)(Nx / 2) * dx;
    double Y = (double)pos[2 * e + 1] + (double)(Ny / 2) * dx;
    EmitterPrep r;
    r.ax = X / ((double)Nx * dx);
    r.ay = Y / ((double)Ny * dx);
    r.phase = phase ? phase[e] : 0.f;
    r.amp = amp ? amp[e] : 1.f;
    out[e] = r;
}

// U0[q][p] = P * sum_e a_e exp(i (phi_e - kx X_e - ky Y_e))   (bb.h bb_multiplex_psf; readings A12-A14).
// kx X_e = 2 pi f_p (X_e / (Nx dx)): the product f_p * ax is reduced mod 1 in double, the remaining
// angle (|.| <= pi + |phi|) goes through single-precision sincos.  Separable form:
// the phase ramp factorises,
//   a_e exp(i (phi_e - kx X_e - ky Y_e)) = [a_e exp(i (phi_e - kx X_e))] [exp(-i ky Y_e)] = EX[e][p] EY[e][q],
// so the sum over emitters is a complex matrix product over the bounding box of the pupil,
//   U0[q][p] = P[q][p] sum_e EY[e][q] EX[e][p]      (M x Wy)^T (M x Wx),
// instead of one sincos per (pixel, emitter).
// Bins f = i - Fx (i < Wx) along x, f = i - Fy (i < Wy) along y: [-F, F] clipped to [-N/2, N/2 - 1].
__global__ void emitter_axis_kernel(const EmitterPrep *__restrict__ em, int M, int Fx, int Wx, int Fy, int Wy,
                                    float2 *__restrict__ EX, float2 *__restrict__ EY) {
    const int e = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    const EmitterPrep E = em[e];
    if (i < Wx) {
        const double tt = (double)(i - Fx) * E.ax;
        const float r = (float)(tt - rint(tt));
        float s, c;
        sincosf(fmaf(-6.283185307179586f, r, E.phase), &s, &c);
        EX[(size_t)e * Wx + i] = make_float2(E.amp * c, E.amp * s);
    }
    if (i < Wy) {
        const double tt = (double)(i - Fy) * E.ay;
        const float r = (float)(tt - rint(tt));
        float s, c;
        sincosf(-6.283185307179586f * r, &s, &c);
        EY[(size_t)e * Wy + i] = make_float2(c, s);
    }
}

// U0 over the pupil's bounding box: 32 x 32 outputs per CTA (256 threads, 2 x 2 each), emitters in
// chunks of 32 through shared memory.  U0 must have been zeroed (pixels outside the box stay zero).
__global__ void __launch_bounds__(256) multiplex_gemm_kernel(float2 *__restrict__ U0, int Nx, int Ny, double dx, double ki2, double kc2,
                                                             const float2 *__restrict__ EX, const float2 *__restrict__ EY,
                                                             int M, int Fx, int Wx, int Fy, int Wy) {
    const double two_pi = 6.283185307179586476925286766559;
    constexpr int TK = 32;
    __shared__ float2 sx[TK][32], sy[TK][32];
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;           // outputs (ty + 16 a, tx + 16 b), a, b < 2
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    float2 acc[2][2] = {};
    for (int e0 = 0; e0 < M; e0 += TK) {
        __syncthreads();
        for (int l = threadIdx.x; l < TK * 32; l += 256) {
            const int k = l / 32, c = l % 32, e = e0 + k;
            sx[k][c] = (e < M && i0 + c < Wx) ? EX[(size_t)e * Wx + i0 + c] : make_float2(0.f, 0.f);
            sy[k][c] = (e < M && j0 + c < Wy) ? EY[(size_t)e * Wy + j0 + c] : make_float2(0.f, 0.f);
        }
        __syncthreads();
#pragma unroll 8
        for (int k = 0; k < TK; ++k) {
            const float2 x0 = sx[k][tx], x1 = sx[k][tx + 16], y0 = sy[k][ty], y1 = sy[k][ty + 16];
            acc[0][0].x = fmaf(y0.x, x0.x, fmaf(-y0.y, x0.y, acc[0][0].x)); acc[0][0].y = fmaf(y0.x, x0.y, fmaf(y0.y, x0.x, acc[0][0].y));
            acc[0][1].x = fmaf(y0.x, x1.x, fmaf(-y0.y, x1.y, acc[0][1].x)); acc[0][1].y = fmaf(y0.x, x1.y, fmaf(y0.y, x1.x, acc[0][1].y));
            acc[1][0].x = fmaf(y1.x, x0.x, fmaf(-y1.y, x0.y, acc[1][0].x)); acc[1][0].y = fmaf(y1.x, x0.y, fmaf(y1.y, x0.x, acc[1][0].y));
            acc[1][1].x = fmaf(y1.x, x1.x, fmaf(-y1.y, x1.y, acc[1][1].x)); acc[1][1].y = fmaf(y1.x, x1.y, fmaf(y1.y, x1.x, acc[1][1].y));
        }
    }
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const int j = j0 + ty + 16 * a, i = i0 + tx + 16 * b;
            if (j >= Wy || i >= Wx) continue;
            const int fq = j - Fy, fp = i - Fx;
            const double kx = __ddiv_rn(__dmul_rn(two_pi, (double)fp), __dmul_rn((double)Nx, dx));
            const double ky = __ddiv_rn(__dmul_rn(two_pi, (double)fq), __dmul_rn((double)Ny, dx));
            const double k2 = __dadd_rn(__dmul_rn(kx, kx), __dmul_rn(ky, ky));
            if (!(k2 <= kc2 && k2 >= ki2)) continue;                  // pupil: disk, or annulus (bb_multiplex_annular)
            const int p = fp >= 0 ? fp : fp + Nx, q = fq >= 0 ? fq : fq + Ny;
            U0[(size_t)q * Nx + p] = acc[a][b];
        }
}

// Per-slice partial sums of dn in double: partial[j][blockIdx.x] (fixed summation order,
// so the result is reproducible).  Used by bb_nref_from_dn.
__global__ void slice_sum_kernel(const float *__restrict__ dn, size_t npx, double *__restrict__ partial) {
    __shared__ double sm[256];
    const float *p = dn + (size_t)blockIdx.y * npx;
    size_t chunk = (npx + gridDim.x - 1) / gridDim.x;
    size_t i0 = (size_t)blockIdx.x * chunk, i1 = i0 + chunk < npx ? i0 + chunk : npx;
    double s = 0.0;
    for (size_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) s += (double)p[i];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) sm[threadIdx.x] += sm[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = sm[0];
}

// T x T windows around the emitters of every plane of a stack (bb_extract_tiles): out[e][z][ty][tx] =
// src[z][(cy - T/2 + ty) mod Ny][(cx - T/2 + tx) mod Nx], (cx, cy) = nearest pixel of emitter e; ELEM floats per pixel.
// One CTA per (emitter, plane): window origin once per CTA, 32-bit index arithmetic, rows of T contiguous pixels.
template <int ELEM>
__global__ void __launch_bounds__(256) extract_tiles_kernel(const float *__restrict__ src, int Nx, int Ny, int Np,
                                                            const float *__restrict__ pos, int M, double dx, int T,
                                                            float *__restrict__ out) {
    const int e = blockIdx.y, z = blockIdx.x;
    const long long cx = (long long)floor(__ddiv_rn((double)pos[2 * e], dx) + 0.5) + Nx / 2;
    const long long cy = (long long)floor(__ddiv_rn((double)pos[2 * e + 1], dx) + 0.5) + Ny / 2;
    const int x0 = (int)(((cx - T / 2) % Nx + Nx) % Nx), y0 = (int)(((cy - T / 2) % Ny + Ny) % Ny);
    const float *plane = src + (size_t)z * Ny * Nx * ELEM;
    float *op = out + ((size_t)e * Np + z) * T * T * ELEM;
    const int n = T * T * ELEM, rowlen = T * ELEM;
    for (int i = threadIdx.x; i < n; i += 256) {
        const int ty = i / rowlen, r = i - ty * rowlen, tx = r / ELEM, c = r - tx * ELEM;
        int x = x0 + tx, y = y0 + ty;
        if (x >= Nx) x -= Nx;
        if (y >= Ny) y -= Ny;
        op[i] = plane[((size_t)y * Nx + x) * ELEM + c];
    }
}

// Waist profile of the cylindrical light sheet (bb_lightsheet): u[y][x] = exp(-y^2 / w0^2), y = (i - Ny/2) dx.
__global__ void gaussian_sheet_kernel(float2 *__restrict__ u, int Nx, int Ny, double dx, double w0) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, yi = blockIdx.y;
    if (x >= Nx) return;
    const double y = (double)(yi - Ny / 2) * dx;
    u[(size_t)yi * Nx + x] = make_float2((float)exp(-(y * y) / (w0 * w0)), 0.f);
}

// Image formation (bb_image_formation), step 1: the emitter nearest to every pixel (periodic distance, lowest
// index on ties; double, no fused multiply-adds: the comparison is a decision).  The squared distance separates,
// d2 = ddx^2 + ddy^2 with ddx a function of (x, emitter) and ddy of (y, emitter): the expensive part (a division and
// a floor per component) is tabulated per axis, the per-pixel search is one addition and one comparison per emitter.
//   axis2[e][i] = (d - L floor(d / L + 0.5))^2,  d = (i - N/2) dx - pos[e][axis]
__global__ void emitter_axis_dist2_kernel(int N, const float *__restrict__ pos, int axis, int M, double dx, double *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, e = blockIdx.y;
    if (i >= N) return;
    const double L = __dmul_rn((double)N, dx);
    double d = __dsub_rn(__dmul_rn((double)(i - N / 2), dx), (double)pos[2 * e + axis]);
    d = __dsub_rn(d, __dmul_rn(L, floor(__dadd_rn(__ddiv_rn(d, L), 0.5))));
    out[(size_t)e * N + i] = __dmul_rn(d, d);
}
// 128 x 8 pixels per CTA, one column of 8 pixels per thread (8 running minima in registers); the axis values of 32
// emitters at a time go through shared memory: one 64-bit load of dx2 and four 128-bit broadcast loads of dy2 per
// eight distance tests.
__global__ void __launch_bounds__(128) nearest_emitter_kernel(int Nx, int Ny, int M, const double *__restrict__ dx2,
                                                              const double *__restrict__ dy2, int *__restrict__ owner) {
    __shared__ double sx[32][128];
    __shared__ __align__(16) double sy[32][8];
    const int lx = threadIdx.x;
    const int x0 = blockIdx.x * 128, y0 = blockIdx.y * 8;
    int best[8];
    double bd[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) { best[r] = 0; bd[r] = 0.0; }
    for (int e0 = 0; e0 < M; e0 += 32) {
        __syncthreads();
        for (int l = threadIdx.x; l < 32 * 128; l += 128) {
            const int k = l / 128, c = l % 128;
            sx[k][c] = (e0 + k < M && x0 + c < Nx) ? dx2[(size_t)(e0 + k) * Nx + x0 + c] : 0.0;
        }
        for (int l = threadIdx.x; l < 32 * 8; l += 128) {
            const int k = l / 8, c = l % 8;
            sy[k][c] = (e0 + k < M && y0 + c < Ny) ? dy2[(size_t)(e0 + k) * Ny + y0 + c] : 0.0;
        }
        __syncthreads();
        const int ne = min(32, M - e0);
        for (int k = 0; k < ne; ++k) {
            const double ax = sx[k][lx];
            const double2 *yp = reinterpret_cast<const double2 *>(sy[k]);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const double2 y2 = yp[h];
                const double da = __dadd_rn(ax, y2.x), db = __dadd_rn(ax, y2.y);
                if ((e0 + k) == 0 || da < bd[2 * h]) { bd[2 * h] = da; best[2 * h] = e0 + k; }
                if ((e0 + k) == 0 || db < bd[2 * h + 1]) { bd[2 * h + 1] = db; best[2 * h + 1] = e0 + k; }
            }
        }
    }
    if (x0 + lx < Nx) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
            if (y0 + r < Ny) owner[(size_t)(y0 + r) * Nx + x0 + lx] = best[r];
    }
}

// Step 2: image[r] = sum over the T x T taps t of S[r - (t - T/2)] psf[owner[r - (t - T/2)]][t] (periodic).
// A CTA computes a 32 x 8 patch; the (32 + T - 1) x (8 + T - 1) halo of S and owner sits in shared memory.  The
// owner map is piecewise constant, so a halo sees only a few emitters: their tiles are staged in shared memory too
// (up to K of them, found with a small hash set) and the inner loop is three shared-memory loads and one FFMA per
// tap; a halo with more than K emitters (cells much smaller than the tiles) gathers the tile values from global memory.
__global__ void __launch_bounds__(256) image_formation_kernel(const float *__restrict__ S, const int *__restrict__ owner, int Nx, int Ny,
                                                              const float *__restrict__ psf, int T, int K, float *__restrict__ image) {
    extern __shared__ float sm_if[];
    __shared__ int tab[64], slot_of[64], list[16], cnt, overflow;
    const int HW = 32 + T - 1, HH = 8 + T - 1, TT = T * T;
    float *sS = sm_if;
    int *sO = reinterpret_cast<int *>(sm_if + HW * HH);
    float *sP = sm_if + 2 * HW * HH;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 8;
    // halo origin: source pixel r' = r - (t - T/2) ranges over [r - (T - 1 - T/2), r + T/2]
    const int hx0 = x0 - (T - 1 - T / 2), hy0 = y0 - (T - 1 - T / 2);
    if (threadIdx.x < 64) tab[threadIdx.x] = -1;
    if (threadIdx.x == 0) { cnt = 0; overflow = 0; }
    for (int i = threadIdx.x; i < HW * HH; i += 256) {
        const int hy = i / HW, hx = i - hy * HW;
        const int sx = ((hx0 + hx) % Nx + Nx) % Nx, sy = ((hy0 + hy) % Ny + Ny) % Ny;
        sS[i] = S[(size_t)sy * Nx + sx];
        sO[i] = owner[(size_t)sy * Nx + sx];
    }
    __syncthreads();
    // the set of emitters in the halo
    for (int i = threadIdx.x; i < HW * HH; i += 256) {
        const int o = sO[i];
        int h = o & 63, tries = 0;
        for (; tries < 64; ++tries) {
            const int prev = atomicCAS(&tab[h], -1, o);
            if (prev == -1 || prev == o) break;
            h = (h + 1) & 63;
        }
        if (tries == 64) overflow = 1;
    }
    __syncthreads();
    if (threadIdx.x < 64 && tab[threadIdx.x] >= 0) {
        const int sl = atomicAdd(&cnt, 1);
        slot_of[threadIdx.x] = sl;
        if (sl < K) list[sl] = tab[threadIdx.x];
    }
    __syncthreads();
    const bool staged = !overflow && cnt <= K;
    if (staged) {
        const int n = cnt;
        for (int i = threadIdx.x; i < n * TT; i += 256) {
            const int sl = i / TT;
            sP[i] = psf[(size_t)list[sl] * TT + (i - sl * TT)];
        }
        for (int i = threadIdx.x; i < HW * HH; i += 256) {
            const int o = sO[i];
            int h = o & 63;
            while (tab[h] != o) h = (h + 1) & 63;
            sO[i] = slot_of[h] * TT;
        }
    }
    __syncthreads();
    const int lx = threadIdx.x % 32, ly = threadIdx.x / 32;
    const int x = x0 + lx, y = y0 + ly;
    if (x >= Nx || y >= Ny) return;
    float acc = 0.f;
    if (staged) {
        for (int ty = 0; ty < T; ++ty) {
            const int hrow = (ly + T - 1 - ty) * HW + lx + T - 1, trow = ty * T;
#pragma unroll 4
            for (int tx = 0; tx < T; ++tx) acc = fmaf(sS[hrow - tx], sP[sO[hrow - tx] + trow + tx], acc);
        }
    } else {
        for (int ty = 0; ty < T; ++ty)
            for (int tx = 0; tx < T; ++tx) {
                // r' = r - (t - T/2)  ->  halo index r' - h0 = l + (T - 1 - T/2) - (t - T/2) = l + T - 1 - t
                const int hi = (ly + T - 1 - ty) * HW + (lx + T - 1 - tx);
                acc = fmaf(sS[hi], __ldg(psf + ((size_t)sO[hi] * T + ty) * T + tx), acc);
            }
    }
    image[(size_t)y * Nx + x] = acc;
}

}  // namespace bb
