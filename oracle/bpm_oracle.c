/*
 * bpm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision CPU statement of the split-step beam
 * propagation method (BPM) of biobeam (arxiv 1706.02261), used only to check
 * the CUDA path.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or constant with paper_1706_02261_b200/csrc.
 *
 * What it follows.  The paper's main text ("beam-propagation
 * model (BPM) ... we use the exact propagator together with a locally adapted
 * expansion of refractive indices"; "novel multiplexing scheme") names the
 * method; its formulas are in supplementary notes that are not available, so
 * the per-slice operations are the ones BASELINE.json:north_star spells out
 * (FFT2 -> x exp(i dz sqrt(k^2-kx^2-ky^2)), evanescent cut -> IFFT2 ->
 * x exp(i k0 (n - n_ref) dz) -> record |u|^2), with the readings of
 * SURVEY.md section 8(c) (restated in DESIGN.md "Readings").  BPM is an
 * approximation scheme, so this file is the algorithm step by step in that
 * order ("Algorithm O"), not a closed form.
 *
 * Pins (tests/test_oracle_*.py, all CPU): own FFT vs the O(N^2) DFT below and
 * vs numpy's pocketfft; tilted plane wave; uniform slab with adapted n_ref;
 * step splitting; Gaussian beam vs a Hankel-quadrature angular-spectrum
 * integral and vs the paraxial closed form; Parseval; reversibility;
 * linearity / multiplex superposition; shift / transpose equivariance;
 * multiplex vs brute-force direct sum and vs the Airy amplitude; n_ref means.
 * NEXT rows (end of file; tests/test_oracle_next.py): refocus vs the plane-wave
 * closed form, vs chained homogeneous steps and its own inverse; backward run
 * vs the forward run it undoes; tiles vs array slicing; light sheet vs its
 * waist after forward propagation and vs the paraxial cylindrical beam; the
 * annular pupil vs Algorithm M and vs J0; image formation vs a delta object,
 * a single-emitter convolution by numpy FFT and linearity.
 * "parity unpinned": the paper's own Mie validation (Supp. Fig. 1) -- the
 * supplementary material is not available.
 *
 * Conventions (readings A2, A4-A10): time convention exp(-i w t);
 * forward DFT kernel exp(-i k.r), unnormalised; inverse carries 1/(Nx Ny);
 * arrays are [y][x] with x fastest; dy = dx; periodic boundaries; all scalar
 * arguments are float32 values promoted to double (the CUDA library receives
 * the same float32 values); evanescent test is s > 0 strictly, s evaluated as
 * k*k - kx*kx - ky*ky in double.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_PI 3.14159265358979323846264338327950288

typedef struct { double re, im; } cplx;

static inline cplx cmul(cplx a, cplx b) {
    cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re };
    return r;
}

/* ------------------------------------------------------------------ */
/* Brute-force DFT straight from the definition (pin P1).              */
/* out[q][p] = sum_y sum_x in[y][x] exp(sign*2*pi*i*(p x/Nx + q y/Ny)) */
/* sign = -1 forward, +1 inverse (inverse also divides by Nx*Ny).      */
/* ------------------------------------------------------------------ */
void oracle_dft2_bruteforce(const double *in, double *out, int Nx, int Ny, int sign)
{
    const cplx *a = (const cplx *)in;
    cplx *b = (cplx *)out;
    for (int q = 0; q < Ny; ++q)
        for (int p = 0; p < Nx; ++p) {
            double sr = 0.0, si = 0.0;
            for (int y = 0; y < Ny; ++y)
                for (int x = 0; x < Nx; ++x) {
                    double ph = sign * 2.0 * ORACLE_PI *
                                ((double)p * x / Nx + (double)q * y / Ny);
                    double c = cos(ph), s = sin(ph);
                    cplx v = a[(size_t)y * Nx + x];
                    sr += v.re * c - v.im * s;
                    si += v.re * s + v.im * c;
                }
            if (sign > 0) { sr /= (double)Nx * Ny; si /= (double)Nx * Ny; }
            b[(size_t)q * Nx + p].re = sr;
            b[(size_t)q * Nx + p].im = si;
        }
}

/* ------------------------------------------------------------------ */
/* Own FFT: iterative radix-2 decimation in time, power-of-two n.      */
/* Every twiddle is a direct cos/sin evaluation (no recurrences).      */
/* X[k] = sum_n x[n] exp(sign*2*pi*i*n*k/n_len); no normalisation.     */
/* ------------------------------------------------------------------ */
static void fft1_inplace(cplx *x, int n, int sign, const cplx *tw /* n/2 entries: exp(sign 2 pi i m / n) */)
{
    /* bit reversal permutation */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    (void)sign;
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, stride = n / len;
        for (int base = 0; base < n; base += len)
            for (int m = 0; m < half; ++m) {
                cplx w = tw[m * stride];
                cplx u = x[base + m];
                cplx v = cmul(x[base + m + half], w);
                x[base + m].re = u.re + v.re;  x[base + m].im = u.im + v.im;
                x[base + m + half].re = u.re - v.re;  x[base + m + half].im = u.im - v.im;
            }
    }
}

static cplx *make_twiddles(int n, int sign)
{
    int h = n / 2 > 0 ? n / 2 : 1;
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)h);
    for (int m = 0; m < h; ++m) {
        double ph = sign * 2.0 * ORACLE_PI * (double)m / (double)n;
        tw[m].re = cos(ph); tw[m].im = sin(ph);
    }
    return tw;
}

static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* 1-D transform of a contiguous line (exported for the FFT pins). */
int oracle_fft1(double *data, int n, int sign)
{
    if (!is_pow2(n)) return 1;
    cplx *tw = make_twiddles(n, sign);
    fft1_inplace((cplx *)data, n, sign, tw);
    free(tw);
    if (sign > 0) for (int i = 0; i < 2 * n; ++i) data[i] /= (double)n;
    return 0;
}

/* 2-D transform, rows (x) then columns (y).  sign=-1 forward (unnormalised),
 * sign=+1 inverse (divides by Nx*Ny).  Reading A7. */
int oracle_fft2(double *data, int Nx, int Ny, int sign)
{
    if (!is_pow2(Nx) || !is_pow2(Ny)) return 1;
    cplx *a = (cplx *)data;
    cplx *twx = make_twiddles(Nx, sign), *twy = make_twiddles(Ny, sign);
    #pragma omp parallel
    {
        cplx *col = (cplx *)malloc(sizeof(cplx) * (size_t)Ny);
        #pragma omp for schedule(static)
        for (int y = 0; y < Ny; ++y) fft1_inplace(a + (size_t)y * Nx, Nx, sign, twx);
        #pragma omp for schedule(static)
        for (int x = 0; x < Nx; ++x) {
            for (int y = 0; y < Ny; ++y) col[y] = a[(size_t)y * Nx + x];
            fft1_inplace(col, Ny, sign, twy);
            for (int y = 0; y < Ny; ++y) a[(size_t)y * Nx + x] = col[y];
        }
        free(col);
    }
    if (sign > 0) {
        double inv = 1.0 / ((double)Nx * (double)Ny);
        #pragma omp parallel for schedule(static)
        for (long i = 0; i < 2L * Nx * Ny; ++i) data[i] *= inv;
    }
    free(twx); free(twy);
    return 0;
}

/* Angular frequency of DFT bin p on an n-point grid of pitch d (reading A2):
 * kx[p] = 2 pi (p < n/2 ? p : p - n) / (n d). */
static inline double kfreq(int p, int n, double d)
{
    int f = (p < n / 2) ? p : p - n;
    return 2.0 * ORACLE_PI * (double)f / ((double)n * d);
}

/* ------------------------------------------------------------------ */
/* One BPM step, Algorithm O body (north_star sentence 2; readings     */
/* A2, A4-A7):                                                         */
/*   U = FFT2(u);  U *= (s>0) ? exp(+i dz sqrt(s)) : 0,                */
/*                 s = k^2 - kx^2 - ky^2,  k = k0*nref                 */
/*   u = IFFT2(U); u *= exp(+i k0 dz (n0 + dn - nref))                 */
/*   I = |u|^2   (written if I_out != NULL)                            */
/* u: double complex [Ny][Nx] in place; dn: float32 slice [Ny][Nx] or  */
/* NULL (= 0).  Scalars are float32 promoted (header).                 */
/* ------------------------------------------------------------------ */
int oracle_bpm_step(double *u, int Nx, int Ny, const float *dn,
                    float dx_f, float dz_f, float lambda_f, float n0_f, float nref_f,
                    double *I_out)
{
    const double dx = dx_f, dz = dz_f, lambda = lambda_f, n0 = n0_f, nref = nref_f;
    const double k0 = 2.0 * ORACLE_PI / lambda;
    const double k = k0 * nref;
    if (oracle_fft2(u, Nx, Ny, -1)) return 1;
    cplx *a = (cplx *)u;
    #pragma omp parallel for schedule(static)
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        for (int p = 0; p < Nx; ++p) {
            double kx = kfreq(p, Nx, dx);
            double s = k * k - kx * kx - ky * ky;
            cplx *v = &a[(size_t)q * Nx + p];
            if (s > 0.0) {
                double ph = dz * sqrt(s);
                cplx h = { cos(ph), sin(ph) };
                *v = cmul(*v, h);
            } else {
                v->re = 0.0; v->im = 0.0;
            }
        }
    }
    if (oracle_fft2(u, Nx, Ny, +1)) return 1;
    #pragma omp parallel for schedule(static)
    for (int y = 0; y < Ny; ++y)
        for (int x = 0; x < Nx; ++x) {
            size_t i = (size_t)y * Nx + x;
            double d = dn ? (double)dn[i] : 0.0;
            double ph = k0 * dz * (n0 + d - nref);
            cplx e = { cos(ph), sin(ph) };
            a[i] = cmul(a[i], e);
            if (I_out) I_out[i] = a[i].re * a[i].re + a[i].im * a[i].im;
        }
    return 0;
}

/* Conjugate (time-reversed) step, used by the reversibility pin P8:
 * u *= conj(screen);  U = FFT2(u);  U *= (s>0) ? conj(H) : 0;  u = IFFT2(U). */
int oracle_bpm_step_backward(double *u, int Nx, int Ny, const float *dn,
                             float dx_f, float dz_f, float lambda_f, float n0_f, float nref_f)
{
    const double dx = dx_f, dz = dz_f, lambda = lambda_f, n0 = n0_f, nref = nref_f;
    const double k0 = 2.0 * ORACLE_PI / lambda;
    const double k = k0 * nref;
    cplx *a = (cplx *)u;
    for (int y = 0; y < Ny; ++y)
        for (int x = 0; x < Nx; ++x) {
            size_t i = (size_t)y * Nx + x;
            double d = dn ? (double)dn[i] : 0.0;
            double ph = -k0 * dz * (n0 + d - nref);
            cplx e = { cos(ph), sin(ph) };
            a[i] = cmul(a[i], e);
        }
    if (oracle_fft2(u, Nx, Ny, -1)) return 1;
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        for (int p = 0; p < Nx; ++p) {
            double kx = kfreq(p, Nx, dx);
            double s = k * k - kx * kx - ky * ky;
            cplx *v = &a[(size_t)q * Nx + p];
            if (s > 0.0) {
                double ph = -dz * sqrt(s);
                cplx h = { cos(ph), sin(ph) };
                *v = cmul(*v, h);
            } else { v->re = 0.0; v->im = 0.0; }
        }
    }
    return oracle_fft2(u, Nx, Ny, +1);
}

/* ------------------------------------------------------------------ */
/* Algorithm O, whole propagation of ONE field (reading A6: Nz steps,  */
/* step j uses dn[j], I[j] is the intensity after step j).             */
/* field_c64: float pairs [Ny][Nx] (the same complex64 array the CUDA  */
/* path receives), promoted to double.  nref: float[Nz] or NULL (=n0). */
/* field_out: double complex [Ny][Nx].  intensity: double [Nz][Ny][Nx] */
/* or NULL; accumulate != 0 adds to its contents (reading A11).        */
/* ------------------------------------------------------------------ */
int oracle_propagate(const float *field_c64, const float *dn, int Nx, int Ny, int Nz,
                     float dx, float dz, float lambda, float n0, const float *nref,
                     double *field_out, double *intensity, int accumulate)
{
    size_t npx = (size_t)Nx * Ny;
    for (size_t i = 0; i < 2 * npx; ++i) field_out[i] = (double)field_c64[i];
    double *Itmp = NULL;
    if (intensity && accumulate) Itmp = (double *)malloc(sizeof(double) * npx);
    for (int j = 0; j < Nz; ++j) {
        float nr = nref ? nref[j] : n0;
        double *Ij = intensity ? (accumulate ? Itmp : intensity + (size_t)j * npx) : NULL;
        int rc = oracle_bpm_step(field_out, Nx, Ny, dn ? dn + (size_t)j * npx : NULL,
                                 dx, dz, lambda, n0, nr, Ij);
        if (rc) { free(Itmp); return rc; }
        if (intensity && accumulate)
            for (size_t i = 0; i < npx; ++i) intensity[(size_t)j * npx + i] += Itmp[i];
    }
    free(Itmp);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Algorithm M (multiplexed point sources; "sets of   */
/* 100s to 1000s of mutually independent ... PSFs ... within single,   */
/* highly multiplexed simulations", line 29 "multiplexed diffraction-  */
/* limited point-sources"; readings A12-A14):                          */
/*   P[q][p]  = 1 if kx^2 + ky^2 <= (k0 NA)^2 else 0                   */
/*   U0[q][p] = P * sum_e a_e exp(i (phi_e - kx X_e - ky Y_e)),        */
/*              X_e = x_e + (Nx/2) dx,  Y_e = y_e + (Ny/2) dx          */
/*   u0 = IFFT2(U0) * (Nx Ny / sum P)                                  */
/* pos: float[M][2] (x,y) in um, origin at pixel (Nx/2, Ny/2).         */
/* phase/amp may be NULL (0 / 1).  out: double complex [Ny][Nx].       */
/* ------------------------------------------------------------------ */
int oracle_multiplex_psf(const float *pos, const float *phase, const float *amp, int M,
                         float NA_f, int Nx, int Ny, float dx_f, float lambda_f, double *out)
{
    const double dx = dx_f, lambda = lambda_f, NA = NA_f;
    const double k0 = 2.0 * ORACLE_PI / lambda;
    const double kc2 = (k0 * NA) * (k0 * NA);
    cplx *a = (cplx *)out;
    long count = 0;
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        for (int p = 0; p < Nx; ++p) {
            double kx = kfreq(p, Nx, dx);
            if (kx * kx + ky * ky <= kc2) ++count;
        }
    }
    if (count == 0) return 2;
    #pragma omp parallel for schedule(dynamic, 4)
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        for (int p = 0; p < Nx; ++p) {
            double kx = kfreq(p, Nx, dx);
            double sr = 0.0, si = 0.0;
            if (kx * kx + ky * ky <= kc2) {
                for (int e = 0; e < M; ++e) {
                    double X = (double)pos[2 * e] + (double)(Nx / 2) * dx;
                    double Y = (double)pos[2 * e + 1] + (double)(Ny / 2) * dx;
                    double ph = (phase ? (double)phase[e] : 0.0) - kx * X - ky * Y;
                    double am = amp ? (double)amp[e] : 1.0;
                    sr += am * cos(ph);
                    si += am * sin(ph);
                }
            }
            a[(size_t)q * Nx + p].re = sr;
            a[(size_t)q * Nx + p].im = si;
        }
    }
    if (oracle_fft2(out, Nx, Ny, +1)) return 1;
    double scale = (double)Nx * (double)Ny / (double)count;
    for (size_t i = 0; i < 2 * (size_t)Nx * Ny; ++i) out[i] *= scale;
    return 0;
}

/* ------------------------------------------------------------------ */
/* Locally adapted reference index (reading A3): n_ref[j] = n0 + mean  */
/* of dn over the slab of `slab` consecutive slices that contains j    */
/* (last slab may be short).  Result rounded to float32.               */
/* ------------------------------------------------------------------ */
int oracle_nref_from_dn(const float *dn, int Nx, int Ny, int Nz, float n0, int slab, float *nref_out)
{
    if (slab < 1) return 1;
    size_t npx = (size_t)Nx * Ny;
    for (int j0 = 0; j0 < Nz; j0 += slab) {
        int j1 = j0 + slab < Nz ? j0 + slab : Nz;
        long double sum = 0.0L;
        for (int j = j0; j < j1; ++j) {
            double s = 0.0;
            for (size_t i = 0; i < npx; ++i) s += (double)dn[(size_t)j * npx + i];
            sum += s;
        }
        double mean = (double)(sum / ((long double)npx * (long double)(j1 - j0)));
        float v = (float)((double)n0 + mean);
        for (int j = j0; j < j1; ++j) nref_out[j] = v;
    }
    return 0;
}

/* ================================================================== */
/* NEXT rows of SURVEY.md section 8(f).  Each restates a passage of    */
/* the paper in the notation of Algorithm O; pins in                   */
/* tests/test_oracle_next.py.                                          */
/* ================================================================== */

/* ------------------------------------------------------------------ */
/* NEXT-4 (Fig. 2c "reversal of guide star emitted   */
/* light fields"; line 33).  Time-reversed propagation: for j = Nz-1   */
/* .. 0 record I[j] = |u|^2 (the plane z = (j+1) dz the forward run    */
/* recorded as I[j]) and undo step j with oracle_bpm_step_backward     */
/* (pin P8, reading A4: every phase factor conjugated, evanescent      */
/* modes stay cut).  intensity may be NULL.                            */
/* ------------------------------------------------------------------ */
int oracle_propagate_backward(const float *field_c64, const float *dn, int Nx, int Ny, int Nz,
                              float dx, float dz, float lambda, float n0, const float *nref,
                              double *field_out, double *intensity)
{
    size_t npx = (size_t)Nx * Ny;
    for (size_t i = 0; i < 2 * npx; ++i) field_out[i] = (double)field_c64[i];
    for (int j = Nz - 1; j >= 0; --j) {
        if (intensity)
            for (size_t i = 0; i < npx; ++i)
                intensity[(size_t)j * npx + i] = field_out[2 * i] * field_out[2 * i] + field_out[2 * i + 1] * field_out[2 * i + 1];
        int rc = oracle_bpm_step_backward(field_out, Nx, Ny, dn + (size_t)j * npx, dx, dz, lambda, n0,
                                          nref ? nref[j] : n0);
        if (rc) return rc;
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* NEXT-1 ("propagating light ... through an     */
/* idealized, refocusing lens towards the camera").  The idealised     */
/* lens is free-space propagation in a homogeneous medium of index n   */
/* over a SIGNED distance dz (negative: back to the emitter plane):    */
/*   U = FFT2(u);  U *= (s > 0) ? exp(i dz sqrt(s)) : 0;  u = IFFT2(U) */
/* with s = k^2 - kx^2 - ky^2, k = k0 n: one diffraction half of an    */
/* Algorithm-O step, no screen.                                        */
/* ------------------------------------------------------------------ */
int oracle_refocus(double *u, int Nx, int Ny, float dx_f, float dz_f, float lambda_f, float n_f)
{
    const double dx = dx_f, dz = dz_f, lambda = lambda_f, n = n_f;
    const double k = 2.0 * ORACLE_PI / lambda * n;
    cplx *a = (cplx *)u;
    if (oracle_fft2(u, Nx, Ny, -1)) return 1;
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        for (int p = 0; p < Nx; ++p) {
            double kx = kfreq(p, Nx, dx);
            double s = k * k - kx * kx - ky * ky;
            cplx *v = &a[(size_t)q * Nx + p];
            if (s > 0.0) {
                double ph = dz * sqrt(s);
                cplx h = { cos(ph), sin(ph) };
                *v = cmul(*v, h);
            } else { v->re = 0.0; v->im = 0.0; }
        }
    }
    return oracle_fft2(u, Nx, Ny, +1);
}

/* ------------------------------------------------------------------ */
/* NEXT-1, second half ("quasi-continuum of          */
/* spatially-dependent, volumetric PSFs"): the T x T window around     */
/* every emitter of every plane of a stack.  src: [Np][Ny][Nx] of      */
/* `elem` doubles per pixel (1 intensity, 2 complex); centre pixel of  */
/* emitter e: (floor(x_e / dx + 0.5) + Nx/2, floor(y_e / dx + 0.5) +   */
/* Ny/2) (emitter coordinates as in oracle_multiplex_psf); window      */
/* [c - T/2, c - T/2 + T) per axis, periodic.  out: [M][Np][T][T].     */
/* ------------------------------------------------------------------ */
int oracle_extract_tiles(const double *src, int elem, int Nx, int Ny, int Np, const float *pos, int M,
                         float dx_f, int T, double *out)
{
    if ((elem != 1 && elem != 2) || T < 1 || T > Nx || T > Ny) return 1;
    const double dx = dx_f;
    for (int e = 0; e < M; ++e) {
        long cx = (long)floor((double)pos[2 * e] / dx + 0.5) + Nx / 2;
        long cy = (long)floor((double)pos[2 * e + 1] / dx + 0.5) + Ny / 2;
        for (int z = 0; z < Np; ++z)
            for (int ty = 0; ty < T; ++ty)
                for (int tx = 0; tx < T; ++tx) {
                    long x = ((cx - T / 2 + tx) % Nx + Nx) % Nx;
                    long y = ((cy - T / 2 + ty) % Ny + Ny) % Ny;
                    for (int c = 0; c < elem; ++c)
                        out[((((size_t)e * Np + z) * T + ty) * T + tx) * elem + c] =
                            src[(((size_t)z * Ny + y) * Nx + x) * elem + c];
                }
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* NEXT-2 ("a cylindrical sheet of light is          */
/* propagated"; BASELINE.json configs[1]: "cylindrically focused       */
/* Gaussian sheet (NA 0.1 in y, flat in x)").  Reading: */
/* the field at the input plane is the waist profile exp(-y^2 / w0^2), */
/* w0 = lambda / (pi NA), propagated BACK by z_focus in the            */
/* homogeneous medium n0 -- a one-dimensional angular spectrum:        */
/*   g = IFFT_y[ exp(-i z_f sqrt(k^2 - ky^2)) FFT_y[ exp(-y^2/w0^2) ] ]*/
/* (evanescent ky cut), y_i = (i - Ny/2) dx, uniform in x.             */
/* out: double complex [Ny][Nx].                                       */
/* ------------------------------------------------------------------ */
int oracle_lightsheet(int Nx, int Ny, float dx_f, float lambda_f, float n0_f, float NA_f, float zf_f, double *out)
{
    const double dx = dx_f, lambda = lambda_f, n0 = n0_f, NA = NA_f, zf = zf_f;
    const double k = 2.0 * ORACLE_PI / lambda * n0;
    const double w0 = lambda / (ORACLE_PI * NA);
    if (!is_pow2(Ny)) return 1;
    cplx *g = (cplx *)malloc((size_t)Ny * sizeof(cplx));
    if (!g) return 3;
    for (int i = 0; i < Ny; ++i) {
        double y = (double)(i - Ny / 2) * dx;
        g[i].re = exp(-(y * y) / (w0 * w0));
        g[i].im = 0.0;
    }
    if (oracle_fft1((double *)g, Ny, -1)) { free(g); return 1; }
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        double s = k * k - ky * ky;
        if (s > 0.0) {
            double ph = -zf * sqrt(s);
            cplx h = { cos(ph), sin(ph) };
            g[q] = cmul(g[q], h);
        } else { g[q].re = 0.0; g[q].im = 0.0; }
    }
    if (oracle_fft1((double *)g, Ny, +1)) { free(g); return 1; }
    cplx *a = (cplx *)out;
    for (int y = 0; y < Ny; ++y)
        for (int x = 0; x < Nx; ++x) a[(size_t)y * Nx + x] = g[y];
    free(g);
    return 0;
}

/* ------------------------------------------------------------------ */
/* NEXT-2, Bessel beams and lattices ("Bessel         */
/* lattices"; line 17, Fig. 1d).  Algorithm M with an ANNULAR pupil:   */
/*   P[q][p] = 1 if (k0 NA_in)^2 <= kx^2 + ky^2 <= (k0 NA_out)^2       */
/* every "emitter" is then a Bessel-beam focus (a thin annulus gives   */
/* J0(k0 NA r)); a lattice is a row of them.  NA_in = 0 is Algorithm M.*/
/* ------------------------------------------------------------------ */
int oracle_multiplex_annular(const float *pos, const float *phase, const float *amp, int M,
                             float NAin_f, float NAout_f, int Nx, int Ny, float dx_f, float lambda_f, double *out)
{
    const double dx = dx_f, lambda = lambda_f;
    const double k0 = 2.0 * ORACLE_PI / lambda;
    const double ki2 = (k0 * (double)NAin_f) * (k0 * (double)NAin_f);
    const double kc2 = (k0 * (double)NAout_f) * (k0 * (double)NAout_f);
    cplx *a = (cplx *)out;
    long count = 0;
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        for (int p = 0; p < Nx; ++p) {
            double kx = kfreq(p, Nx, dx);
            double k2 = kx * kx + ky * ky;
            if (k2 <= kc2 && k2 >= ki2) ++count;
        }
    }
    if (count == 0) return 2;
    #pragma omp parallel for schedule(dynamic, 4)
    for (int q = 0; q < Ny; ++q) {
        double ky = kfreq(q, Ny, dx);
        for (int p = 0; p < Nx; ++p) {
            double kx = kfreq(p, Nx, dx);
            double k2 = kx * kx + ky * ky;
            double sr = 0.0, si = 0.0;
            if (k2 <= kc2 && k2 >= ki2) {
                for (int e = 0; e < M; ++e) {
                    double X = (double)pos[2 * e] + (double)(Nx / 2) * dx;
                    double Y = (double)pos[2 * e + 1] + (double)(Ny / 2) * dx;
                    double ph = (phase ? (double)phase[e] : 0.0) - kx * X - ky * Y;
                    double am = amp ? (double)amp[e] : 1.0;
                    sr += am * cos(ph);
                    si += am * sin(ph);
                }
            }
            a[(size_t)q * Nx + p].re = sr;
            a[(size_t)q * Nx + p].im = si;
        }
    }
    if (oracle_fft2(out, Nx, Ny, +1)) return 1;
    double scale = (double)Nx * (double)Ny / (double)count;
    for (size_t i = 0; i < 2 * (size_t)Nx * Ny; ++i) out[i] *= scale;
    return 0;
}

/* ------------------------------------------------------------------ */
/* NEXT-3 ("Convolving the exhaustively sampled set  */
/* of spatially-varying PSFs with the fluorescent object"; line 17,    */
/* Fig. 1c).  Reading (A18): the PSF is piecewise constant   */
/* over the cells of the emitter grid -- a source pixel r' radiates    */
/* with the intensity PSF tile of the emitter NEAREST to it (ties: the */
/* lowest emitter index) -- and the camera image of one object plane is*/
/*   image[r] = sum_{r'} S[r'] psf[e(r')][r - r' + T/2],  S = F * E    */
/* (fluorophore density times excitation intensity), the sum over the  */
/* r' whose T x T tile covers r, periodic.  psf: [M][T][T] (tile       */
/* centre at index T/2), S: [Ny][Nx], image: [Ny][Nx].                 */
/* ------------------------------------------------------------------ */
int oracle_image_formation(const double *S, int Nx, int Ny, const float *pos, int M, float dx_f,
                           const double *psf, int T, double *image)
{
    if (T < 1 || T > Nx || T > Ny || M < 1) return 1;
    const double dx = dx_f;
    int *owner = (int *)malloc((size_t)Nx * Ny * sizeof(int));
    if (!owner) return 3;
    for (int y = 0; y < Ny; ++y)
        for (int x = 0; x < Nx; ++x) {
            double px = (double)(x - Nx / 2) * dx, py = (double)(y - Ny / 2) * dx;
            int best = 0;
            double bd = 0.0;
            for (int e = 0; e < M; ++e) {
                double ddx = px - (double)pos[2 * e], ddy = py - (double)pos[2 * e + 1];
                /* periodic distance */
                double Lx = (double)Nx * dx, Ly = (double)Ny * dx;
                ddx -= Lx * floor(ddx / Lx + 0.5);
                ddy -= Ly * floor(ddy / Ly + 0.5);
                double d2 = ddx * ddx + ddy * ddy;
                if (e == 0 || d2 < bd) { bd = d2; best = e; }
            }
            owner[(size_t)y * Nx + x] = best;
        }
    #pragma omp parallel for schedule(static)
    for (int y = 0; y < Ny; ++y)
        for (int x = 0; x < Nx; ++x) {
            double acc = 0.0;
            for (int ty = 0; ty < T; ++ty)
                for (int tx = 0; tx < T; ++tx) {
                    /* source pixel r' = r - (t - T/2) */
                    int sx = ((x - (tx - T / 2)) % Nx + Nx) % Nx;
                    int sy = ((y - (ty - T / 2)) % Ny + Ny) % Ny;
                    size_t si = (size_t)sy * Nx + sx;
                    acc += S[si] * psf[((size_t)owner[si] * T + ty) * T + tx];
                }
            image[(size_t)y * Nx + x] = acc;
        }
    free(owner);
    return 0;
}

int oracle_abi_version(void) { return 2; }
