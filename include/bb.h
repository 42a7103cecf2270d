/*
 * bb.h -- C ABI of libbiobeam_b200.so: the split-step beam-propagation (BPM) hot path of
 * biobeam (arxiv 1706.02261), hand-written for NVIDIA B200 (sm_100a).
 *
 * What the library computes.  The paper's main text names the method (PAPER.md line 21:
 * "beam-propagation model (BPM) ... we use the exact propagator together with a locally
 * adapted expansion of refractive indices", and the "novel multiplexing scheme" that
 * propagates 100s-1000s of point sources in one field); its formulas are in supplementary
 * notes that are not available, so the per-slice operations are the ones
 * BASELINE.json:north_star states, with the readings listed in DESIGN.md ("Readings"):
 *
 *   for j = 0 .. Nz-1:                                    (reading A5, A6)
 *       U  = FFT2(u)                                      unnormalised, kernel exp(-i k.r)
 *       U *= (s > 0) ? exp(+i dz sqrt(s)) : 0             s = k^2 - kx^2 - ky^2,  k = k0 n_ref[j]
 *       u  = IFFT2(U)                                     with 1/(Nx Ny)
 *       u *= exp(+i k0 dz (n0 + dn[j] - n_ref[j]))        k0 = 2 pi / lambda
 *       I[j] = sum over batch |u|^2                       (or per field / accumulated)
 *
 *   kx[p] = 2 pi (p < Nx/2 ? p : p - Nx) / (Nx dx), likewise ky with Ny and dy = dx.
 *
 * Conventions.  All lengths in micrometres; lambda is the vacuum wavelength.  Arrays are
 * row-major with x fastest: field [B][Ny][Nx] of float pairs (re, im) = complex64,
 * volumes [Nz][Ny][Nx] float32.  Scalars are float32; every table is built in double from
 * the float32 values promoted to double.  Nx and Ny must be powers of two in [32, 2048]
 * (Nx != Ny allowed; SURVEY 8b asks for [128, 2048], PAPER.md line 31 uses 1024 x 2048); a grid
 * with a 2048-point side needs both sides >= 256.
 * Periodic lateral boundaries (plain FFT).
 *
 * Pointers.  Unless a parameter says HOST, pointers are DEVICE pointers on the current CUDA
 * device (e.g. torch tensor data_ptr()).  The caller owns every buffer in a signature; the
 * library owns only its plan cache (twiddle tables, propagator tables, a few KB of
 * workspace), created lazily and released by bb_shutdown().  The library never copies user
 * data between host and device except in bb_propagate_host() and for the small HOST arrays.
 *
 * Execution.  Device-pointer calls enqueue work on the given stream and return without
 * waiting for it (they may synchronise the first time a shape or reference index is seen,
 * while tables are built).  Calls on one device must not overlap on different streams.
 * There is no CPU fallback and no other backend: on a device that is not sm_100 every
 * compute call returns BB_ERR_ARCH.
 *
 * Errors.  Every call returns a bb_status; nothing throws or aborts.  Arguments are
 * checked before any launch.  bb_last_error() returns a thread-local message for the last
 * non-OK status.
 */
#ifndef BIOBEAM_B200_BB_H
#define BIOBEAM_B200_BB_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    BB_OK = 0,
    BB_ERR_INVALID_ARG = 1,        /* NULL pointer, non-positive scalar, bad count, bad flags */
    BB_ERR_UNSUPPORTED_SHAPE = 2,  /* Nx or Ny not a power of two in the supported range (see above) */
    BB_ERR_CUDA = 3,               /* a CUDA call failed (message in bb_last_error) */
    BB_ERR_OOM = 4,                /* device or host allocation failed */
    BB_ERR_ARCH = 5,               /* current device is not compute capability 10.x */
    BB_ERR_INTERNAL = 6            /* device-side watchdog tripped (grid barrier timeout) */
} bb_status;

/* bb_opts.flags */
#define BB_ACCUMULATE          1u  /* intensity_out += |u|^2 instead of = (reading A11) */
#define BB_INTENSITY_PER_FIELD 2u  /* intensity_out is [B][Nz][Ny][Nx], not summed over the batch */
#define BB_LAUNCH_PER_PHASE    4u  /* diagnostic: one kernel launch per half-step instead of one
                                      persistent cooperative kernel (same arithmetic, same results) */
#define BB_BACKWARD            8u  /* time-reversed (phase-conjugate) propagation, PAPER.md line 27 (Fig. 2c: "reversal
                                      of guide star emitted light fields") and line 33: for j = Nz-1 .. 0
                                          I[j] = |u|^2;  u *= conj(screen_j);  U = FFT2(u);  U *= conj(H_j);  u = IFFT2(U)
                                      (evanescent modes stay cut).  field in: u at z = Nz dz; out: u at z = 0.
                                      Undoes a forward run exactly where no mode is evanescent. */
#define BB_HOMOGENEOUS        16u  /* no sample: Nz steps through the medium n0 (no phase screen; dn_volume is not
                                      read and may be NULL; nref must be NULL).  intensity_out[j] = |u|^2 after step j:
                                      the through-focus stack of a field ("volumetric PSFs") */

typedef struct {
    int struct_size;     /* sizeof(bb_opts); lets the struct grow compatibly */
    int batch;           /* B >= 1 independent fields, contiguous [B][Ny][Nx], one shared dn volume
                            (north_star item 4, BASELINE.json configs[4]) */
    const float *nref;   /* HOST float[Nz]: reference index n_ref[j] of step j (reading A3),
                            or NULL = n0 for every step.  HOST, not device (a deviation from SURVEY 8b):
                            the host picks the cached propagator table of every step and the live
                            kx band from n_ref before it enqueues anything; a device array would have
                            to be copied back and waited for at that point. */
    unsigned flags;      /* BB_ACCUMULATE | BB_INTENSITY_PER_FIELD | BB_LAUNCH_PER_PHASE | BB_BACKWARD | BB_HOMOGENEOUS */
    void *stream;        /* cudaStream_t; NULL = the legacy default stream */
} bb_opts;

/*
 * bb_propagate -- north_star: "bb_propagate(field, dn_volume, Nx, Ny, Nz, dx, dz, lambda, n0,
 * intensity_out)".  Algorithm above with B = 1, n_ref = n0, flags = 0, default stream.
 *   field          in: u at the input plane z = 0; out: u after Nz steps (in place)
 *   dn_volume      float[Nz][Ny][Nx] = n - n0; step j uses slice j
 *   intensity_out  float[Nz][Ny][Nx], slice j = |u|^2 after step j (z = (j+1) dz); may be NULL
 */
int bb_propagate(void *field, const float *dn_volume, int Nx, int Ny, int Nz,
                 float dx, float dz, float lambda, float n0, float *intensity_out);

/* Same with options (batch, adapted n_ref, accumulate / per-field intensity, backward, homogeneous,
 * stream).  opts may be NULL.  Kernel selection (results do not depend on it beyond rounding): grids
 * with both sides in {128, 256} and at least one side of 128 run the cluster kernel -- one thread-block
 * cluster of 16 CTAs (8 if the device cannot place 16) per field, the field resident in the cluster's
 * distributed shared memory for the whole call, dn and the intensity the only per-step global traffic;
 * batches take one cluster per field, and a summed batch intensity is then added up with global atomics
 * into slices the call zeroes first (BB_KC_FORCE=1 in the environment: 256 x 256 as well; BB_DISABLE_KC=1:
 * never) -- other grids
 * with sides in {256, 512, 1024, 2048} run the 16-point-thread kernel -- for a batch only while the screen
 * factors of a CTA's rows fit its buffer, ceil(Ny / SMs) * Nx <= 8192; a larger batch runs field by field
 * on the single-field variant (dn is then read once per field) -- everything else the 32-point-thread kernel
 * (sides up to 1024).  The 8-point-thread kernel runs the transforms of bb_fft2 / bb_multiplex_* on grids with a 2048-point
 * side and, with BB_USE_K8=1 in the environment, propagations.  The summed intensity of a
 * batch is accumulated with atomics (shared memory, or global memory in the cluster kernel): its summation order, hence its last bits, can
 * differ between runs (tolerance contract: relative L2 <= 1e-4 against the definition). */
int bb_propagate_ex(void *field, const float *dn_volume, int Nx, int Ny, int Nz,
                    float dx, float dz, float lambda, float n0, float *intensity_out,
                    const bb_opts *opts);

/*
 * bb_propagate_host -- the same computation for HOST buffers: field, dn_volume and
 * intensity_out are HOST pointers (pinned memory gives overlap of the copies with the
 * kernels; pageable memory works but serialises).  The dn volume is streamed to the device
 * in z-chunks while earlier chunks are computed and their intensity slices are streamed back;
 * every step still runs in the CUDA kernels.  Synchronous: returns when the results are in
 * host memory.  opts->stream is ignored (the call owns its streams).
 */
int bb_propagate_host(void *field_host, const float *dn_volume_host, int Nx, int Ny, int Nz,
                      float dx, float dz, float lambda, float n0, float *intensity_out_host,
                      const bb_opts *opts);

/*
 * bb_nref_from_dn -- locally adapted reference index ("locally adapted
 * expansion of refractive indices"; reading A3): n_ref[j] = n0 + mean of dn over the slab of
 * `slab` consecutive slices that contains j (the last slab may be short), means in double,
 * result rounded to float32.  dn is a DEVICE pointer, nref_out a HOST float[Nz].
 * Synchronises the stream.
 */
int bb_nref_from_dn(const float *dn_volume, int Nx, int Ny, int Nz, float n0, int slab,
                    float *nref_out_host, void *stream);

/*
 * bb_nref_from_dn_static -- the same n_ref[j] (reading A3; same arithmetic, results
 * equal to bb_nref_from_dn's to one float32 ulp) for callers that must not allocate.  bb_nref_from_dn
 * grows a device workspace with cudaFree + cudaMalloc and fills a host vector.  That is wrong for a
 * pipeline that works out n_ref of the next volume on a side stream while a propagation runs (cudaMalloc
 * and cudaFree wait for the whole device, so the propagation stalls), and for a process whose own
 * allocator already holds nearly all device memory (a raw cudaMalloc then fails).  This entry point makes
 * no cudaMalloc / cudaFree / host allocation and no copy: two kernel launches on `stream`, returning
 * without waiting.
 *   dn_volume   DEVICE float[Nz][Ny][Nx] (any Nx, Ny >= 1)
 *   nref_out    DEVICE float[Nz], caller-owned -- not the HOST array of bb_nref_from_dn; copy it to the
 *               host yourself (bb_opts.nref wants it there), into memory you already own
 * Scratch: Nz x 16 doubles of per-slice partial sums in a fixed array inside the library's device
 * image, BB_STATIC_MAX_NZ slices deep = 512 KiB, resident on every GPU whose context loads this library
 * until the process exits.  Nz > BB_STATIC_MAX_NZ returns BB_ERR_INVALID_ARG (message names the limit);
 * split deeper volumes along z on slab boundaries, or use bb_nref_from_dn.
 * First call on each device: looks up the array's device address (cudaGetSymbolAddress, once per device,
 * cached; that device must be current, as for every call here).  Make that first call outside any stream
 * capture.
 * All calls on one device share the array.  Nothing needs to start at zero: each call overwrites every
 * element it later reads, so the previous call's contents never show.  But two calls that can overlap on
 * the GPU (different streams without an event between them) race on it and both results are garbage; on
 * one stream they are ordered and safe.
 */
#define BB_STATIC_MAX_NZ 4096
int bb_nref_from_dn_static(const float *dn_volume, int Nx, int Ny, int Nz, float n0, int slab,
                           float *nref_out, void *stream);
int bb_static_max_nz(void);             /* BB_STATIC_MAX_NZ of the loaded library */

/*
 * bb_multiplex_psf -- north_star: "bb_multiplex_psf(emitter_positions, NA, ...)"; PAPER.md
 * line 21 ("sets of 100s to 1000s of mutually independent ... PSFs ... within single, highly
 * multiplexed simulations") and line 29 ("multiplexed diffraction-limited point-sources").
 * Readings A12-A14:
 *   P[q][p]  = 1 if kx^2 + ky^2 <= (k0 NA)^2 else 0
 *   U0[q][p] = P * sum_e a_e exp(i (phi_e - kx X_e - ky Y_e)),  X_e = x_e + (Nx/2) dx, Y_e likewise
 *   field    = IFFT2(U0) * (Nx Ny / sum P)          (an on-grid unit emitter has field 1 at its pixel)
 *   emitter_positions  float[M][2] (x, y) in um, origin at pixel (Nx/2, Ny/2)
 *   emitter_phase      float[M] rad, or NULL = 0;   emitter_amp  float[M], or NULL = 1
 *   field_out          float pairs [Ny][Nx]
 */
int bb_multiplex_psf(const float *emitter_positions, const float *emitter_phase,
                     const float *emitter_amp, int M, float NA,
                     int Nx, int Ny, float dx, float lambda, void *field_out, void *stream);

/*
 * bb_multiplex_annular -- the same with an annular pupil NA_inner <= |k| / k0 <= NA: every "emitter"
 * is a Bessel-beam focus (a thin annulus gives J0(k0 NA r)), a row of them a Bessel lattice
 * ("Bessel lattices"; line 17, Fig. 1d).  NA_inner = 0 is bb_multiplex_psf.
 */
int bb_multiplex_annular(const float *emitter_positions, const float *emitter_phase,
                         const float *emitter_amp, int M, float NA_inner, float NA,
                         int Nx, int Ny, float dx, float lambda, void *field_out, void *stream);

/*
 * bb_lightsheet -- PAPER.md line 29 ("a cylindrical sheet of light is propagated"), BASELINE.json
 * configs[1] ("cylindrically focused Gaussian sheet (NA 0.1 in y, flat in x)"): the input-plane field of
 * a sheet whose waist exp(-y^2 / w0^2), w0 = lambda / (pi NA), lies z_focus behind the input plane in
 * the medium n0 -- the waist propagated back by z_focus with the exact propagator (evanescent ky
 * cut), uniform in x, y_i = (i - Ny/2) dx.  field_out: float pairs [Ny][Nx].
 */
int bb_lightsheet(int Nx, int Ny, float dx, float lambda, float n0, float NA, float z_focus,
                  void *field_out, void *stream);

/*
 * bb_refocus -- PAPER.md lines 29-31 ("propagating light from multiplexed diffraction-limited
 * point-sources orthogonally through an idealized, refocusing lens towards the camera"): free-space
 * propagation of `batch` fields over the SIGNED distance dz in a homogeneous medium of index n,
 *     U = FFT2(u);  U *= (s > 0) ? exp(i dz sqrt(s)) : 0;  u = IFFT2(U),   s = (k0 n)^2 - kx^2 - ky^2
 * in place (dz < 0 refocuses the exit field of a sample onto the emitter plane; dz = 0 only cuts the
 * evanescent modes).  A through-focus stack is bb_propagate_ex with BB_HOMOGENEOUS.
 */
int bb_refocus(void *field, int Nx, int Ny, int batch, float dx, float dz, float lambda, float n, void *stream);

/*
 * bb_extract_tiles -- PAPER.md line 31 ("quasi-continuum of spatially-dependent, volumetric PSFs"): the
 * T x T window around every emitter in every plane of a stack.  src: [Nplanes][Ny][Nx] of `elem` floats
 * per pixel (1: intensity, 2: complex field); emitter e has centre pixel (floor(x_e / dx + 0.5) + Nx/2,
 * floor(y_e / dx + 0.5) + Ny/2) (coordinates as in bb_multiplex_psf) and window [c - T/2, c - T/2 + T) per
 * axis, periodic.  tiles_out: [M][Nplanes][T][T] of `elem` floats.
 */
int bb_extract_tiles(const void *src, int elem, int Nx, int Ny, int Nplanes, const float *emitter_positions,
                     int M, float dx, int T, void *tiles_out, void *stream);

/*
 * bb_image_formation -- PAPER.md line 31 ("Convolving the exhaustively sampled set of spatially-varying PSFs
 * with the fluorescent object"; line 17, Fig. 1c), reading A18: the PSF is piecewise constant over
 * the cells of the emitter grid.  source S = fluorophore density x excitation intensity, float [Ny][Nx]; a source
 * pixel r' radiates with the intensity tile of the emitter nearest to it (periodic distance, lowest index on ties):
 *     image[r] = sum_{r'} S[r'] psf[e(r')][r - r' + T/2]        (r' over the T x T neighbourhood, periodic)
 * psf_tiles: float [M][T][T] (e.g. from bb_extract_tiles, T <= 96), image_out: float [Ny][Nx].  Uses the
 * library's workspace: calls on one device must not overlap.
 */
int bb_image_formation(const float *source, int Nx, int Ny, const float *emitter_positions, int M, float dx,
                       const float *psf_tiles, int T, float *image_out, void *stream);

/*
 * Building blocks, exported so that each can be checked against the oracle on its own.
 * bb_fft2: in-place 2-D DFT of `batch` fields; sign = -1 forward (unnormalised), +1 inverse
 * (divides by Nx Ny).  bb_propagator_table: the table the propagator multiply uses,
 * H[q][p] = (s > 0 ? exp(i dz sqrt(s)) : 0) / (Nx Ny) as float pairs [Ny][Nx] (the 1/(Nx Ny) of
 * the inverse transform is folded in; a power of two, so exact).
 */
int bb_fft2(void *field, int Nx, int Ny, int batch, int sign, void *stream);
int bb_propagator_table(int Nx, int Ny, float dx, float dz, float lambda, float nref,
                        void *table_out, void *stream);

const char *bb_last_error(void);        /* thread-local; "" if none */
int bb_version(void);                   /* 100 * major + minor */
void bb_shutdown(void);                 /* frees cached plans, tables and workspace (synchronises) */
unsigned long long bb_launch_count(void); /* kernels launched by this library since load */
const char *bb_last_kernel(void);        /* name of the BPM kernel the last propagation launched ("" if none yet) */
int bb_device_status(void);             /* synchronises the device; BB_ERR_INTERNAL if a device-side
                                           watchdog tripped since the last call, else BB_OK */


/*
 * Measurement support: the roofline denominators MEASURED_PEAKS.json does
 * not hold.  Synchronous; allocate and free their own buffers; not used by the BPM path.
 * bb_probe_l2_bandwidth: GB/s over a `bytes`-sized buffer that stays in L2 (mode 0: copy, counts
 * bytes read + written; mode 1: read only).  bb_probe_fp32: TFLOP/s of dependent-free FMA chains,
 * packed = 0 scalar FFMA, 1 = FFMA2 (fma.rn.f32x2); packed = 2: the library's own butterflies of one
 * phase of a 1024-point line (radix-16, twiddles, radix-16, radix-4 class step, pointwise multiply, and
 * back) run from registers with no memory access at the occupancy of the 16-point-thread kernel, credited
 * with SURVEY 8d's 120 flop per point and phase -- the FP32 ceiling of this instruction mix, against which
 * the kernel's algorithmic flop rate can be held.
 */
int bb_probe_l2_bandwidth(unsigned long long bytes, int iters, int mode, double *gb_per_s);
int bb_probe_fp32(int iters, int packed, double *tflops);
/*
 * bb_probe_trace: timeline of the persistent kernel, for profiling only.  device_buf is a DEVICE
 * long long[phases][SM count][6] or NULL to switch tracing off.  While set, every propagation of at
 * most (phases - 1) / 2 steps records, per phase and CTA (index = blockIdx.x, which must stay below the
 * SM count), the SM clock at phase start, work done, barrier arrived, pointwise factors staged and
 * barrier released, and the global nanosecond timer at release.  Traced: the 16- and 8-point-thread
 * grid kernels (sides 256 .. 2048; grid <= SM count, single fields and batches) and the cluster kernel
 * for a SINGLE field (a 128-point side; its grid is the cluster size, 8 or 16 CTAs).  A batch on the
 * cluster kernel launches cluster size x B CTAs, more than the buffer has rows for, and is not traced.
 */
int bb_probe_trace(long long *device_buf, int phases);

#ifdef __cplusplus
}
#endif
#endif /* BIOBEAM_B200_BB_H */
