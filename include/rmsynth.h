/*
 * rmsynth.h -- C-ABI boundary of librmsynth.so: Faraday rotation-measure synthesis on one
 * NVIDIA B200 (sm_100a).  Operation (arxiv 1810.06250; P:L<n> = line n of PAPER.md):
 *
 *   F(phi_k) = K sum_i w_i (Q_i + iU_i) exp(-2i phi_k (lambda_i^2 - lambda_0^2))    Eq. 11
 *   FQ = K sum_i w_i (Q_i cos th_ik + U_i sin th_ik)                                Eq. 15/18
 *   FU = K sum_i w_i (U_i cos th_ik - Q_i sin th_ik)                                Eq. 16/19
 *   th_ik = 2 phi_k (lambda_i^2 - lambda_0^2),  K = 1/sum w_i (Eq. 13),
 *   lambda_i^2 = (c/nu_i)^2,  lambda_0^2 = K sum w_i lambda_i^2 (weighted-mean reading)
 *   R(phi) = K sum_i w_i exp(-2i phi (lambda_i^2 - lambda_0^2))                     Eq. 12
 *
 * for every line of sight (pixel) of a Q/U cube.  The weights multiply every term (they are
 * the W(lambda^2) of Eq. 7).  All entry points return an rmsynth_status; nothing
 * throws or aborts.  The library never falls back to the CPU: without a usable sm_100
 * device every compute call fails with RMSYNTH_EUNSUPPORTED / RMSYNTH_ECUDA.
 *
 * Ownership: the caller owns every buffer it passes.  A plan owns only what it allocated
 * and is immutable after creation.  Inputs are never modified.  Q/U must not alias FQ/FU.
 * Cube pointers need 4-byte alignment only (16-byte alignment enables the TMA fast paths).
 */
#ifndef RMSYNTH_H
#define RMSYNTH_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rmsynth_plan rmsynth_plan; /* opaque */

typedef enum {
    RMSYNTH_OK = 0,
    RMSYNTH_EINVAL = 1,       /* bad argument (see each call)                          */
    RMSYNTH_ENOMEM = 2,       /* host or device allocation failed                      */
    RMSYNTH_ECUDA = 3,        /* a CUDA call failed; text in rmsynth_last_error()      */
    RMSYNTH_EUNSUPPORTED = 4  /* device is not compute capability 10.x, or the scheme   */
                              /* cannot serve this shape/alignment                      */
} rmsynth_status;

/* layout = one RMSYNTH_IN_* | one RMSYNTH_OUT_*.  p = y*NX + x is the pixel index.
 *   IN_LOS_MAJOR   Q[p*n_chan + i]   (frequency fastest; cuFFS "rotated" cubes)
 *   IN_FREQ_MAJOR  Q[i*n_pix + p]    (FITS order, frequency slowest)
 *   OUT_LOS_MAJOR  F[p*n_phi + k]    (phi fastest: the paper's output order)
 *   OUT_PHI_MAJOR  F[k*n_pix + p]    (phi as third/slowest axis: after the paper's
 *                                     "derotation", Table 1 note (c))           */
enum {
    RMSYNTH_IN_LOS_MAJOR = 0,
    RMSYNTH_IN_FREQ_MAJOR = 1,
    RMSYNTH_OUT_LOS_MAJOR = 0,
    RMSYNTH_OUT_PHI_MAJOR = 2
};

/* Arithmetic scheme of the contraction (rows a5/a9 of the scope table).              */
enum {
    RMSYNTH_SCHEME_AUTO = 0,        /* F16X3; TF32X3 when the positive weights span more */
                                    /* than 2^18 or n_chan < 384 (rmsynth_plan_info tells) */
    RMSYNTH_SCHEME_TF32X3 = 1,      /* tcgen05 tensor cores, split-precision 3xTF32,     */
                                    /* FP32 accumulate in TMEM                           */
    RMSYNTH_SCHEME_F16X3 = 2,       /* tcgen05 tensor cores, block-scaled FP16 hi/lo split    */
                                    /* (3 products at twice the TF32 rate), FP32 accumulate.  */
                                    /* Each 32-channel chunk of a line of sight is scaled by  */
                                    /* its own maximum, floored at 2^(eB - 112) ~ 1e-27 (eB = */
                                    /* the plan's power-of-two scale of K w, 23-24 for a few  */
                                    /* hundred channels): a smaller chunk is scaled by the    */
                                    /* floor's power and loses one bit per factor two under   */
                                    /* it (parity-grade to ~1e-28, plain FP16 accuracy below, */
                                    /* never flushed to zero); the other schemes have no floor */
    RMSYNTH_SCHEME_FP32_TABLE = 3,  /* CUDA cores, FP32 FMA, reads the plan's cos/sin    */
    RMSYNTH_SCHEME_FP32_SINCOS = 4  /* CUDA cores, sincos on the fly, one (pixel,phi)    */
                                    /* per thread -- the paper's kernel shape    */
};

typedef struct {
    int struct_size;   /* sizeof(rmsynth_options); lets the struct grow                   */
    int scheme;        /* RMSYNTH_SCHEME_*                                                */
    int lambda0_mode;  /* 0 weighted mean (default), 1 plain mean, 2 explicit lambda0_sq  */
    int device;        /* CUDA device ordinal, -1 = the caller's current device.  Every call  */
                       /* on the plan runs on this device and restores the caller's current   */
                       /* device before returning; streams passed in must belong to it.       */
    double lambda0_sq; /* used when lambda0_mode == 2 (0 reproduces Fig. 1 left)  */
    long long host_chunk_pixels; /* pixels per chunk of rmsynth_execute_host / _stream (rounded */
                       /* to a multiple of 4); 0 = automatic (~256 MB of device buffers per slot) */
} rmsynth_options;

/* Build a plan: lambda_i^2, K, lambda_0^2 on the host in FP64 ("computed only once"),
 * then on the device the FP64 sincos phase matrix K w_i cos/sin th_ik, rounded to the
 * scheme's operand format, and R(phi) on the plan grid (Eq. 12).
 *   nu_hz[n_chan]  HOST, channel centre frequencies in Hz, finite and > 0
 *   w[n_chan]      HOST, weights >= 0, finite, sum > 0; NULL = all ones
 *   phi[n_phi]     HOST, Faraday depths in rad m^-2, finite, any order or spacing
 *   opt            NULL = defaults
 * Host arrays are copied.  Synchronous.  EINVAL on n_chan < 1, n_phi < 1, NULL plan/nu/phi,
 * bad values, unknown scheme/mode. */
rmsynth_status rmsynth_plan_create(rmsynth_plan **plan, const double *nu_hz, const double *w,
                                   int n_chan, const double *phi, int n_phi,
                                   const rmsynth_options *opt);
rmsynth_status rmsynth_plan_destroy(rmsynth_plan *plan); /* NULL is a no-op */

/* Scalars of the plan (any out pointer may be NULL). */
rmsynth_status rmsynth_plan_info(const rmsynth_plan *plan, double *lambda0_sq, double *K,
                                 int *n_chan, int *n_phi, int *scheme);

/* Copy the plan's FP32-rounded phase matrix to HOST arrays cos_kw[n_chan*n_phi],
 * sin_kw[n_chan*n_phi], index i*n_phi + k, value K w_i cos/sin th_ik (either may be NULL).
 * For tests of row a2.  Synchronous. */
rmsynth_status rmsynth_plan_phase_matrix(const rmsynth_plan *plan, float *cos_kw, float *sin_kw);

/* Eqs. 15-16 for n_pix lines of sight.
 *   Q, U    DEVICE, n_pix*n_chan floats each, input layout per `layout`
 *   FQ, FU  DEVICE, n_pix*n_phi floats each, output layout per `layout`
 *   stream  a cudaStream_t (NULL = default stream).  The call only enqueues work and never
 *           synchronises.  Per-stream workspace (peak records, check-in counters) is allocated
 *           on the first call of a (stream, size) and only ever grows; outgrown buffers stay
 *           alive until rmsynth_plan_destroy, so a CUDA graph captured from an earlier call
 *           remains valid.  Inside a stream capture the workspace cannot grow (EINVAL): run
 *           the shape once on that stream before capturing.
 * n_pix == 0 is a successful no-op.  EINVAL: n_pix < 0, NULL Q/U/FQ/FU, unknown layout bits.
 * Non-finite samples propagate to the outputs of their pixel (its cubes are NaN, its maps NaN
 * with peak_index -1).  Channels with w_i = 0 are REMOVED (reading A13): every scheme ignores
 * their samples altogether, non-finite or not -- a NaN-blanked flagged plane does no harm. */
rmsynth_status rmsynth_execute(const rmsynth_plan *plan, const float *Q, const float *U,
                               long long n_pix, int layout, float *FQ, float *FU, void *stream);

/* rmsynth_execute plus the fused peak epilogue (Eq. 14, Eq. 17):
 * per pixel k* = argmax_k |F_k| (lowest k on ties, |F| compared in FP32), three-point
 * parabolic refinement of (phi, |F|) on the plan's grid (none at the grid edges or when the
 * three points are not strictly concave), and
 *   pa_lambda0 = 0.5 atan2(FU_k*, FQ_k*)                      angle at lambda_0^2
 *   pa_zero    = pa_lambda0 - peak_phi * lambda_0^2           wrapped to [-pi/2, pi/2)
 * FQ/FU may both be NULL (maps only).  Each map is DEVICE [n_pix] and may be NULL;
 * peak_index (int) receives k*. */
rmsynth_status rmsynth_execute_peaks(const rmsynth_plan *plan, const float *Q, const float *U,
                                     long long n_pix, int layout, float *FQ, float *FU,
                                     float *peak_amp, float *peak_phi, float *pa_lambda0,
                                     float *pa_zero, int *peak_index, void *stream);

/* Every output of the path in one call (NEXT-1 of the scope table: the paper's third cube).
 * Any subset may be requested; at least one pointer must be non-NULL.
 *   FQ, FU     DEVICE cubes, both or neither
 *   F_abs      DEVICE cube |F| = sqrt(FQ^2 + FU^2) (Eq. 17; cuFFS writes it as a third
 *              cube), same layout as FQ/FU; formed in FP32 from the FP32 FQ, FU
 *   peak_*     as in rmsynth_execute_peaks
 * With FQ = FU = F_abs = NULL no cube is written at all ("maps only": half of the HBM traffic). */
typedef struct {
    int struct_size;                 /* sizeof(rmsynth_outputs) */
    float *FQ, *FU, *F_abs;
    float *peak_amp, *peak_phi, *pa_lambda0, *pa_zero;
    int *peak_index;
} rmsynth_outputs;
rmsynth_status rmsynth_execute_ex(const rmsynth_plan *plan, const float *Q, const float *U,
                                  long long n_pix, int layout, const rmsynth_outputs *out,
                                  void *stream);

/* Same as rmsynth_execute_peaks with every cube/map pointer in HOST memory (pinned memory
 * gives full PCIe rate): the library streams pixel chunks host->device->host through three
 * sets of device buffers, with H2D of chunk i+1, the kernels of chunk i and D2H of chunk i-1
 * overlapping, and returns when the outputs are complete.  Chunk size: the plan's
 * host_chunk_pixels.  Each datum crosses the bus once (the paper's transfer rule,
 * P:L200-210).  Synchronous. */
rmsynth_status rmsynth_execute_host(const rmsynth_plan *plan, const float *Q, const float *U,
                                    long long n_pix, int layout, float *FQ, float *FU,
                                    float *peak_amp, float *peak_phi, float *pa_lambda0,
                                    float *pa_zero, int *peak_index);

/* Out-of-core form of rmsynth_execute_host for cubes that do not fit in host memory (the paper's LOFAR_HR
 * shape is 110 GB in and > 1 TB out): the library owns three sets of pinned staging buffers and
 * calls back on the caller's thread, in chunk order,
 *   n = fill(user, i, Q, U, max_pix)   write chunk i (n <= max_pix lines of sight, n = 0 ends the run) into
 *                                      the HOST staging buffers Q, U: compact, input layout per `layout`,
 *                                      i.e. Q[c*n + p] (IN_FREQ_MAJOR) or Q[p*n_chan + c] (IN_LOS_MAJOR)
 *   drain(user, i, n, out)             chunk i is complete: out->FQ/FU (compact [k*n + p] or [p*n_phi + k],
 *                                      if RMSYNTH_WANT_CUBES) and out->peak_* (if RMSYNTH_WANT_MAPS) point
 *                                      into HOST staging that is valid only during the call
 * while chunks i+1, i+2 are in flight (H2D, kernels and D2H overlap; each datum crosses the bus once,
 * P:L200-210).  max_pix is the plan's host_chunk_pixels (or the automatic size).  *n_pix_done (may be
 * NULL) receives the number of lines of sight processed.  Synchronous; EINVAL on NULL callbacks, unknown
 * flags, or a fill() that returns more than max_pix. */
enum { RMSYNTH_WANT_CUBES = 1, RMSYNTH_WANT_MAPS = 2 };
typedef long long (*rmsynth_fill_fn)(void *user, long long chunk_index, float *Q, float *U, long long max_pix);
typedef void (*rmsynth_drain_fn)(void *user, long long chunk_index, long long n_pix, const rmsynth_outputs *out);
rmsynth_status rmsynth_execute_stream(const rmsynth_plan *plan, int layout, int outputs,
                                      rmsynth_fill_fn fill, rmsynth_drain_fn drain, void *user,
                                      long long *n_pix_done);

/* Approximate fast path: Eqs. 15-16 by FFT instead of DFT (the paper's outlook).  Channels are not uniform
 * in lambda^2, so this is a non-uniform FFT per line of sight (readings F1-F6 of DESIGN.md): samples are spread
 * onto a fine uniform lambda^2 grid of M = 2^ceil(log2(oversampling * n_phi)) points with a Kaiser-Bessel window of
 * `window` points, transformed by an M-point FFT and deapodised.  Same arguments and layouts as rmsynth_execute.
 * It is an APPROXIMATION: max |F_fft - F| <= eps(window, oversampling) * T_p per line of sight, with
 * eps ~ 2e-6 for the defaults (window 6, oversampling 2; measured 1.3e-6 in FP64 plus ~1e-6 of FP32 FFT rounding)
 * and falling about a decade per unit of `window`.  Needs a uniform depth grid (else EUNSUPPORTED).
 * params NULL = defaults.  EINVAL: window odd or outside 2..16, oversampling outside [1.25, 8].  Only enqueues,
 * except when (window, oversampling) differ from the plan's last call (tables are rebuilt synchronously). */
typedef struct {
    int struct_size;      /* sizeof(rmsynth_fft_params) */
    int window;           /* Kaiser-Bessel window width W in fine-grid points, even; 0 = 6 */
    float oversampling;   /* sigma; 0 = 2 */
} rmsynth_fft_params;
rmsynth_status rmsynth_execute_fft(const rmsynth_plan *plan, const float *Q, const float *U, long long n_pix,
                                   int layout, float *FQ, float *FU, const rmsynth_fft_params *params,
                                   void *stream);

/* RM-CLEAN per line of sight (the deconvolution the paper names as the use of Eq. 12, footnote 6
 * the paper defines no step of it; the loop is reading C1-C8 of DESIGN.md): Hogbom CLEAN
 * of the complex dirty spectrum F~ = FQ + i FU with the complex RMSF as the beam.
 *   r <- F~, m <- 0; repeat up to max_iter times: k* = lowest index of max |r_k|; stop if |r_k*| < cutoff;
 *   c = gain r_k*; m_k* += c; r_k -= c R(phi_k - phi_k*) for all k.
 *   restored_k = sum_j m_j G(phi_k - phi_j) + r_k, G a real Gaussian of FWHM `fwhm` (<= 0: the FWHM of |R|).
 *   FQ, FU            DEVICE dirty cubes, n_pix*n_phi floats each, laid out per the RMSYNTH_OUT_* bit of `layout`
 *                     (what rmsynth_execute wrote); the RMSYNTH_IN_* bit is ignored
 *   model_*, resid_*  DEVICE output cubes, same layout; rest_* likewise or both NULL
 *   n_iter            DEVICE [n_pix] iterations done per line of sight, or NULL
 * A line of sight holding a non-finite sample is passed through (model 0, residual = restored = input, 0
 * iterations).  Needs a uniform depth grid (else EUNSUPPORTED) of at most 14336 depths.  Only enqueues on
 * `stream`, except the first call of a plan (and a change of fwhm), which builds the beam synchronously.
 * EINVAL: gain outside (0, 1], cutoff < 0, max_iter < 0, NULL cubes. */
typedef struct {
    int struct_size;   /* sizeof(rmsynth_clean_params) */
    float gain;
    float cutoff;      /* absolute, in the units of F */
    int max_iter;
    float fwhm;        /* rad m^-2; <= 0 = FWHM of |R| measured on the plan's grid */
} rmsynth_clean_params;
rmsynth_status rmsynth_rmclean(const rmsynth_plan *plan, const float *FQ, const float *FU, long long n_pix,
                               int layout, const rmsynth_clean_params *params, float *model_q,
                               float *model_u, float *resid_q, float *resid_u, float *rest_q,
                               float *rest_u, int *n_iter, void *stream);

/* Peak maps (Eq. 14, Eq. 17; same rules as rmsynth_execute_peaks) of FQ/FU cubes that are
 * already in device memory -- what rmsynth_execute, rmsynth_execute_fft or rmsynth_rmclean wrote -- through a call
 * that ALLOCATES NOTHING, now or later.  It exists for callers that cannot call cudaMalloc once they are running: a
 * framework whose own pool took the whole device at start-up (a library's late cudaMalloc just fails there), a
 * client under a fixed device-memory cap (MPS / MIG share), a real-time loop that cannot take cudaMalloc's
 * device-wide synchronisation and millisecond latency.  Every other call that produces maps fetches its workspace
 * with cudaMalloc the first time it sees a (stream, size); this one keeps its per-(pixel, depth segment) records in
 * a 32 MiB array inside the library image.
 *   plan        supplies the depth grid, n_phi and lambda_0^2 (allocated when the plan was created, not here)
 *   FQ, FU      DEVICE cubes, laid out per the RMSYNTH_OUT_* bit of `layout` (the RMSYNTH_IN_* bit is ignored)
 *   ld          row pitch in floats: F[k*ld + p] (OUT_PHI_MAJOR, ld >= n_pix) or F[p*ld + k] (OUT_LOS_MAJOR,
 *               ld >= n_phi); 0 = dense.  With a pointer offset it selects a slab of pixels of a larger cube.
 *   peak_*, pa_*  DEVICE [n_pix], any may be NULL, at least one must not be
 * LIMIT: n_pix <= 1 048 576 per call (the records must fit the array); more is EINVAL with a message that says so --
 * split the image into slabs.  Cost: 32 MiB of every GPU on which the library is loaded, held until the process
 * exits, used or not.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, which also makes the driver load
 * the module that holds the array).  Make that call during start-up, before any stream capture begins; later calls
 * only enqueue two kernels on `stream`.  Never synchronises, never calls cudaMalloc / cudaFree.
 * The array is shared by ALL calls on a device, whatever the plan or stream, and is left holding the last call's
 * records.  A call depends on none of that (it overwrites every record it reads), but two calls that may run on the
 * GPU at the same time -- different streams, or different host threads without ordering between them -- race on it
 * and return garbage: keep calls to this entry point on one stream, or order them with events.
 * n_pix == 0 is a successful no-op.  EINVAL: NULL plan or cubes, n_pix < 0 or beyond the limit, unknown layout bits,
 * ld below the dense length, no map requested. */
rmsynth_status rmsynth_peaks_static(const rmsynth_plan *plan, const float *FQ, const float *FU, long long n_pix,
                                    long long ld, int layout, float *peak_amp, float *peak_phi,
                                    float *pa_lambda0, float *pa_zero, int *peak_index, void *stream);

/* R(phi) of Eq. 12 in FP64.  phi_eval HOST [n] or NULL for the plan grid (then n must be
 * n_phi); R_re, R_im HOST [n].  Synchronous. */
rmsynth_status rmsynth_rmsf(const rmsynth_plan *plan, const double *phi_eval, int n,
                            double *R_re, double *R_im);

/* Number of kernels this library has launched in this process (for bench.py's
 * gpu_launches claim); pass reset != 0 to zero the counter after reading. */
long long rmsynth_launch_count(int reset);

const char *rmsynth_strerror(rmsynth_status s);
const char *rmsynth_last_error(void); /* thread-local detail of the last failure */
const char *rmsynth_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RMSYNTH_H */
