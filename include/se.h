/*
 * se.h -- C-ABI of the B200 spectral Ewald library (libse_b200.so).
 *
 * Evaluates the triply periodic Stokeslet sum
 *     u(x_i) = sum_j sum_{p in L Z^3} G(x_i - x_j + p) f_j ,   G(r) = I/|r| + r (x) r/|r|^3
 * (eq. (2.1)) with the Hasimoto split G = G^N + G^F
 * (eq. (2.3), eq. (2.4b)) by the spectral Ewald method
 * (Algorithm 2.1): P2P + P2G + FFT + CNV + IFFT + G2P + SUM, with a
 * Gaussian window over P^3 grid points (reading S4) or the paper's truncated
 * Kaiser-Bessel window in piecewise-polynomial form (eq. (2.8),
 * PAPER.md:421-427; readings S18-S20).  Targets = sources by default: the i = j, p = 0 pair
 * is excluded and the self term -(4 xi/sqrt(pi)) f_i is added (reading S3); a plan may
 * instead carry its own N_t target points (eq. (1.1)/(2.1)).
 * The k = 0 mode is dropped (reading S2); G carries no 1/(8 pi mu).
 *
 * Conventions
 *   - All x, f, u arrays are N x 3, row-major (AoS), in the plan's precision
 *     (double for SE_FP64, float for SE_FP32).
 *   - Unless a function says "host", every pointer is a DEVICE pointer owned by the
 *     caller.  The plan owns all workspace; se_eval allocates nothing, never
 *     synchronises the host, is asynchronous on `stream`, does not modify x or f and
 *     OVERWRITES u.  A plan may be evaluated any number of times with new x, f.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - A plan is bound to the CUDA device current at se_plan_create and is not
 *     thread-safe; every later call on it must be made with that device current
 *     (SE_EINVAL otherwise).
 *   - Every entry point returns a status; nothing aborts or throws.  NaN/Inf inputs give
 *     unspecified values but never out-of-bounds accesses.
 *   - There is no CPU fallback: without a CUDA device se_plan_create returns SE_ECUDA.
 *   - Environment variables read at se_plan_create (experiments and tests only; results do not change beyond
 *     rounding order): SE_GRID_MODE = tile (force the generic gridding kernel; default: the FP64 tensor-core
 *     sweep for fp64 plans with even 4 <= P <= 24 and fp32 plans with even 4 <= P <= 16, else the generic tile kernel),
 *     SE_NCHUNK and SE_NCHUNK_G2P (x-chunks of K3 / K5), SE_OVERLAP = 1 (K2 on a side stream next to the FFT
 *     stages), SE_FFT_MODE = 3d (se_eval with the 3-D transforms and the stand-alone K4 instead of the fused path, see
 *     the stages below) or cufft2d (fused path with cuFFT's 2-D transforms instead of the library's own), SE_XF_BW = n (block shape of the fused kernel: n lanes per column, instead of timing the
 *     candidates at plan creation).
 */
#ifndef SE_B200_H
#define SE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct se_plan se_plan;                      /* opaque, owned by the library */

typedef enum { SE_FP64 = 0, SE_FP32 = 1 } se_precision;

/* Window of the P2G / G2P steps.
 *   SE_WINDOW_GAUSSIAN       w(r) = (a/pi)^{3/2} e^{-a r^2}, a = 2 xi^2/eta, eta = (P h xi/m)^2, m = 0.95 sqrt(pi P)
 *                            (the "classic" window the paper names at PAPER.md:103; reading S4); deconvolved with
 *                            w_hat(k) = e^{-eta k^2/8 xi^2}.
 *   SE_WINDOW_KAISER_BESSEL  w0(r) = I0(beta sqrt(1 - r^2/a_w^2))/I0(beta), |r| < a_w, beta = 2.5 P, a_w = P h/2
 *                            (eq. (2.8)), evaluated as one polynomial of degree nu = min(P + 3, 13) per
 *                            bin of width h by Horner's rule (reading S19), deconvolved with its
 *                            closed-form transform (reading S20). */
typedef enum { SE_WINDOW_GAUSSIAN = 0, SE_WINDOW_KAISER_BESSEL = 1 } se_window;

typedef enum {
    SE_OK = 0,
    SE_EINVAL = 1,   /* bad argument (see se_plan_create) or null pointer            */
    SE_ENOMEM = 2,   /* device or host allocation failed                             */
    SE_ECUDA = 3,    /* a CUDA runtime call or kernel launch failed / no device      */
    SE_ECUFFT = 4,   /* a cuFFT call failed                                          */
    SE_ELIMIT = 5    /* a size beyond the fixed capacity of an entry point that allocates nothing (se_scale_noalloc) */
} se_status;

/* Stages of Algorithm 2.1 as this library runs them. */
enum {
    SE_STAGE_SORT = 0,   /* K1: wrap, bin, counting sort (near cells + grid bins) */
    SE_STAGE_P2P = 1,    /* K2: near field u^N, eq. (2.2)/(2.3)  */
    SE_STAGE_P2G = 2,    /* K3: Gaussian spreading, eq. (2.5)  */
    SE_STAGE_FFT = 3,    /* cuFFT R2C, 3 components     */
    SE_STAGE_SCALE = 4,  /* K4: CNV, eq. (2.6) with (2.4b)  */
    SE_STAGE_IFFT = 5,   /* cuFFT C2R, 3 components     */
    SE_STAGE_G2P = 6,    /* K5: gather, eq. (2.7)  */
    SE_STAGE_SUM = 7,    /* K6: u = u^N + u^F - (4 xi/sqrt(pi)) f, user order    */
    SE_NSTAGES = 8
};
/* se_eval_stage runs stages 3-5 as written above (3-D transforms, spectrum readable in between).  se_eval, se_eval_targets
 * and se_eval_host run them FUSED when se_info.fft_fused is 1 (M has no prime factor above 7 and 3 x 4 (fp32: 3 x 8) columns
 * of M modes fit in shared memory; SE_FFT_MODE=3d at plan creation switches it off): stage 3 = cuFFT 2-D R2C over (y, z) of
 * every x-plane, stage 4 = ONE kernel that transforms over x, applies K4 and transforms back over x (a 3-D transform is the
 * 2-D transforms followed by 1-D transforms over x, and K4 is diagonal in k), stage 5 = cuFFT 2-D C2R; with
 * se_info.fft_planes_own the 2-D transforms are the library's own kernels as well (no cuFFT call in se_eval).  The result H~ is the
 * same up to rounding; SE_BUF_SPEC then holds the 2-D spectra of the planes (with fft_planes_own: their second axis in the
 * digit-reversed order of the library's transform over y -- an internal order, read the spectrum through the staged interface
 * instead), and se_stage_ms reports the three parts under the same names. */

/* Internal buffers visible to tests and the benchmark through se_buffer_read/write. */
enum {
    SE_BUF_UN = 0,        /* u^N, N x 3 reals, NEAR-sorted order                                   */
    SE_BUF_UF = 1,        /* u^F, N x 3 reals, GRID-sorted order                                   */
    SE_BUF_GRID = 2,      /* real grid H (after P2G) / H~ (after IFFT): 3 x M x M x M reals, z fastest */
    SE_BUF_SPEC = 3,      /* spectrum: 3 x M x M x (M/2+1) complex (re,im) reals, halved axis last  */
    SE_BUF_PERM_NEAR = 4, /* int32[N]: sorted position -> user index, near-cell order              */
    SE_BUF_PERM_GRID = 5, /* int32[N]: sorted position -> user index, grid-bin order               */
    SE_BUF_CELL_START = 6,/* int32[ncell^3 + 1]: CSR offsets of the near cells                     */
    SE_BUF_BIN_START = 7, /* int32[nbins_total + 1]: CSR offsets of the grid bins.  grid_mode 0: bins of 8^3 grid
                             cells, key (bx, by, bz); grid_mode 2: key (anchor plane a_x, a_z / 8, a_y)     */
    SE_NBUFS = 8
};
/* For plans with their own targets (Nt > 0) SE_BUF_UN / SE_BUF_UF hold Nt x 3 reals in the TARGETS' near / grid
 * order and SE_BUF_PERM_* / SE_BUF_*_START describe the SOURCES; add SE_BUF_TARGETS to a PERM / START id to read
 * the target set's array instead. */
enum { SE_BUF_TARGETS = 16 };

typedef struct {
    int64_t N;
    int M, P, precision;
    double L, xi, rc;
    double h;            /* L / M                                                        */
    double m;            /* Gaussian shape parameter, 0.95 sqrt(pi P)      (reading S4)  */
    double eta;          /* (P h xi / m)^2                                               */
    double a;            /* window exponent 2 xi^2 / eta : w(r) = c_w exp(-a r^2)        */
    double cw;           /* (a/pi)^{3/2}                                                 */
    int ncell;           /* near cells per dimension, floor(L/rc)          (reading S7)  */
    int nbin;            /* grid bins per dimension: ceil(M/8)                          */
    int grid_mode;       /* gridding kernels: 0 = tile-stationary (any even P), 2 = FP64 tensor-core sweep */
    int nbins_total;     /* entries of SE_BUF_BIN_START minus 1: nbin^3 (mode 0), M * nbin * M (mode 2)    */
    int nchunk;          /* tensor-core sweep: chunks along x (P2G)                      */
    int64_t nmodes;      /* M * M * (M/2+1) stored modes per component                   */
    size_t workspace_bytes; /* device memory owned by the plan (incl. cuFFT work area)   */
    int64_t Nt;          /* targets (0: the targets are the sources)                     */
    int window;          /* se_window                                                    */
    int nu;              /* Kaiser-Bessel: degree of the piecewise polynomial            */
    double kb_beta;      /* Kaiser-Bessel: beta = 2.5 P ; a_w = P h / 2                  */
    int Mx, px0;         /* planes of the plan's grid along x (M unless a slab plan) and global index of plane 0 */
    int fft_fused;       /* 1: se_eval / se_eval_targets / se_eval_host run the transform over x, K4 and the inverse transform
                            over x as one kernel between cuFFT 2-D transforms of the x-planes (see SE_STAGE_SCALE below) */
    int fft_threads;     /* fused plans: threads per block of that kernel (timed once at plan creation; SE_XF_BW = lanes per
                            column fixes it instead); 0 otherwise */
    int fft_planes_own;  /* fused plans: 1 if the 2-D transforms of the x-planes are the library's own kernels (a real-to-complex
                            pass over z, a pass over y that leaves k_y in digit-reversed order for the fused kernel), 0 if
                            cuFFT's (SE_FFT_MODE = cufft2d, or shapes the own kernels do not cover) */
} se_info;

/* Everything se_plan_create takes, plus the window and an optional separate target count. */
typedef struct {
    int64_t N;           /* source points                                                */
    int64_t Nt;          /* target points; 0 = the targets are the sources (self term added, se_eval);
                            > 0 = own targets (no self term, se_eval_targets)            */
    double L, xi, rc;
    int M, P;
    int precision;       /* se_precision */
    int window;          /* se_window    */
    int Mx;              /* 0: the plan's grid is the whole M^3 grid.  > 0: SLAB plan ("equisized slabs along the
                            periodic spatial dimension"): the plan's grid holds Mx x M x M points, local plane l being global
                            plane (px0 + l) mod M; every SOURCE / TARGET handed to it must have its window inside that
                            range, i.e. floor(x/h) - (P/2 - 1) - px0 (mod M) in [0, Mx - P].  A slab plan runs the stages
                            SORT, P2P, P2G, G2P, SUM; FFT / SCALE / IFFT return SE_EINVAL (the transform of the assembled
                            grid belongs to a whole-grid plan).  Needs a (P, precision) of the tensor-core gridding
                            kernels and Mx >= P rounded up to a multiple of 8. */
    int px0;             /* slab plans: global index of local plane 0, in [0, M)            */
    int64_t Nown;        /* slab plans with targets (Nt > 0): 0, or Nown == Nt: the targets ARE the first Nt sources (the
                            points this slab owns; the sources behind them are ghost copies of the neighbours' points, needed by
                            P2P only, "exchanging ghost source points").  Then K3 spreads only the first Nown
                            sources and SE_STAGE_SUM adds the self term with f[0 .. Nt).  */
} se_plan_desc;

/*
 * Create a plan.  N particles in the periodic cube [0,L)^3, split parameter xi,
 * near-field cutoff rc, M^3 Fourier grid, Gaussian support P grid points per dimension.
 * SE_EINVAL if: out == NULL, N < 1, N >= 2^31, L <= 0, xi <= 0, rc <= 0, M < 2, M odd,
 * M > 4096, P < 2, P odd, P > 32, P > M, floor(L/rc) < 3 (the 27-cell stencil would
 * alias, reading S7), or an unknown precision.  On any failure *out is NULL.
 */
se_status se_plan_create(se_plan **out, int64_t N, double L, double xi, double rc,
                         int M, int P, se_precision prec);

/* Same with a descriptor: Gaussian or Kaiser-Bessel window (for which cw = 1 and eta, m, a are reported as 0),
 * optional separate targets.  Kaiser-Bessel needs 2 <= P <= 16 as well. */
se_status se_plan_create_ex(se_plan **out, const se_plan_desc *desc);

/* Full evaluation, all stages; x, f, u are device pointers (N x 3).  Plans with Nt = 0 only. */
se_status se_eval(se_plan *p, const void *x, const void *f, void *u, void *stream);

/*
 * Plans with Nt > 0: u_t(x_i) = sum_j sum_p G(x_i - y_j + p) f_j at the Nt targets xt (Nt x 3, device) from the
 * N sources xs, f (N x 3, device); ut is Nt x 3 (eq. (1.1)).  No self term.  A target that coincides
 * with a source skips that pair in the near sum only (r = 0 is never evaluated); its smooth far part
 * stays.  The per-stage hook se_eval_stage takes xt through se_set_targets.
 */
se_status se_eval_targets(se_plan *p, const void *xs, const void *f, const void *xt, void *ut, void *stream);

/*
 * Same, with HOST buffers (pinned or pageable): copies x, f host->device into plan-owned
 * staging buffers (allocated at plan creation like all other workspace), runs se_eval, copies u
 * device->host, all asynchronously on `stream` (the caller synchronises the stream before
 * reading u_host).  Plans with Nt = 0 only.
 */
se_status se_eval_host(se_plan *p, const void *x_host, const void *f_host, void *u_host,
                       void *stream);

se_status se_plan_destroy(se_plan *p);            /* NULL is accepted and ignored */
const char *se_strerror(se_status s);
se_status se_plan_info(const se_plan *p, se_info *out);

/* ---- per-stage hooks: used only by the tests and the benchmark ------------------------ */

/*
 * Run ONE stage on the plan's internal state.  SE_STAGE_SORT needs x and f (device);
 * SE_STAGE_SUM needs f (device, user order) and writes u (device, user order); the other
 * stages take NULL for x, f, u and read/write the plan's buffers (SE_BUF_*).
 * Stages must be run in the order of the enum after a SORT of the same inputs, except
 * that SCALE and G2P may also be run on buffers filled with se_buffer_write.
 */
se_status se_eval_stage(se_plan *p, int stage, const void *x, const void *f, void *u,
                        void *stream);

/* Plans with Nt > 0: the target positions (Nt x 3, device) the next se_eval_stage(SE_STAGE_SORT) bins. */
se_status se_set_targets(se_plan *p, const void *xt);

/* Copy an internal buffer to / from caller DEVICE memory (`bytes` must equal its size,
 * obtainable with dst == NULL: *size_out is set and nothing is copied). */
se_status se_buffer_read(se_plan *p, int which, void *dst, size_t bytes, size_t *size_out,
                         void *stream);
se_status se_buffer_write(se_plan *p, int which, const void *src, size_t bytes, void *stream);

/*
 * Stage timing.  se_set_profiling(p, 1) makes every later se_eval record CUDA events
 * around each stage (no host synchronisation inside se_eval); se_stage_ms synchronises on
 * those events and returns the per-stage milliseconds of the LAST profiled se_eval.
 */
se_status se_set_profiling(se_plan *p, int on);
se_status se_stage_ms(se_plan *p, float ms[SE_NSTAGES]);

/* Number of this library's own kernel launches issued by the last se_eval (cuFFT's are
 * not counted). */
se_status se_last_launch_count(const se_plan *p, int *count);

/* Benchmark diagnostics, not on the evaluation path: over the point sets of the last se_eval / SE_STAGE_SORT, the number
 * of (target, source) candidates in the 27 colleague cells and of pairs with 0 < r <= rc, counted in FP32
 * cell-relative coordinates (a pair within ~1e-6 rc of the cutoff may fall on either side).  bench.py rates K2 by
 * in-range pairs per second with them.  Synchronises the device. */
se_status se_count_pairs(se_plan *p, int64_t *candidates, int64_t *in_range);

/*
 * K4 (SE_STAGE_SCALE, eq. (2.6)) on a caller-owned DEVICE block of the spectrum: spec = [3][M][nky][M/2 + 1]
 * complex numbers of the plan's precision, holding the modes (i_x, i_y, i_z) with ky0 <= i_y < ky0 + nky (all i_x, all stored
 * i_z): what one rank holds between the two 1-D transforms of a slab-decomposed 3-D FFT (PAPER.md:664 (4)).  In place,
 * asynchronous on `stream`; valid on slab plans (only the plan's multiplier tables are used).  SE_EINVAL on a null pointer or a
 * range outside [0, M).
 */
se_status se_scale_block(se_plan *p, void *spec, int ky0, int nky, void *stream);

/*
 * K4 (eq. (2.6) with (2.4b) and the Gaussian window's deconvolution, reading S4) WITHOUT A PLAN AND WITHOUT ANY
 * ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the same kernel as se_scale_block on a caller-owned DEVICE block spec = [3][M][nky][M/2 + 1] complex numbers of
 * `precision` (modes ky0 <= i_y < ky0 + nky), in place, asynchronous on `stream`, for the multiplier of a Gaussian-window plan
 * with parameters (M, P, L, xi) -- the result equals se_scale_block's on such a plan up to the rounding of the multiplier table
 * (built here in double on the device, there in long double on the host).  Kaiser-Bessel plans are not covered.
 * The multiplier table (2 M reals) lives in a static device array of FIXED size inside the library: M <= 4096, i.e. 64 KB that
 * every GPU which loads the library holds until the process exits.  The call makes no cudaMalloc / cudaFree and calls no
 * library routine that allocates; its first call on a device looks up the array's address (cudaGetSymbolAddress), so make one
 * call per device before starting a graph capture.  The array is shared by all calls and is refilled by each of them (it keeps
 * the last call's table; nothing has to be cleared): calls that overlap on the GPU -- different streams, or graphs replayed
 * side by side -- RACE on it; calls ordered on one stream do not.
 * Errors: SE_EINVAL for a null pointer, odd or too small M or P, P > M, L or xi not positive, a ky range outside [0, M) or an
 * unknown precision; SE_ELIMIT for M > 4096 (or a device ordinal >= 64); SE_ECUDA if the look-up or a launch fails.
 */
se_status se_scale_noalloc(void *spec, int M, int P, double L, double xi, se_precision precision, int ky0, int nky, void *stream);

/* ---- parameter selection from a tolerance (section 2.4, eq. (2.9)) ------- */

typedef struct {
    double rc, xi;       /* cutoff and split parameter                                    */
    int M, P;            /* grid points per dimension (even, 2^a 3^b 5^c 7^d), window support */
    double EN, EF, Ew;   /* the three terms of eq. (2.9) at the chosen parameters          */
    double s;            /* mean points per near cell, N rc^3 / L^3                        */
    double model_ms;     /* the stage-time model's estimate for one evaluation on a B200   */
} se_params;

/*
 * HOST ONLY, no CUDA call: choose (rc, xi, M, P) for N points in [0,L)^3 so that each term of the error
 * estimate (2.9) is below eps/3 and the modelled time of Algorithm 2.1 is least
 * (min over rc of T(rc) subject to E_rms <= eps).  eps is the absolute RMS error for
 * sum_j |f_j|^2 = 1 in the unit box, as in the paper; E^N and E^F are (2.9)'s; E^w, whose constant C(xi) the paper
 * does not print, is the window's aliasing + truncation error at the chosen h and xi (reading S21).  P is rounded up
 * to a support the tensor-core gridding kernels are built for.  SE_EINVAL if N < 1, L <= 0, eps outside
 * (1e-15, 1e-1), or no admissible choice exists.
 */
se_status se_select_params(int64_t N, double L, double eps, se_window window, se_precision prec, se_params *out);

/* se_select_params followed by se_plan_create_ex (Nt as in se_plan_desc); *chosen (optional) receives the choice. */
se_status se_plan_create_tol(se_plan **out, int64_t N, int64_t Nt, double L, double eps, se_window window,
                             se_precision prec, se_params *chosen);

/* ---- measured arithmetic peaks (bench.py's roofline denominators) ------------------------------- */

/*
 * Time register-only dependent chains on the current device: which = 0 FP64 DFMA, 1 FP64 tensor op
 * (mma.sync m8n8k4 f64), 2 FP32 FFMA: *tflops receives 2 x FMA / s (in TFLOP/s) of the best of `reps` launches.
 * which = 3: an in-place streaming pass over 2 GiB, every 16 bytes read and written once (the access pattern of K4):
 * *tflops receives (bytes read + written) / s in TB/s.  Allocates and frees its own buffers; synchronises the device.
 */
se_status se_measure_peak(int which, int reps, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* SE_B200_H */
