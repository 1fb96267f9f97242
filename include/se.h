/*
 * se.h -- C-ABI of the B200 spectral Ewald library (libse_b200.so).
 *
 * Evaluates the triply periodic Stokeslet sum
 *     u(x_i) = sum_j sum_{p in L Z^3} G(x_i - x_j + p) f_j ,   G(r) = I/|r| + r (x) r/|r|^3
 * (eq. (2.1)) with the Hasimoto split G = G^N + G^F
 * (eq. (2.3), eq. (2.4b)) by the spectral Ewald method
 * (Algorithm 2.1): P2P + P2G + FFT + CNV + IFFT + G2P + SUM, with a
 * Gaussian window over P^3 grid points (reading S4).  Targets = sources; the
 * i = j, p = 0 pair is excluded and the self term -(4 xi/sqrt(pi)) f_i is added
 * (reading S3); the k = 0 mode is dropped (reading S2); G carries no 1/(8 pi mu).
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
 *     thread-safe.
 *   - Every entry point returns a status; nothing aborts or throws.  NaN/Inf inputs give
 *     unspecified values but never out-of-bounds accesses.
 *   - There is no CPU fallback: without a CUDA device se_plan_create returns SE_ECUDA.
 *   - Environment variables read at se_plan_create (experiments and tests only; results do not change beyond
 *     rounding order): SE_GRID_MODE = tile (force the generic gridding kernel; default: the FP64 tensor-core
 *     sweep for fp64 plans with P = 16, 24 and fp32 plans with P = 12, else the generic tile kernel), SE_NCHUNK and
 *     SE_NCHUNK_G2P (x-chunks of K3 / K5), SE_OVERLAP = 1 (K2 on a side stream next to the FFT stages).
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

typedef enum {
    SE_OK = 0,
    SE_EINVAL = 1,   /* bad argument (see se_plan_create) or null pointer            */
    SE_ENOMEM = 2,   /* device or host allocation failed                             */
    SE_ECUDA = 3,    /* a CUDA runtime call or kernel launch failed / no device      */
    SE_ECUFFT = 4    /* a cuFFT call failed                                          */
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

/* Internal buffers visible to tests and the benchmark through se_buffer_read/write. */
enum {
    SE_BUF_UN = 0,        /* u^N, N x 3 reals, NEAR-sorted order                                   */
    SE_BUF_UF = 1,        /* u^F, N x 3 reals, GRID-sorted order                                   */
    SE_BUF_GRID = 2,      /* real grid H (after P2G) / H~ (after IFFT): 3 x M x M x M reals, z fastest */
    SE_BUF_SPEC = 3,      /* spectrum: 3 x M x M x (M/2+1) complex (re,im) reals, halved axis last  */
    SE_BUF_PERM_NEAR = 4, /* int32[N]: sorted position -> user index, near-cell order              */
    SE_BUF_PERM_GRID = 5, /* int32[N]: sorted position -> user index, grid-bin order               */
    SE_BUF_CELL_START = 6,/* int32[ncell^3 + 1]: CSR offsets of the near cells                     */
    SE_BUF_BIN_START = 7, /* int32[nbins_total + 1]: CSR offsets of the grid bins.  Mode 0: bins of 8^3 grid
                             cells, key (bx, by, bz); mode 1: key (base plane ix, by/4, bz/4)               */
    SE_NBUFS = 8
};

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
    int nbins_total;     /* entries of SE_BUF_BIN_START minus 1: nbin^3 (mode 0), M * nbin^2 (mode 1)      */
    int nchunk;          /* tensor-core sweep: chunks along x (P2G)                      */
    int64_t nmodes;      /* M * M * (M/2+1) stored modes per component                   */
    size_t workspace_bytes; /* device memory owned by the plan (incl. cuFFT work area)   */
} se_info;

/*
 * Create a plan.  N particles in the periodic cube [0,L)^3, split parameter xi,
 * near-field cutoff rc, M^3 Fourier grid, Gaussian support P grid points per dimension.
 * SE_EINVAL if: out == NULL, N < 1, N >= 2^31, L <= 0, xi <= 0, rc <= 0, M < 2, M odd,
 * M > 4096, P < 2, P odd, P > 32, P > M, floor(L/rc) < 3 (the 27-cell stencil would
 * alias, reading S7), or an unknown precision.  On any failure *out is NULL.
 */
se_status se_plan_create(se_plan **out, int64_t N, double L, double xi, double rc,
                         int M, int P, se_precision prec);

/* Full evaluation, all stages; x, f, u are device pointers (N x 3). */
se_status se_eval(se_plan *p, const void *x, const void *f, void *u, void *stream);

/*
 * Same, with HOST buffers (pinned or pageable): copies x, f host->device into plan-owned
 * staging buffers, runs se_eval, copies u device->host, all asynchronously on `stream`
 * (the caller synchronises the stream before reading u_host).
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

#ifdef __cplusplus
}
#endif
#endif /* SE_B200_H */
