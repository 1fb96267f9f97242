// Internal definitions shared by the kernels of libse_b200.so (sm_100a only).
// Boundary and semantics: include/se.h.  Paper citations are PAPER.md line numbers.
#pragma once

#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>

#include "../../include/se.h"

#define SE_PI 3.14159265358979323846264338327950288

// ---- geometry of the gridding kernels (K3 P2G / K5 G2P) ---------------------------------
// Output tile owned by one block: TX x TY x TZ grid points; one thread per (x,y) column,
// TZ accumulators x 3 components in registers.  Particles are sorted by bins of BIN^3
// grid cells (z fastest) so that the candidates of a tile are a few contiguous runs.
constexpr int SE_TX = 16;
constexpr int SE_TY = 16;
constexpr int SE_TZ = 8;
constexpr int SE_BIN = 8;
constexpr int SE_GRID_THREADS = SE_TX * SE_TY;      // 256
constexpr int SE_ROUND = 128;                        // candidates examined per staging round
constexpr int SE_PMAX = 32;                          // largest window support
// FP64 tensor-core gridding kernels (se_mma.cu): particles sorted by (anchor plane, anchor_z / ZBIN, anchor_y);
// a block of NWY x NWZ consumer warps (+ the producer warpgroup) owns 4 NWY x 4 NWZ (y, z) columns.  K1 writes two
// 16-byte aligned records per particle in sorted order (always double, also for fp32 plans; anchors as two int32
// in one double slot; R = P rounded up to a multiple of 8, Rg = P rounded up to a multiple of 4, rows zero beyond P):
//   spread record, SE_MMA_RECS(R) doubles: c_w f_x Wx[R] | c_w f_y Wx[R] | c_w f_z Wx[R] | Wy[R] | Wz[R] | (a_y, a_z) | pad
//   gather record, SE_MMA_RECG(Rg) doubles: Wx[Rg] | Wy[Rg] | Wz[Rg] | (a_y, a_z) | pad
// (sizes = 24 mod 32 four-byte words, so that consecutive records start in different shared-memory bank octets)
constexpr int SE_MMA_ZBIN = 8;
constexpr int SE_MMA_NWY = 2, SE_MMA_NWZ = 6;
#define SE_MMA_RECS(P) (5 * (P) + 4)
#define SE_MMA_RECG(P) (3 * (P) + 4)
#define SE_XP_LEN(n) (((n) + 1) / 2 + 1)

// Passed to every kernel BY VALUE and captured by the kernels' lambdas: keep it at 128 bytes (at 136 the compiler stopped
// keeping its fields in registers: k_mma<gather> executed 5.6 % more instructions, 5.76 -> 6.14 ms on config 3).
struct SeGeom {
    int64_t N;          // points of the set a launch works on (sources or targets; the launchers set it)
    int M, P;
    int Mx, px0;        // planes of the grid along x (M unless a slab plan) and global index of local plane 0
    int ncell;          // near cells per dimension
    int nbin;           // grid bins per dimension = ceil(M / SE_BIN) (tile mode) or z-bins ceil(M / 8) (mma mode)
    int nbins_total;    // nbin^3 (tile mode), Mx * nbin * M (mma mode)
    int nchunk;         // mma mode: chunks along x (P2G)
    int nchunk_g2p;     // mma mode: chunks along x (G2P)
    int nfull, nsplit;  // mma mode, P2G with nchunk = 1: the last `tiles - nfull` block tiles (those of the partly filled
                        // last wave) are split into nsplit x-chunks each (nsplit = 1: no split)
    short window;       // se_window
    short nu;           // Kaiser-Bessel: polynomial degree per bin
    short grid_mode;    // 0: tile-stationary k_grid (any even P),
                        // 2: FP64 tensor-core sweep (se_mma.cu; fp64 any even P <= 24, fp32 any even P <= 16)
    short ring;         // mma mode: row stride of the spread records = P rounded up to a multiple of 8
    short rel_coords;   // 1: near-sorted positions are cell-relative (fp32 path)
    short ring_g;       // mma mode: row stride of the gather records = P rounded up to a multiple of 4
    double L, xi, rc;
    double h;           // L / M
    double wcell;       // L / ncell
    double beta;        // a h^2 : window = exp(-beta (l' - frac)^2) in grid units
    double cw;          // (a/pi)^{3/2}
    double eta;
};
static_assert(sizeof(SeGeom) == 128, "SeGeom is a by-value kernel parameter: see the comment above");

// One point set (the sources, or a plan's own targets) in its two sorted orders.
struct SeSet {
    int64_t n;
    // near field (K1a, K2)
    int *cell_of;                  // [n]  near cell of user particle i
    int *cell_start;               // [ncell^3 + 1]
    int *cell_cursor;              // [ncell^3 + 1] scatter cursors
    int *perm_near;                // [n] sorted pos -> user index
    int *inv_near;                 // [n] user index -> sorted pos
    int *cell_sorted;              // [n] packed cell coordinates (cx << 20 | cy << 10 | cz) of sorted particle
    void *src_near;                // [n][6] Real: x, y, z (absolute fp64 / cell-relative fp32), f_x, f_y, f_z (0 for targets)
    void *xq;                      // [n] float4: cell-relative x, y, z and absolute z in FP32 (K2: the targets' side of the filter)
    void *xp;                      // K2 candidate filter, the sources' side: FP16 PAIR records (x0 x1 | y0 y1 | z0 z1 | 0), coordinates
                                   // relative to the cell in units of the cell width; two arrays of SE_XP_LEN(n) records: [0] pairs
                                   // (2m, 2m + 1), [1] pairs (2m + 1, 2m + 2), so that a cell's sources pair up from its first one
    // grid path (K1b, K3, K5)
    int *bin_of;                   // [n]
    int *bin_start;                // [nbins_total + 1]
    int *bin_cursor;               // [nbins_total + 1]
    int *perm_grid;                // [n]
    int *inv_grid;                 // [n]
    short4 *anchor;                // [n] (a_x, a_y, a_z, 0): anchor grid index in [0, M)
    void *wtab;                    // [n][3][P] Real: 1-D window values of every particle (mma mode: spread records)
    void *recg;                    // mma mode: gather records
    void *fs_grid;                 // [n][3] Real
};

struct se_plan {
    SeGeom g;
    int precision;
    int device;
    int profiling;
    int launches;
    size_t real_bytes;             // sizeof(Real)
    SeSet S;                       // sources
    SeSet T;                       // targets: a copy of S (same pointers) unless the plan has its own targets
    int own_targets;               // 1: T has its own arrays (se_eval_targets)
    int slab;                      // 1: slab plan (grid Mx x M x M, no transforms; se.h se_plan_desc)
    int64_t nown;                  // slab plans with ghost sources: the first nown sources are spread, the targets are those points
    const void *xt_stage;          // se_set_targets: target positions for se_eval_stage(SE_STAGE_SORT)
    double *wcoef;                 // Kaiser-Bessel: [P][nu + 1] polynomial coefficients (always double)
    void *uN;                      // [Nt][3] Real, the targets' near-sorted order
    void *uF;                      // [Nt][3] Real, the targets' grid-sorted order (unscaled sum)
    void *uFpart;                  // mma mode: [slots][Nt][3] double per-(particle, block tile) partial sums
    // grids
    void *grid;                    // [3][M][M][M] Real
    void *spec;                    // [3][M][M][M/2+1] complex Real
    void *ktab;                    // [2][M] Real : k value, exp factor per 1-D index
    double *mtab;                  // K2 function tables (se_p2p.cu): erfcx pieces + exp polynomial, always double
    cufftHandle fft_fwd, fft_inv;
    int fft_ok;
    // fused x-transform + K4 (se_scale.cu, K4x): se_eval runs cuFFT 2-D over (y, z) per x-plane, k_xfft_scale, cuFFT 2-D back
    cufftHandle fft2_fwd, fft2_inv;
    int fft2_ok;
    int xf_ok, xf_tz, xf_nst, xf_radix[12], xf_threads, xf_r16;
    unsigned xf_magic[12];
    void *xf_tw;                   // [M] complex Real: w_M^t
    void *xf_xk;                   // [M] complex Real: (k_x, e_x) of the mode at position p after the forward stages
    // own 2-D transforms of the x-planes (se_scale.cu k_zr2c / k_zc2r / k_yfft) instead of cuFFT's, when f2_ok
    int f2_ok, f2_rb, f2_rbi, f2_rbmax, f2_rs, f2_zthreads, f2_zithreads, f2_ythreads;
    int f2z_nst, f2z_radix[12], f2y_nst, f2y_radix[12];
    unsigned f2z_magic[12], f2y_magic[12];
    int *f2_zpos;                  // [M/2] position of frequency k after the forward stages of the M/2-point transform over z
    void *f2_ykk;                  // [M] complex Real: (k_y, e_y) of the mode at position p of the second axis (digit-reversed)
    size_t fft_work_bytes;
    // host-buffer entry point staging
    void *hx, *hf, *hu;            // device staging [N][3] Real each
    size_t workspace_bytes;
    cudaEvent_t ev[SE_NSTAGES + 1];
    int ev_ok, ev_recorded;
    // SE_OVERLAP=1: se_eval runs K2 P2P (plain-ALU bound) on a side stream, forked after K3 and joined before K6,
    // next to the HBM-bound FFT / scale / IFFT stages (PAPER.md:690 notes the two chains are independent)
    cudaStream_t side;
    cudaEvent_t ev_fork, ev_join, ev_p2p[2];
    int overlap, side_ok;
};

// ---- launchers implemented in the .cu files -------------------------------------------------
cudaError_t se_launch_sort(se_plan *p, const void *x, const void *f, const void *xt, cudaStream_t s);
cudaError_t se_launch_p2p(se_plan *p, cudaStream_t s);
cudaError_t se_launch_p2g(se_plan *p, cudaStream_t s);
cudaError_t se_launch_scale(se_plan *p, cudaStream_t s);
cudaError_t se_build_xfft(se_plan *p);       // se_scale.cu: decides p->xf_ok, builds the tables of the fused x-transform
cudaError_t se_launch_xfft_scale(se_plan *p, cudaStream_t s);
cudaError_t se_launch_fft2(se_plan *p, bool forward, cudaStream_t s);   // se_scale.cu: own 2-D transforms (p->f2_ok)
cudaError_t se_tune_xfft(se_plan *p);        // se_scale.cu: K4x's mode table (after se_build_ktab) and its block shape, timed once
cudaError_t se_launch_g2p(se_plan *p, cudaStream_t s);
cudaError_t se_launch_sum(se_plan *p, const void *f, void *u, cudaStream_t s);
cudaError_t se_build_ktab(se_plan *p);      // se_window.cu: k values and the deconvolution factor per 1-D index
cudaError_t se_build_wcoef(se_plan *p);     // se_window.cu: allocates and fills p->wcoef (Kaiser-Bessel plans)
cudaError_t se_build_mtab(se_plan *p);      // allocates and fills p->mtab
cudaError_t se_prepare_mma(se_plan *p);     // per-plan kernel attributes (dynamic shared memory opt-in) on the plan's device
cudaError_t se_prepare_grid(se_plan *p);
int se_kb_degree(int P);                    // reading S19
// Chebyshev-node interpolant of fn on [c - hw, c + hw], degree deg <= 23, as monomials in (x - c)/hw (host, long double)
void se_cheb_fit(long double (*fn)(long double, const void *), const void *ctx, long double c, long double hw, int deg,
                 double *out);
cudaError_t se_launch_mma_p2g(se_plan *p, cudaStream_t s);
cudaError_t se_launch_mma_g2p(se_plan *p, cudaStream_t s);
bool se_mma_supported(int P, int precision);
int se_mma_slots(int P);
int se_mma_ring(int P);
int se_mma_ring_g(int P);
