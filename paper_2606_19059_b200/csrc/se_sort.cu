// K1: wrap + bin + counting sort, for both orderings the later stages need
//   (a) near cells of width L/ncell >= rc  -> K2 P2P
//   (b) grid bins of SE_BIN^3 Fourier-grid cells (the paper's C^F) -> K3 P2G, K5 G2P
// Unlike the paper's padded cell lists (two passes + max-occupancy padding)
// the lists are CSR (start offsets + a permutation), so clustered inputs cost no padding.
// The grid ordering also stores, per particle, the anchor grid index and the
// three 1-D Gaussian window tables of P values each, so that P2G and G2P never evaluate exp.
#include <cuda_fp16.h>

#include "se_common.cuh"

namespace {

__device__ __forceinline__ double wrap1(double x, double L)
{
    double v = x - L * floor(x / L);
    if (!(v >= 0.0 && v < L)) v = 0.0;      // also catches NaN/Inf: no out-of-range bins
    return v;
}

__device__ __forceinline__ int near_cell1(double v, const SeGeom &g)
{
    int c = (int)floor(v / g.wcell);
    return min(max(c, 0), g.ncell - 1);
}

// base grid index floor(x/h), in [0, M], and fractional offset in grid units.  M itself happens for the last few
// representable points below L, where x/h rounds up to M: the window then starts at anchor M - (P/2 - 1) and wraps
// like any other (the oracle's window_1d takes the same floor and wraps the indices), so the callers
// wrap the index instead of clamping it to M - 1 (which would truncate the window one plane earlier)
__device__ __forceinline__ int grid_base1(double v, const SeGeom &g, double &frac)
{
    double q = v / g.h;
    int i0 = (int)floor(q);
    i0 = min(max(i0, 0), g.M);
    frac = q - (double)i0;
    return i0;
}

template <typename Real>
__global__ void k_bin(SeGeom g, const Real *__restrict__ x, int *__restrict__ cell_of,
                      int *__restrict__ bin_of, int *__restrict__ cell_cnt, int *__restrict__ bin_cnt, int64_t nspread)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    int c[3], b[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double v = wrap1((double)x[3 * i + d], g.L);
        c[d] = near_cell1(v, g);
        double fr;
        b[d] = grid_base1(v, g, fr);
        if (b[d] == g.M) b[d] = 0;
    }
    int ci = (c[0] * g.ncell + c[1]) * g.ncell + c[2];
    int bi;
    if (g.grid_mode == 2) {
        int a[3];                                    // anchors, wrapped into [0, M)
#pragma unroll
        for (int d = 0; d < 3; ++d) { a[d] = b[d] - (g.P / 2 - 1); if (a[d] < 0) a[d] += g.M; }
        // slab plans: local plane of the anchor (a point whose window leaves the slab is the caller's error: clamped)
        a[0] -= g.px0; if (a[0] < 0) a[0] += g.M;
        if (g.Mx < g.M) a[0] = min(a[0], g.Mx - g.P);
        bi = (a[0] * g.nbin + a[2] / SE_MMA_ZBIN) * g.M + a[1];
    } else
        bi = ((b[0] / SE_BIN) * g.nbin + b[1] / SE_BIN) * g.nbin + b[2] / SE_BIN;
    if (i >= nspread) bi = g.nbins_total;          // ghost sources of a slab plan: the extra bin no gridding tile visits
    cell_of[i] = ci;
    bin_of[i] = bi;
    atomicAdd(&cell_cnt[ci], 1);
    atomicAdd(&bin_cnt[bi], 1);
}

// ---- exclusive scan of the two histograms: tile sums, then per-tile scan -----------------
constexpr int SCAN_T = 256;            // threads
constexpr int SCAN_E = 8;              // elements per thread
constexpr int SCAN_TILE = SCAN_T * SCAN_E;

__device__ __forceinline__ int block_sum(int v, int *sm)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    int t = 0;
    for (int w = 0; w < SCAN_T / 32; ++w) t += sm[w];
    __syncthreads();
    return t;
}

// which = blockIdx.y (0: near cells, 1: grid bins)
__global__ void __launch_bounds__(SCAN_T) k_tile_sums(const int *cntA, int nA, int *sumsA,
                                                      const int *cntB, int nB, int *sumsB)
{
    __shared__ int sm[SCAN_T / 32];
    const int *cnt = blockIdx.y ? cntB : cntA;
    int n = blockIdx.y ? nB : nA;
    int *sums = blockIdx.y ? sumsB : sumsA;
    int base = blockIdx.x * SCAN_TILE;
    if (base >= n) return;
    int v = 0;
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        int i = base + e * SCAN_T + threadIdx.x;
        if (i < n) v += cnt[i];
    }
    int t = block_sum(v, sm);
    if (threadIdx.x == 0) sums[blockIdx.x] = t;
}

// cursor (in: counts) -> cursor = start (exclusive prefix), start[0..n] likewise
__global__ void __launch_bounds__(SCAN_T) k_tile_scan(int *curA, int *startA, int nA, const int *sumsA,
                                                      int *curB, int *startB, int nB, const int *sumsB)
{
    __shared__ int sm[SCAN_T / 32];
    __shared__ int wsum[SCAN_T / 32];
    int *cur = blockIdx.y ? curB : curA;
    int *start = blockIdx.y ? startB : startA;
    int n = blockIdx.y ? nB : nA;
    const int *sums = blockIdx.y ? sumsB : sumsA;
    int base = blockIdx.x * SCAN_TILE;
    if (base >= n) return;
    // offset of this tile = sum of the preceding tile sums
    int pre = 0;
    for (int b = threadIdx.x; b < (int)blockIdx.x; b += SCAN_T) pre += sums[b];
    pre = block_sum(pre, sm);
    // each thread owns SCAN_E consecutive elements
    int i0 = base + threadIdx.x * SCAN_E;
    int v[SCAN_E], tot = 0;
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        v[e] = (i0 + e < n) ? cur[i0 + e] : 0;
        tot += v[e];
    }
    // inclusive warp scan of tot
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += y;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    int woff = 0;
    for (int q = 0; q < w; ++q) woff += wsum[q];
    int run = pre + woff + inc - tot;
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        if (i0 + e < n) { cur[i0 + e] = run; start[i0 + e] = run; }
        run += v[e];
        if (i0 + e == n - 1) start[n] = run;
    }
}

__global__ void k_scatter(int64_t N, const int *__restrict__ cell_of, const int *__restrict__ bin_of,
                          int *__restrict__ cell_cur, int *__restrict__ bin_cur,
                          int *__restrict__ perm_near, int *__restrict__ inv_near,
                          int *__restrict__ perm_grid, int *__restrict__ inv_grid)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int p = atomicAdd(&cell_cur[cell_of[i]], 1);
    perm_near[p] = (int)i;
    inv_near[i] = p;
    int q = atomicAdd(&bin_cur[bin_of[i]], 1);
    perm_grid[q] = (int)i;
    inv_grid[i] = q;
}

// The slot a particle gets inside its cell depends on atomic arrival order.  Re-rank every
// cell segment by user index so that the sorted order (hence every later floating-point
// summation order) is a pure function of the input.  One thread per sorted slot, O(s) each.
__global__ void k_rank_in_cell(int64_t N, const int *__restrict__ key_of, const int *__restrict__ start,
                               const int *__restrict__ perm_in, int *__restrict__ perm_out,
                               int *__restrict__ inv, int skip_key)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    int i = perm_in[p];
    int c = key_of[i];
    if (c == skip_key) {                 // the bin of a slab plan's ghost sources: never gridded, any order will do (it
        perm_out[p] = i;                 // can hold tens of thousands of points, and the ranking below is O(occupancy))
        inv[i] = (int)p;
        return;
    }
    int s = start[c], e = start[c + 1];
    int r = 0;
    for (int q = s; q < e; ++q) r += (perm_in[q] < i);
    perm_out[s + r] = i;
    inv[i] = s + r;
}

// Near-sorted copies for K2: src[p] = (x, y, z, f_x, f_y, f_z) in the plan's precision (absolute wrapped
// coordinates for fp64 plans, cell-relative for fp32 plans), xq[p] = (x, y, z relative to the cell origin, absolute z)
// in FP32 for the candidate filter, cellp[p] = packed cell coordinates (cx << 20 | cy << 10 | cz; ncell <= 1024).
template <typename Real>
__global__ void k_gather_near(SeGeom g, const Real *__restrict__ x, const Real *__restrict__ f,
                              const int *__restrict__ perm, const int *__restrict__ cell_of,
                              Real *__restrict__ src, float4 *__restrict__ xq, unsigned short *__restrict__ xp,
                              int *__restrict__ cellp)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= g.N) return;
    int i = perm[p];
    int ci = cell_of[i];
    int c[3] = {ci / (g.ncell * g.ncell), (ci / g.ncell) % g.ncell, ci % g.ncell};
    float q[4];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double v = wrap1((double)x[3 * (int64_t)i + d], g.L);
        double rel = v - (double)c[d] * g.wcell;            // cell-relative, rounded once
        q[d] = (float)rel;
        if (d == 2) q[3] = (float)v;
        src[6 * p + d] = (Real)(g.rel_coords ? rel : v);
        src[6 * p + 3 + d] = f ? f[3 * (int64_t)i + d] : (Real)0;      // a target set carries no strengths
    }
    xq[p] = make_float4(q[0], q[1], q[2], q[3]);
    cellp[p] = (c[0] << 20) | (c[1] << 10) | c[2];
    // FP16 pair records of the K2 filter (se_common.cuh): this point is half (p & 1) of even pair p >> 1 and half
    // ((p - 1) & 1) of odd pair (p - 1) >> 1; a half without a point (past the end) holds a coordinate that is never in range
    const size_t odd = (size_t)SE_XP_LEN(g.N) * 8;             // offset of the odd-pair array, in halves
    const unsigned short farh = 0xd640;                         // -100 in FP16
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const unsigned short hv = __half_as_ushort(__float2half_rn(q[d] * (float)(1.0 / g.wcell)));
        xp[(size_t)(p >> 1) * 8 + 2 * d + (p & 1)] = hv;
        if (p > 0) xp[odd + (size_t)((p - 1) >> 1) * 8 + 2 * d + ((p - 1) & 1)] = hv;
        if (p == g.N - 1) {                                     // the halves behind the last point
            if (!(p & 1)) xp[(size_t)(p >> 1) * 8 + 2 * d + 1] = farh;
            if (p > 0 && !((p - 1) & 1)) xp[odd + (size_t)((p - 1) >> 1) * 8 + 2 * d + 1] = farh;
        }
    }
}

// one thread per (sorted particle, dim, l): window value at the physical offset t_l = (anchor + l) h - x
// (reading S11).  Gaussian: exp(-beta (l - (P/2-1) - frac)^2) = exp(-a t_l^2).  Kaiser-Bessel
// (eq. (2.8)): the polynomial of bin l, degree nu, in s = 2 (t_l/h - (l - P/2)) - 1 by Horner's rule
// (PAPER.md:421-427), coefficients wcoef[l][0..nu].  Always evaluated in double and rounded once to Rec.  In mma
// mode the values go into the per-particle spread and gather records of se_mma.cu (layout in se_common.cuh;
// either pointer may be null: a source-only set has no gather records, a target set no spread records)
// instead of the plain [N][3][P] table.
// KB: Kaiser-Bessel plans (compile-time: the Gaussian path keeps its registers and its schedule)
template <typename Real, typename Rec, bool KB>
__global__ void k_gather_grid(SeGeom g, const Real *__restrict__ x, const Real *__restrict__ f,
                              const int *__restrict__ perm, short4 *__restrict__ anchor,
                              Rec *__restrict__ wtab, Rec *__restrict__ recg, Real *__restrict__ fs,
                              const double *__restrict__ wcoef)
{
    // LP = 16 or 32 lanes per particle: lane d < 3 of the group wraps coordinate d and finds its base index once,
    // the group shares them by shuffle, then lane l < P evaluates window value l of each dimension and the rows
    // are written with consecutive lanes on consecutive addresses
    const int P = g.P, P3 = 3 * P;
    const int LP = P <= 16 ? 16 : 32;
    const int lane = threadIdx.x & 31, l = lane & (LP - 1), gbase = lane & ~(LP - 1);
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t p = warp * (32 / LP) + (lane / LP);
    const bool live = p < g.N;
    const int64_t pc = live ? p : g.N - 1;
    const int i = perm[pc];
    double frac = 0.0, xw = 0.0;
    int i0 = 0;
    Real fd = (Real)0;
    if (l < 3) {
        xw = wrap1((double)x[3 * (int64_t)i + l], g.L);
        i0 = grid_base1(xw, g, frac);
        fd = f ? f[3 * (int64_t)i + l] : (Real)0;
    }
    const bool recs = g.grid_mode == 2;
    const int R = recs ? g.ring : P, Rg = recs ? g.ring_g : P;         // row strides (R >= Rg >= P)
    Rec *rs = wtab + pc * SE_MMA_RECS(R), *rg = recg + pc * SE_MMA_RECG(Rg);
    Rec cf[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) cf[c] = (Rec)g.cw * (Rec)__shfl_sync(0xffffffffu, fd, gbase + c);   // c_w of eq. (2.5) folded in
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double fr = __shfl_sync(0xffffffffu, frac, gbase + d);
        const double xd = __shfl_sync(0xffffffffu, xw, gbase + d);
        const int id = __shfl_sync(0xffffffffu, i0, gbase + d);
        if (!live || l >= R) continue;
        double wv = 0.0;                                                // rows are zero beyond the window
        if (l < P) {
            if (KB) {
                const double t = (double)(id - (P / 2 - 1) + l) * g.h - xd;
                const double sv = 2.0 * (t / g.h - (double)(l - P / 2)) - 1.0;
                const double *cc = wcoef + l * (g.nu + 1);
                wv = __ldg(cc + g.nu);
                for (int k = g.nu - 1; k >= 0; --k) wv = fma(wv, sv, __ldg(cc + k));
            } else {
                const double u = (double)(l - (P / 2 - 1)) - fr;
                wv = exp(-g.beta * u * u);
            }
        }
        const Rec w = (Rec)wv;
        if (recs) {
            if (recg && l < Rg) rg[d * Rg + l] = w;
            if (wtab) {
                if (d == 0) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) rs[c * R + l] = cf[c] * w;
                } else
                    rs[(d + 2) * R + l] = w;
            }
        } else if (l < P)
            wtab[pc * P3 + d * P + l] = w;
    }
    if (live && l < 3) {
        int a = i0 - (P / 2 - 1);
        if (a < 0) a += g.M;
        if (a >= g.M) a -= g.M;
        short *ap = reinterpret_cast<short *>(&anchor[p]);
        ap[l] = (short)a;
        if (l == 0) ap[3] = 0;
        fs[3 * p + l] = fd;
        if (recs && l > 0) {
            if (wtab) reinterpret_cast<int *>(&rs[5 * R])[l - 1] = a;
            if (recg) reinterpret_cast<int *>(&rg[3 * Rg])[l - 1] = a;
        }
    }
}

template <typename Real>
__global__ void k_sum(int64_t N, const Real *__restrict__ uN, const Real *__restrict__ uF,
                      const Real *__restrict__ f, const int *__restrict__ inv_near,
                      const int *__restrict__ inv_grid, Real far_scale, Real cself, Real *__restrict__ u)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * N) return;
    int64_t i = t / 3;
    int c = (int)(t - 3 * i);
    Real v = uN[3 * (int64_t)inv_near[i] + c] + far_scale * uF[3 * (int64_t)inv_grid[i] + c];
    if (f) v -= cself * f[t];                        // self term: only when the targets are the sources (reading S3)
    u[t] = v;
}

// Sort one point set.  f == nullptr: a target set (no strengths).  spread / gather: which mma-mode records to write.
template <typename Real>
cudaError_t sort_set(se_plan *p, SeSet &S, const void *xv, const void *fv, bool spread, bool gather, cudaStream_t s)
{
    SeGeom g = p->g;
    g.N = S.n;
    const Real *x = (const Real *)xv, *f = (const Real *)fv;
    int nc3 = g.ncell * g.ncell * g.ncell, nb3 = g.nbins_total + 1;
    cudaError_t e = cudaMemsetAsync(S.cell_cursor, 0, sizeof(int) * (nc3 + 1), s);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(S.bin_cursor, 0, sizeof(int) * (nb3 + 1), s);
    if (e != cudaSuccess) return e;
    int T = 256;
    unsigned nblk = (unsigned)((g.N + T - 1) / T);
    k_bin<Real><<<nblk, T, 0, s>>>(g, x, S.cell_of, S.bin_of, S.cell_cursor, S.bin_cursor,
                                   (spread && p->nown > 0) ? p->nown : g.N);
    int tilesA = (nc3 + SCAN_TILE - 1) / SCAN_TILE, tilesB = (nb3 + SCAN_TILE - 1) / SCAN_TILE;
    int tiles = tilesA > tilesB ? tilesA : tilesB;
    // tile sums live behind the CSR arrays: the plan allocates cell_start / bin_start with room for them after entry n
    int *sumsA = S.cell_start + (nc3 + 1), *sumsB = S.bin_start + (nb3 + 1);
    k_tile_sums<<<dim3(tiles, 2), SCAN_T, 0, s>>>(S.cell_cursor, nc3, sumsA, S.bin_cursor, nb3, sumsB);
    k_tile_scan<<<dim3(tiles, 2), SCAN_T, 0, s>>>(S.cell_cursor, S.cell_start, nc3, sumsA,
                                                   S.bin_cursor, S.bin_start, nb3, sumsB);
    // scatter into scratch permutations (cell_sorted and the fs_grid array double as scratch), then re-rank
    int *tmp_near = S.cell_sorted, *tmp_grid = (int *)S.fs_grid;  // both >= n ints, overwritten later
    k_scatter<<<nblk, T, 0, s>>>(g.N, S.cell_of, S.bin_of, S.cell_cursor, S.bin_cursor,
                                 tmp_near, S.inv_near, tmp_grid, S.inv_grid);
    k_rank_in_cell<<<nblk, T, 0, s>>>(g.N, S.cell_of, S.cell_start, tmp_near, S.perm_near, S.inv_near, -1);
    k_rank_in_cell<<<nblk, T, 0, s>>>(g.N, S.bin_of, S.bin_start, tmp_grid, S.perm_grid, S.inv_grid, g.nbins_total);
    k_gather_near<Real><<<nblk, T, 0, s>>>(g, x, f, S.perm_near, S.cell_of, (Real *)S.src_near,
                                           (float4 *)S.xq, (unsigned short *)S.xp, S.cell_sorted);
    int64_t nt = (g.N + (g.P <= 16 ? 1 : 0)) / (g.P <= 16 ? 2 : 1) * 32;   // 16 or 32 lanes per particle
    const unsigned ngb = (unsigned)((nt + T - 1) / T);
    const bool kb = g.window == SE_WINDOW_KAISER_BESSEL;
    if (g.grid_mode == 2) {                                    // records are double for every plan precision
        double *ws = spread ? (double *)S.wtab : nullptr, *wg = gather ? (double *)S.recg : nullptr;
        if (kb)
            k_gather_grid<Real, double, true><<<ngb, T, 0, s>>>(g, x, f, S.perm_grid, S.anchor, ws, wg, (Real *)S.fs_grid, p->wcoef);
        else
            k_gather_grid<Real, double, false><<<ngb, T, 0, s>>>(g, x, f, S.perm_grid, S.anchor, ws, wg, (Real *)S.fs_grid, p->wcoef);
    } else if (kb)
        k_gather_grid<Real, Real, true><<<ngb, T, 0, s>>>(g, x, f, S.perm_grid, S.anchor, (Real *)S.wtab, (Real *)S.recg,
                                                            (Real *)S.fs_grid, p->wcoef);
    else
        k_gather_grid<Real, Real, false><<<ngb, T, 0, s>>>(g, x, f, S.perm_grid, S.anchor, (Real *)S.wtab, (Real *)S.recg,
                                                             (Real *)S.fs_grid, p->wcoef);
    p->launches += 8;
    return cudaGetLastError();
}

template <typename Real>
cudaError_t sort_impl(se_plan *p, const void *xv, const void *fv, const void *xt, cudaStream_t s)
{
    if (!p->own_targets) return sort_set<Real>(p, p->S, xv, fv, true, true, s);
    cudaError_t e = sort_set<Real>(p, p->S, xv, fv, true, false, s);
    if (e != cudaSuccess) return e;
    return sort_set<Real>(p, p->T, xt, nullptr, false, true, s);
}

template <typename Real>
cudaError_t sum_impl(se_plan *p, const void *f, void *u, cudaStream_t s)
{
    const SeGeom &g = p->g;
    double far_scale = g.h * g.h * g.h * g.cw;                 // eq. (2.7) h^3 and the window's c_w
    double cself = 4.0 * g.xi / sqrt(SE_PI);                   // self term, reading S3
    int T = 256;
    const int64_t nt = p->T.n;
    k_sum<Real><<<(unsigned)((3 * nt + T - 1) / T), T, 0, s>>>(nt, (const Real *)p->uN, (const Real *)p->uF,
                                                              (p->own_targets && !p->nown) ? nullptr : (const Real *)f,
                                                              p->T.inv_near, p->T.inv_grid,
                                                              (Real)far_scale, (Real)cself, (Real *)u);
    p->launches += 1;
    return cudaGetLastError();
}

}  // namespace

cudaError_t se_launch_sort(se_plan *p, const void *x, const void *f, const void *xt, cudaStream_t s)
{
    return p->precision == SE_FP64 ? sort_impl<double>(p, x, f, xt, s) : sort_impl<float>(p, x, f, xt, s);
}

cudaError_t se_launch_sum(se_plan *p, const void *f, void *u, cudaStream_t s)
{
    return p->precision == SE_FP64 ? sum_impl<double>(p, f, u, s) : sum_impl<float>(p, f, u, s);
}
