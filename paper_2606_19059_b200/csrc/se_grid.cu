// K3 P2G (spreading, eq. (2.5)) and K5 G2P (gather, eq. (2.7)).
//
// Design for B200 (differs from the paper's P2G-hybrid, which flushes
// per-thread partial sums with O(27 N) global atomics, and from its thread-per-target G2P,
// PAPER.md:394, which re-reads P^3 grid values per target through L2):
//   * OUTPUT-STATIONARY P2G: a block owns a TX x TY x TZ tile of the Fourier grid; each
//     thread owns one (x,y) column of the tile and keeps its TZ x 3 accumulators in
//     registers.  The block walks the particles whose P^3 support can touch the tile
//     (contiguous runs of the bin-sorted order), stages their 1-D window slices in shared
//     memory, and every thread adds  W1[i] W2[j] * (f_c W3[k]).  The tile is written once
//     with plain stores: no atomics, no zero-fill pass, deterministic.
//   * GRID-STATIONARY G2P: the transpose.  The thread loads its column of the
//     three component grids into registers once and reuses it for every overlapping
//     particle; partial sums are reduced across the warp and accumulated per particle.
//   * No exp in these kernels: the window tables come from K1 (se_sort.cu).
// Both are FP64/FP32 FMA-bound at P = 24 / 12 (3 P^3 FMA per particle against ~1 KB of
// compulsory traffic), see DESIGN.md.
#include "se_common.cuh"

namespace {

constexpr int MAXRUN = 128;      // candidate runs per tile (columns x up to 2 z-segments)

template <typename Real>
struct alignas(16) GridSmem {
    Real W1[SE_ROUND][SE_TX];
    Real W2[SE_ROUND][SE_TY];
    Real G[SE_ROUND][3 * SE_TZ];     // P2G: f_c W3[k] (c-major);  G2P: W3[k] in the first TZ
    Real U[SE_ROUND][3];             // G2P: per-particle partial sums of this round
    int pidx[SE_ROUND];              // sorted particle index of accepted candidate
    short lst[SE_ROUND][4];          // first window index of the tile in x, y, z
    unsigned char wlist[SE_GRID_THREADS / 32][SE_ROUND];
    int wcnt[SE_GRID_THREADS / 32];
    int acc_cnt[SE_GRID_THREADS / 32];
    int run_beg[MAXRUN];
    int run_ofs[MAXRUN + 1];
    int nrun;
};

// does window index (l0 + i) mod M fall inside [0, P) for some i in [i0, i1]?  The indices run
// a, a+1, ... (mod M) from a = (l0 + i0) mod M: valid iff the first is (< P) or the run wraps to 0.
__device__ __forceinline__ bool touches(int l0, int i0, int i1, int M, int P)
{
    int a = l0 + i0; if (a >= M) a -= M;
    return (a < P) || (a + (i1 - i0) >= M);
}

// cyclic range of bins that can hold particles whose support meets [X0, X0 + T)
__device__ __forceinline__ void bin_span(int X0, int T, const SeGeom &g, int &b0, int &nb)
{
    int len = T + g.P - 1;                          // base indices i0 in [X0 - P/2, X0 + T + P/2 - 2]
    if (len + SE_BIN > g.M) { b0 = 0; nb = g.nbin; return; }
    int lo = X0 - g.P / 2;       if (lo < 0) lo += g.M;
    int hi = X0 + T + g.P / 2 - 2; if (hi >= g.M) hi -= g.M;
    int blo = lo / SE_BIN, bhi = hi / SE_BIN;
    b0 = blo;
    nb = bhi - blo; if (nb < 0) nb += g.nbin;
    nb += 1;
}

template <typename Real, bool SPREAD>
__global__ void __launch_bounds__(SE_GRID_THREADS)
k_grid(SeGeom g, const short4 *__restrict__ anchor, const Real *__restrict__ wtab,
       const Real *__restrict__ fs, const int *__restrict__ bin_start,
       Real *__restrict__ grid, Real *__restrict__ uF)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    GridSmem<Real> &S = *reinterpret_cast<GridSmem<Real> *>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int M = g.M, P = g.P;
    const int ntz = (M + SE_TZ - 1) / SE_TZ, nty = (M + SE_TY - 1) / SE_TY;
    const int tz = blockIdx.x % ntz, ty = (blockIdx.x / ntz) % nty, tx = blockIdx.x / (ntz * nty);
    const int X0 = tx * SE_TX, Y0 = ty * SE_TY, Z0 = tz * SE_TZ;
    // thread -> column: warp covers 4 (x) x 8 (y); 4 x 2 warps cover 16 x 16
    const int wx0 = (warp >> 1) * 4, wy0 = (warp & 1) * 8;
    const int ti = wx0 + (lane >> 3), tj = wy0 + (lane & 7);
    const size_t M3 = (size_t)M * M * M;
    const bool col_ok = (X0 + ti < M) && (Y0 + tj < M);
    const size_t col = ((size_t)(X0 + ti) * M + (Y0 + tj)) * M + Z0;

    Real acc[3][SE_TZ];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int k = 0; k < SE_TZ; ++k) {
            if (SPREAD) acc[c][k] = 0;
            else acc[c][k] = (col_ok && Z0 + k < M) ? grid[c * M3 + col + k] : (Real)0;
        }

    // ---- candidate runs -------------------------------------------------------------------
    int bx0, nbx, by0, nby, bz0, nbz;
    bin_span(X0, SE_TX, g, bx0, nbx);
    bin_span(Y0, SE_TY, g, by0, nby);
    bin_span(Z0, SE_TZ, g, bz0, nbz);
    const int ncol = nbx * nby;                       // <= 64
    if (tid < ncol) {
        int bx = bx0 + tid / nby; if (bx >= g.nbin) bx -= g.nbin;
        int by = by0 + tid % nby; if (by >= g.nbin) by -= g.nbin;
        int base = (bx * g.nbin + by) * g.nbin;
        int z1 = min(bz0 + nbz, g.nbin);
        int b = bin_start[base + bz0], e = bin_start[base + z1];
        S.run_beg[2 * tid] = b;
        S.run_ofs[2 * tid + 1] = e - b;               // lengths first, scanned below
        int rem = bz0 + nbz - g.nbin;                 // wrapped part [0, rem)
        int b2 = bin_start[base], e2 = rem > 0 ? bin_start[base + rem] : b2;
        S.run_beg[2 * tid + 1] = b2;
        S.run_ofs[2 * tid + 2] = e2 - b2;
    }
    if (tid == 0) { S.run_ofs[0] = 0; S.nrun = 2 * ncol; }
    __syncthreads();
    if (warp == 0) {                                  // inclusive scan of up to 128 lengths
        int nr = 2 * ncol;
        int v[4], t = 0;
#pragma unroll
        for (int q = 0; q < 4; ++q) { int r = lane * 4 + q; v[q] = (r < nr) ? S.run_ofs[r + 1] : 0; t += v[q]; }
        int inc = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
        int run = inc - t;
#pragma unroll
        for (int q = 0; q < 4; ++q) { int r = lane * 4 + q; run += v[q]; if (r < nr) S.run_ofs[r + 1] = run; }
    }
    __syncthreads();
    const int nrun = S.nrun;
    const int total = S.run_ofs[nrun];

    for (int base = 0; base < total; base += SE_ROUND) {
        // ---- test SE_ROUND candidates (threads 0..127) ------------------------------------
        bool ok = false;
        int pidx = 0;
        short l0x = 0, l0y = 0, l0z = 0;
        if (tid < SE_ROUND && base + tid < total) {
            int v = base + tid;
            int lo = 0, hi = nrun;                     // the run r with run_ofs[r] <= v < run_ofs[r+1]
            while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (S.run_ofs[mid] <= v) lo = mid; else hi = mid; }
            pidx = S.run_beg[lo] + (v - S.run_ofs[lo]);
            short4 a = anchor[pidx];
            int lx = X0 - a.x; if (lx < 0) lx += M;
            int ly = Y0 - a.y; if (ly < 0) ly += M;
            int lz = Z0 - a.z; if (lz < 0) lz += M;
            ok = touches(lx, 0, SE_TX - 1, M, P) && touches(ly, 0, SE_TY - 1, M, P) &&
                 touches(lz, 0, SE_TZ - 1, M, P);
            l0x = (short)lx; l0y = (short)ly; l0z = (short)lz;
        }
        {
            unsigned m = __ballot_sync(0xffffffffu, ok);
            if (lane == 0) S.acc_cnt[warp] = __popc(m);
            __syncthreads();
            if (ok) {
                int slot = __popc(m & ((1u << lane) - 1u));
                for (int q = 0; q < warp; ++q) slot += S.acc_cnt[q];
                S.pidx[slot] = pidx;
                S.lst[slot][0] = l0x; S.lst[slot][1] = l0y; S.lst[slot][2] = l0z;
                if (!SPREAD) { S.U[slot][0] = 0; S.U[slot][1] = 0; S.U[slot][2] = 0; }
            }
        }
        __syncthreads();
        const int na = S.acc_cnt[0] + S.acc_cnt[1] + S.acc_cnt[2] + S.acc_cnt[3];

        // ---- build tables: W1, W2 slices (+ f_c W3 products or W3 slice) ---------------------
        {
            constexpr int NW = SE_TX + SE_TY;          // 32 entries of W1|W2 per particle
            for (int it = tid; it < na * NW; it += SE_GRID_THREADS) {
                int a = it / NW, e = it - a * NW;
                int d = e >= SE_TX, i = d ? e - SE_TX : e;
                int l = S.lst[a][d] + i; if (l >= M) l -= M;
                Real w = (l < P) ? wtab[((size_t)S.pidx[a] * 3 + d) * P + l] : (Real)0;
                if (d) S.W2[a][i] = w; else S.W1[a][i] = w;
            }
            constexpr int NG = SPREAD ? 3 * SE_TZ : SE_TZ;
            for (int it = tid; it < na * NG; it += SE_GRID_THREADS) {
                int a = it / NG, e = it - a * NG;
                int c = e / SE_TZ, k = e - c * SE_TZ;
                int l = S.lst[a][2] + k; if (l >= M) l -= M;
                Real w = (l < P) ? wtab[((size_t)S.pidx[a] * 3 + 2) * P + l] : (Real)0;
                if (SPREAD) w *= fs[(size_t)S.pidx[a] * 3 + c];
                S.G[a][e] = w;
            }
        }
        // ---- per-warp list of the particles that touch this warp's 4 x 8 patch ---------------
        {
            int cnt = 0;
            for (int a0 = 0; a0 < na; a0 += 32) {
                int a = a0 + lane;
                bool hit = false;
                if (a < na)
                    hit = touches(S.lst[a][0], wx0, wx0 + 3, M, P) && touches(S.lst[a][1], wy0, wy0 + 7, M, P);
                unsigned m = __ballot_sync(0xffffffffu, hit);
                if (hit) S.wlist[warp][cnt + __popc(m & ((1u << lane) - 1u))] = (unsigned char)a;
                cnt += __popc(m);
            }
            if (lane == 0) S.wcnt[warp] = cnt;
        }
        __syncthreads();

        // ---- accumulate -------------------------------------------------------------------
        const int cnt = S.wcnt[warp];
        if (SPREAD) {
            for (int q = 0; q < cnt; ++q) {
                const int a = S.wlist[warp][q];
                const Real w12 = S.W1[a][ti] * S.W2[a][tj];
                const Real *G = S.G[a];
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int k = 0; k < SE_TZ; ++k) acc[c][k] = fma(w12, G[c * SE_TZ + k], acc[c][k]);
            }
        } else {
            for (int q = 0; q < cnt; ++q) {
                const int a = S.wlist[warp][q];
                const Real w12 = S.W1[a][ti] * S.W2[a][tj];
                const Real *W3 = S.G[a];
                Real s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
                for (int k = 0; k < SE_TZ; ++k) {
                    s0 = fma(W3[k], acc[0][k], s0);
                    s1 = fma(W3[k], acc[1][k], s1);
                    s2 = fma(W3[k], acc[2][k], s2);
                }
                s0 *= w12; s1 *= w12; s2 *= w12;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    s0 += __shfl_xor_sync(0xffffffffu, s0, o);
                    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
                    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
                }
                if (lane == 0) {
                    atomicAdd(&S.U[a][0], s0);
                    atomicAdd(&S.U[a][1], s1);
                    atomicAdd(&S.U[a][2], s2);
                }
            }
        }
        __syncthreads();
        if (!SPREAD) {
            for (int it = tid; it < na * 3; it += SE_GRID_THREADS) {
                int a = it / 3, c = it - 3 * a;
                Real v = S.U[a][c];
                if (v != (Real)0) atomicAdd(&uF[(size_t)S.pidx[a] * 3 + c], v);
            }
            __syncthreads();
        }
    }

    if (SPREAD && col_ok) {
        const Real cw = (Real)g.cw;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int k = 0; k < SE_TZ; ++k)
                if (Z0 + k < M) grid[c * M3 + col + k] = cw * acc[c][k];
    }
}

template <typename Real, bool SPREAD>
cudaError_t grid_impl(se_plan *p, cudaStream_t s, bool prepare = false)
{
    SeGeom g = p->g;
    const SeSet &Q = SPREAD ? p->S : p->T;                     // P2G spreads the sources, G2P gathers at the targets
    g.N = Q.n;
    size_t smem = sizeof(GridSmem<Real>);
    auto kern = k_grid<Real, SPREAD>;
    if (prepare) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int ntz = (g.M + SE_TZ - 1) / SE_TZ, nty = (g.M + SE_TY - 1) / SE_TY, ntx = (g.M + SE_TX - 1) / SE_TX;
    if (!SPREAD) {
        cudaError_t e = cudaMemsetAsync(p->uF, 0, (size_t)g.N * 3 * sizeof(Real), s);
        if (e != cudaSuccess) return e;
    }
    kern<<<(unsigned)(ntx * nty * ntz), SE_GRID_THREADS, smem, s>>>(
        g, Q.anchor, (const Real *)Q.wtab, (const Real *)Q.fs_grid, Q.bin_start, (Real *)p->grid,
        (Real *)p->uF);
    p->launches += 1;
    return cudaGetLastError();
}

}  // namespace

cudaError_t se_launch_p2g(se_plan *p, cudaStream_t s)
{
    if (p->g.grid_mode == 2) return se_launch_mma_p2g(p, s);
    return p->precision == SE_FP64 ? grid_impl<double, true>(p, s) : grid_impl<float, true>(p, s);
}

cudaError_t se_launch_g2p(se_plan *p, cudaStream_t s)
{
    if (p->g.grid_mode == 2) return se_launch_mma_g2p(p, s);
    return p->precision == SE_FP64 ? grid_impl<double, false>(p, s) : grid_impl<float, false>(p, s);
}

cudaError_t se_prepare_grid(se_plan *p)
{
    if (p->g.grid_mode == 2) return se_prepare_mma(p);
    cudaError_t e = p->precision == SE_FP64 ? grid_impl<double, true>(p, nullptr, true) : grid_impl<float, true>(p, nullptr, true);
    if (e != cudaSuccess) return e;
    return p->precision == SE_FP64 ? grid_impl<double, false>(p, nullptr, true) : grid_impl<float, false>(p, nullptr, true);
}
