// K3 P2G (eq. (2.5)) and K5 G2P (eq. (2.7)) as a SWEEP along x with a
// rotating register window -- the B200 design for the window sizes that matter (P = 12, 16, 24).
//
// Why not the paper's kernels: P2G-hybrid flushes per-thread partial sums with
// O(27 N) global atomics and computes 27 (P/2)^3 points for P^3 useful ones; thread-per-target G2P
// re-reads P^3 grid values per target through L2.  With a Gaussian at P = 24 both steps
// are FP64-FMA bound (3 P^3 FMA per particle against ~1 KB of compulsory traffic), so what counts is
// the fraction of issued FMAs that are useful and the number of shared-memory operands per FMA.
//
// Scheme.  Memory order of the grid is (x, y, z), z fastest.  Particles are sorted by
// (base plane ix, y-bin, z-bin) with 4 x 4 bins (K1).  A block owns a TB x TC patch of (y, z) columns
// and walks x plane by plane over a chunk of the grid.  A warp owns a 4 x (2 LC) sub-patch; its 32 lanes
// are NZG "z-groups" x (4 x LC) columns-pairs; a thread keeps, for its 2 adjacent z-columns, R = P/NZG
// of the P planes currently under the window, times 3 components, in registers (36 accumulators at
// P = 24).  The window is a ring: plane t lives in residue t mod P, so a particle whose base plane is
// the current step touches all P residues exactly once and its x-window table is staged in shared
// memory already ROTATED to residue order (and, for P2G, already multiplied by f_c).  Per particle a
// thread issues 2 R 3 FMAs on 3 R + 3 shared operands; every FMA in x is useful (no tile overlap loss
// in the sweep direction), the loss in y, z is (P/(P+3))^2.  When the sweep leaves a plane it is
// complete: P2G writes it once with plain vector stores (no atomics, no zero-fill, deterministic);
// G2P loads the plane entering the window.  G2P reduces the three partial sums over the warp with a
// packed butterfly (6 DADD), over the block's warps through shared memory in fixed order, and writes
// one partial per (particle, tile) into its own slot, summed in fixed order afterwards: no atomics,
// bit-reproducible.
#include "se_common.cuh"

namespace {

constexpr int SLOTS = 64;          // particles staged per round
constexpr int NWARP = 8;
constexpr int NTHREADS = NWARP * 32;
constexpr int MAXRUN = 2 * SE_GSTEPS_MAX * 10;

template <typename Real> struct V2;
template <> struct V2<double> { typedef double2 type; };
template <> struct V2<float> { typedef float2 type; };
template <typename Real> struct V16;
template <> struct V16<double> { typedef double2 type; static constexpr int n = 2; };
template <> struct V16<float> { typedef float4 type; static constexpr int n = 4; };

__device__ __forceinline__ void unpack(const double2 &v, double *o) { o[0] = v.x; o[1] = v.y; }
__device__ __forceinline__ void unpack(const float4 &v, float *o) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }

template <typename Real, int P, int NZG, bool SPREAD>
struct Cfg {
    static constexpr int R = P / NZG;                    // residues (planes) per thread
    static constexpr int XYL = 32 / NZG;                 // column-pair lanes per warp
    static constexpr int LC = XYL / 4;                   // lanes along z
    static constexpr int TB = SE_SWEEP_TB;               // 2 warps x 4 columns in y
    static constexpr int TC = 4 * 2 * LC;                // 4 warps x LC lanes x 2 columns in z
    static constexpr int GV = SPREAD ? 3 * R : R;        // staged x-table values per z-group
    static constexpr int VN = V16<Real>::n;
    static constexpr int GS = (GV + VN - 1) / VN * VN;   // padded to 16 bytes
    static constexpr int EL = TB + TC + (SPREAD ? 3 * P : P);
    static_assert(P % NZG == 0 && 32 % NZG == 0 && XYL % 4 == 0, "lane layout");
};

template <typename Real, int P, int NZG, bool SPREAD>
struct alignas(16) Smem {
    typedef Cfg<Real, P, NZG, SPREAD> C;
    Real G[SLOTS][NZG * C::GS];
    Real Wc[SLOTS][C::TC];
    Real Wb[SLOTS][C::TB];
    Real U[SPREAD ? 1 : SLOTS][NWARP][3];
    int pidx[SLOTS];
    int sid[SLOTS];                  // G2P: partial-sum slot of (particle, this tile), -1 = none
    short lb0[SLOTS], lc0[SLOTS];    // window index of the tile's first column, in [0, M)
    short rot[SLOTS];                // residue of the particle's first window plane
    short srel[SLOTS];               // step - s_lo
    unsigned short wlist[NWARP][SLOTS];
    int wcnt[NWARP];
    int acc_cnt[2];
    int run_beg[MAXRUN];
    int run_ofs[MAXRUN + 1];
};

// does window index (l0 + i) mod M fall inside [0, P) for some i in [i0, i1]?
__device__ __forceinline__ bool touches(int l0, int i0, int i1, int M, int P)
{
    int a = l0 + i0; if (a >= M) a -= M;
    return (a < P) || (a + (i1 - i0) >= M);
}

// cyclic range of 4-wide bins holding every base index whose support meets [X0, X0 + T)
__device__ __forceinline__ void bin_span(int X0, int T, int M, int P, int nbin, int &b0, int &nb)
{
    int len = T + P - 1;
    if (len + SE_SBIN > M) { b0 = 0; nb = nbin; return; }
    int lo = X0 - P / 2;          if (lo < 0) lo += M;
    int hi = X0 + T + P / 2 - 2;  if (hi >= M) hi -= M;
    int blo = lo / SE_SBIN, bhi = hi / SE_SBIN;
    b0 = blo;
    nb = bhi - blo; if (nb < 0) nb += nbin;
    nb += 1;
}

template <typename Real, int P, int NZG, bool SPREAD>
__global__ void __launch_bounds__(NTHREADS, 2)
k_sweep(SeGeom g, const short4 *__restrict__ anchor, const Real *__restrict__ wtab,
        const Real *__restrict__ fs, const int *__restrict__ bin_start,
        Real *__restrict__ grid, Real *__restrict__ uFpart)
{
    typedef Cfg<Real, P, NZG, SPREAD> C;
    typedef typename V2<Real>::type Real2;
    typedef typename V16<Real>::type Vec;
    constexpr int R = C::R, LC = C::LC, TB = C::TB, TC = C::TC, GS = C::GS, XYL = C::XYL;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem<Real, P, NZG, SPREAD> &S = *reinterpret_cast<Smem<Real, P, NZG, SPREAD> *>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int M = g.M, nbin = g.nbin;
    const int ntb = (M + TB - 1) / TB, ntc = (M + TC - 1) / TC;
    const int tci = blockIdx.x % ntc, tbi = (blockIdx.x / ntc) % ntb, chunk = blockIdx.x / (ntc * ntb);
    const int CL = (M + g.nchunk - 1) / g.nchunk;
    const int A0 = chunk * CL;
    const int CLen = min(CL, M - A0);
    if (CLen <= 0) return;
    const int B0 = tbi * TB, C0 = tci * TC;
    // lane -> z-group, column pair
    const int zg = lane / XYL, xl = lane % XYL;
    const int lb = xl / LC, lc = xl % LC;
    const int wb0 = (warp >> 2) * 4, wc0 = (warp & 3) * (2 * LC);
    const int ib = wb0 + lb, ic = wc0 + 2 * lc;              // column (ib, ic), (ib, ic + 1) of the tile
    const bool col_ok = (B0 + ib < M) && (C0 + ic < M);      // M even, ic even: both columns or none
    const size_t M3 = (size_t)M * M * M;
    const size_t col = ((size_t)(B0 + ib)) * M + (C0 + ic);  // + plane * M * M
    const size_t MM = (size_t)M * M;

    // steps: particle base plane of step s is (A0 - shift + s) mod M
    const int shift = SPREAD ? P / 2 : 0;
    const int nsteps = SPREAD ? CLen + P - 1 : CLen;

    Real acc[2][R][3];
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int k = 0; k < R; ++k)
#pragma unroll
            for (int c = 0; c < 3; ++c) acc[j][k][c] = 0;

    // P2G: plane completed by step s (local t = s - (P/2-1)) is written if it lies in the chunk.
    auto flush = [&](int s) {
        const int r = (s + P / 2 + 1) % P;
        const int kz = r % R;
        const bool own = (zg == r / R);
        const bool valid = (s >= P - 1) && (s < P - 1 + CLen) && col_ok;
        const size_t off = (size_t)(A0 + s - (P - 1)) * MM + col;
        const Real cw = (Real)g.cw;
#pragma unroll
        for (int k = 0; k < R; ++k) {
            if (k == kz && own) {
                if (valid) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        Real2 v; v.x = cw * acc[0][k][c]; v.y = cw * acc[1][k][c];
                        *reinterpret_cast<Real2 *>(&grid[c * M3 + off]) = v;
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) { acc[0][k][c] = 0; acc[1][k][c] = 0; }
            }
        }
    };
    // G2P: load local plane t (physical (A0 + t) mod M) into its residue.
    auto load_plane = [&](int t) {
        const int r = (t + P) % P;
        const int kz = r % R;
        const bool own = (zg == r / R);
        int a = A0 + t; if (a < 0) a += M; if (a >= M) a -= M;
        const size_t off = (size_t)a * MM + col;
#pragma unroll
        for (int k = 0; k < R; ++k) {
            if (k == kz && own && col_ok) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    Real2 v = *reinterpret_cast<const Real2 *>(&grid[c * M3 + off]);
                    acc[0][k][c] = v.x; acc[1][k][c] = v.y;
                }
            }
        }
    };

    int cur;
    if (SPREAD) cur = 0;
    else {
        for (int t = -(P / 2 - 1); t <= P / 2 - 1; ++t) load_plane(t);
        cur = -1;
    }

    // bins whose particles can touch the tile
    int bb0, nrb, cb0, ncb;
    bin_span(B0, TB, M, P, nbin, bb0, nrb);
    bin_span(C0, TC, M, P, nbin, cb0, ncb);
    int gsteps = g.gsteps;
    while (gsteps > 1 && 2 * gsteps * nrb > MAXRUN) --gsteps;

    for (int s_lo = 0; s_lo < nsteps; s_lo += gsteps) {
        const int s_hi = min(s_lo + gsteps, nsteps) - 1;
        // ---- candidate runs of this group of planes ---------------------------------------------
        const int ntask = (s_hi - s_lo + 1) * nrb;
        for (int task = tid; task < ntask; task += NTHREADS) {
            int ds = task / nrb, rb = task - ds * nrb;
            int pl = A0 - shift + s_lo + ds;
            pl %= M; if (pl < 0) pl += M;
            int bb = bb0 + rb; if (bb >= nbin) bb -= nbin;
            int base = (pl * nbin + bb) * nbin;
            int z1 = min(cb0 + ncb, nbin);
            int b = bin_start[base + cb0], e = bin_start[base + z1];
            S.run_beg[2 * task] = b;
            S.run_ofs[2 * task + 1] = e - b;
            int rem = cb0 + ncb - nbin;
            int b2 = bin_start[base], e2 = rem > 0 ? bin_start[base + rem] : b2;
            S.run_beg[2 * task + 1] = b2;
            S.run_ofs[2 * task + 2] = e2 - b2;
        }
        if (tid == 0) S.run_ofs[0] = 0;
        __syncthreads();
        const int nrun = 2 * ntask;
        if (warp == 0) {                                    // inclusive scan of the run lengths
            constexpr int PER = (MAXRUN + 31) / 32;
            int v[PER], t = 0;
#pragma unroll
            for (int q = 0; q < PER; ++q) { int r = lane * PER + q; v[q] = (r < nrun) ? S.run_ofs[r + 1] : 0; t += v[q]; }
            int inc = t;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
            int run = inc - t;
#pragma unroll
            for (int q = 0; q < PER; ++q) { int r = lane * PER + q; run += v[q]; if (r < nrun) S.run_ofs[r + 1] = run; }
        }
        __syncthreads();
        const int total = S.run_ofs[nrun];

        for (int base = 0; base < total; base += SLOTS) {
            // ---- test SLOTS candidates (warps 0, 1) ----------------------------------------------
            if (warp < 2) {
                bool ok = false;
                int pidx = 0, lbv = 0, lcv = 0, srel = 0;
                const int v = base + tid;
                if (v < total) {
                    int lo = 0, hi = nrun;              // run r with run_ofs[r] <= v < run_ofs[r+1]
                    while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (S.run_ofs[mid] <= v) lo = mid; else hi = mid; }
                    pidx = S.run_beg[lo] + (v - S.run_ofs[lo]);
                    srel = (lo >> 1) / nrb;
                    short4 a = anchor[pidx];
                    lbv = B0 - a.y; if (lbv < 0) lbv += M;
                    lcv = C0 - a.z; if (lcv < 0) lcv += M;
                    ok = touches(lbv, 0, TB - 1, M, P) && touches(lcv, 0, TC - 1, M, P);
                }
                const unsigned m = __ballot_sync(0xffffffffu, ok);
                if (lane == 0) S.acc_cnt[warp] = __popc(m);
                asm volatile("bar.sync 1, 64;");        // only warps 0 and 1 take part
                if (ok) {
                    int slot = __popc(m & ((1u << lane) - 1u)) + (warp ? S.acc_cnt[0] : 0);
                    S.pidx[slot] = pidx;
                    S.lb0[slot] = (short)lbv; S.lc0[slot] = (short)lcv;
                    S.srel[slot] = (short)srel;
                    S.rot[slot] = (short)((s_lo + srel + P / 2 + 1) % P);
                    if (!SPREAD) {
                        short4 a = anchor[pidx];
                        int rbt = tbi - a.y / TB; if (rbt < 0) rbt += ntb;
                        int rct = tci - a.z / TC; if (rct < 0) rct += ntc;
                        S.sid[slot] = (rbt < SE_NSLOT_B && rct < SE_NSLOT_C) ? rbt * SE_NSLOT_C + rct : -1;
                    }
                }
            }
            __syncthreads();
            const int na = S.acc_cnt[0] + S.acc_cnt[1];

            // ---- tables: y and z slices of the tile, x table rotated to residue order -----------
            for (int it = tid; it < na * C::EL; it += NTHREADS) {
                const int a = it / C::EL, e = it - a * C::EL;
                const size_t wbase = (size_t)S.pidx[a] * 3 * P;
                if (e < TB) {
                    int l = S.lb0[a] + e; if (l >= M) l -= M;
                    S.Wb[a][e] = (l < P) ? wtab[wbase + P + l] : (Real)0;
                } else if (e < TB + TC) {
                    int j = e - TB;
                    int l = S.lc0[a] + j; if (l >= M) l -= M;
                    S.Wc[a][j] = (l < P) ? wtab[wbase + 2 * P + l] : (Real)0;
                } else {
                    int q = e - TB - TC;
                    int r = SPREAD ? q / 3 : q, c = SPREAD ? q - 3 * r : 0;
                    int l = r - S.rot[a]; if (l < 0) l += P;
                    Real w = wtab[wbase + l];
                    if (SPREAD) w *= fs[(size_t)S.pidx[a] * 3 + c];
                    const int z = r / R, k = r - z * R;
                    S.G[a][z * GS + (SPREAD ? k * 3 + c : k)] = w;
                }
            }
            if (!SPREAD)
                for (int it = tid; it < na * NWARP * 3; it += NTHREADS) (&S.U[0][0][0])[it] = 0;
            // ---- per-warp list of the staged particles that touch this warp's columns ------------
            {
                int cnt = 0;
                for (int a0 = 0; a0 < na; a0 += 32) {
                    const int a = a0 + lane;
                    bool hit = false;
                    if (a < na)
                        hit = touches(S.lb0[a], wb0, wb0 + 3, M, P) && touches(S.lc0[a], wc0, wc0 + 2 * LC - 1, M, P);
                    const unsigned m = __ballot_sync(0xffffffffu, hit);
                    if (hit) S.wlist[warp][cnt + __popc(m & ((1u << lane) - 1u))] = (unsigned short)(a | (S.srel[a] << 8));
                    cnt += __popc(m);
                }
                if (lane == 0) S.wcnt[warp] = cnt;
            }
            __syncthreads();

            // ---- accumulate ----------------------------------------------------------------------
            const int cnt = S.wcnt[warp];
            for (int q = 0; q < cnt; ++q) {
                const int e = S.wlist[warp][q];
                const int a = e & 255, sp = s_lo + (e >> 8);
                if (SPREAD) { while (cur < sp) { flush(cur); ++cur; } }
                else { while (cur < sp) { ++cur; load_plane(cur + P / 2); } }
                const Real wb = S.Wb[a][ib];
                const Real2 wc = *reinterpret_cast<const Real2 *>(&S.Wc[a][ic]);
                Real gv[GS];
                const Vec *gp = reinterpret_cast<const Vec *>(&S.G[a][zg * GS]);
#pragma unroll
                for (int v = 0; v < GS / C::VN; ++v) unpack(gp[v], &gv[v * C::VN]);
                if (SPREAD) {
                    const Real w0 = wb * wc.x, w1 = wb * wc.y;
#pragma unroll
                    for (int k = 0; k < R; ++k)
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            acc[0][k][c] = fma(w0, gv[k * 3 + c], acc[0][k][c]);
                            acc[1][k][c] = fma(w1, gv[k * 3 + c], acc[1][k][c]);
                        }
                } else {
                    Real p0[3] = {0, 0, 0}, p1[3] = {0, 0, 0};
#pragma unroll
                    for (int k = 0; k < R; ++k)
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            p0[c] = fma(gv[k], acc[0][k][c], p0[c]);
                            p1[c] = fma(gv[k], acc[1][k][c], p1[c]);
                        }
                    const Real w0 = wb * wc.x, w1 = wb * wc.y;
                    Real v0 = fma(w0, p0[0], w1 * p1[0]);
                    Real v1 = fma(w0, p0[1], w1 * p1[1]);
                    Real v2 = fma(w0, p0[2], w1 * p1[2]);
                    // packed butterfly: 3 values over 32 lanes with 6 adds
                    const bool h16 = lane & 16, h8 = lane & 8;
                    Real snd = h16 ? v0 : v1, kp = h16 ? v1 : v0;
                    kp += __shfl_xor_sync(0xffffffffu, snd, 16);
                    v2 += __shfl_xor_sync(0xffffffffu, v2, 16);
                    snd = h8 ? kp : v2;
                    Real w = h8 ? v2 : kp;
                    w += __shfl_xor_sync(0xffffffffu, snd, 8);
                    w += __shfl_xor_sync(0xffffffffu, w, 4);
                    w += __shfl_xor_sync(0xffffffffu, w, 2);
                    w += __shfl_xor_sync(0xffffffffu, w, 1);
                    if (lane == 0) S.U[a][warp][0] = w;
                    else if (lane == 16) S.U[a][warp][1] = w;
                    else if (lane == 8) S.U[a][warp][2] = w;
                }
            }
            __syncthreads();
            if (!SPREAD) {
                for (int it = tid; it < na * 3; it += NTHREADS) {
                    const int a = it / 3, c = it - 3 * a;
                    Real s = 0;
#pragma unroll
                    for (int w = 0; w < NWARP; ++w) s += S.U[a][w][c];
                    const int sid = S.sid[a];
                    if (sid >= 0) uFpart[((size_t)S.pidx[a] * SE_NSLOT + sid) * 3 + c] = s;
                }
                __syncthreads();
            }
        }
        if (SPREAD) { while (cur <= s_hi) { flush(cur); ++cur; } }
    }
}

template <typename Real>
__global__ void k_reduce_slots(int64_t n3, const Real *__restrict__ part, Real *__restrict__ uF)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n3) return;
    int64_t i = t / 3;
    int c = (int)(t - 3 * i);
    Real s = 0;
#pragma unroll
    for (int q = 0; q < SE_NSLOT; ++q) s += part[(i * SE_NSLOT + q) * 3 + c];
    uF[t] = s;
}

template <typename Real, int P, int NZG, bool SPREAD>
cudaError_t launch(se_plan *p, cudaStream_t s)
{
    typedef Cfg<Real, P, NZG, SPREAD> C;
    const SeGeom &g = p->g;
    static bool attr_set = false;
    const size_t smem = sizeof(Smem<Real, P, NZG, SPREAD>);
    auto kern = k_sweep<Real, P, NZG, SPREAD>;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int ntb = (g.M + C::TB - 1) / C::TB, ntc = (g.M + C::TC - 1) / C::TC;
    if (!SPREAD) {
        cudaError_t e = cudaMemsetAsync(p->uFpart, 0, (size_t)g.N * SE_NSLOT * 3 * sizeof(Real), s);
        if (e != cudaSuccess) return e;
    }
    kern<<<(unsigned)(g.nchunk * ntb * ntc), NTHREADS, smem, s>>>(
        g, p->anchor, (const Real *)p->wtab, (const Real *)p->fs_grid, p->bin_start, (Real *)p->grid,
        (Real *)p->uFpart);
    p->launches += 1;
    if (!SPREAD) {
        int64_t n3 = 3 * g.N;
        k_reduce_slots<Real><<<(unsigned)((n3 + 255) / 256), 256, 0, s>>>(n3, (const Real *)p->uFpart, (Real *)p->uF);
        p->launches += 1;
    }
    return cudaGetLastError();
}

template <bool SPREAD>
cudaError_t dispatch(se_plan *p, cudaStream_t s)
{
    const bool d = p->precision == SE_FP64;
    switch (p->g.P) {
    case 24: return d ? launch<double, 24, 4, SPREAD>(p, s) : launch<float, 24, 4, SPREAD>(p, s);
    case 16: return d ? launch<double, 16, 4, SPREAD>(p, s) : launch<float, 16, 4, SPREAD>(p, s);
    case 12: return d ? launch<double, 12, 2, SPREAD>(p, s) : launch<float, 12, 2, SPREAD>(p, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace

bool se_sweep_supported(int P) { return P == 24 || P == 16 || P == 12; }
cudaError_t se_launch_sweep_p2g(se_plan *p, cudaStream_t s) { return dispatch<true>(p, s); }
cudaError_t se_launch_sweep_g2p(se_plan *p, cudaStream_t s) { return dispatch<false>(p, s); }
