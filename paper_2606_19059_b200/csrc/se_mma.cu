// K3 P2G (eq. (2.5)) and K5 G2P (eq. (2.7)) in FP64 as an x-SWEEP whose inner
// product runs on the FP64 tensor-core instruction (mma.sync m8n8k4 f64 -> DMMA), for P = 16 and 24.
//
// Why.  With a Gaussian window at P = 24 both gridding steps are FP64-arithmetic bound: 3 P^3 = 41,472
// FMA per particle against ~1 KB of compulsory traffic.  On B200 DFMA and DMMA
// share one FP64 datapath (36.7 TFLOP/s either way, profiles/r01b_mma_ws.md), but one DFMA warp
// instruction is 32 FMAs while one DMMA is 256 FMAs and holds the pipe for 16 cycles: the tensor form
// leaves ~15 of every 16 issue slots for the bookkeeping that output-stationary gridding needs.
// tcgen05 has no FP64 kind, so mma.sync is the only tensor path for this precision.
//
// The contraction.  Spreading is  H_c[x,y,z] += sum_n (f_nc Wx_n[x]) * (Wy_n[y] Wz_n[z]); for a set of
// 8 (y,z) columns it is a GEMM  C[(x), (yz)] += A[(x), n] B[n, (yz)]  with K = particles.  A warp owns a
// 4 x 4 patch of (y,z) columns = two n-tiles of 2 x 4 and sweeps x: its accumulators are a RING of the P
// planes currently under the window (plane X lives in residue X mod P, P/8 m-tiles of 8 rows) x 3
// components x 2 n-tiles, i.e. 36 doubles per thread at P = 24.  Particles are sorted by
// (anchor plane a_x, a_z / 8, a_y); all particles of one step have the same a_x, touch every residue
// exactly once, and are consumed 4 at a time (the K of m8n8k4).  When the sweep leaves a plane it is
// complete and is written once with plain 16-byte stores: no atomics, no zero-fill, deterministic.
// Efficiency of issued FMAs: 1 in x (no tile overlap in the sweep direction), P/(P+3) in y and in z.
// Gathering is the transpose: the ring holds the grid planes as A-fragments (rows = planes, k = 4 z),
// B = Wy Wz of 8 particles, D[(plane), particle] is contracted with Wx in a short epilogue and reduced
// over the 8 row-lanes with a packed butterfly; per-(particle, block tile) partial sums go to their own
// slot and are added in a fixed order afterwards (bit-reproducible, no atomics).
//
// Staging.  K1 writes one 16-byte aligned RECORD per particle in sorted order:
//   Wx[P] | Wy[P] | Wz[P] | f[3] | (a_y, a_z)          (3P + 4 doubles = 608 bytes at P = 24)
// The candidates of a (block tile, step) are at most 14 contiguous runs of the sorted order, so ONE
// producer warp stages them with one bulk asynchronous copy (cp.async.bulk, the TMA engine) per run,
// completing on the stage's `full` mbarrier; 12 consumer warps test the raw records against their own
// patch, read window values straight from the record (zero outside the support) and release the stage
// through its `empty` mbarrier.  In G2P the producer also adds the consumers' per-warp partial sums in
// fixed order and writes the slot before it refills a stage.
#include <climits>
#include <type_traits>

#include "se_common.cuh"

namespace {

constexpr int CAP = 48;              // candidates per round (one step's candidates, split if more)
constexpr int NST = 4;               // stages
constexpr int ZBW = SE_MMA_ZBIN;     // z-bin width of the sort key
constexpr int NWY = SE_MMA_NWY, NWZ = SE_MMA_NWZ;

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, int parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// bulk asynchronous copy global -> shared (TMA engine); bytes % 16 == 0, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

template <int P>
struct Cfg {
    static constexpr int NCW = NWY * NWZ;                      // consumer warps
    static constexpr int NT = (NCW + 1) * 32;                  // + one producer warp
    static constexpr int BY = 4 * NWY, BZ = 4 * NWZ;           // block tile (columns)
    static constexpr int MT = P / 8;                           // m-tiles in the ring
    static constexpr int REC = SE_MMA_REC(P);                  // doubles per record
    static constexpr int OY = P, OZ = 2 * P, OF = 3 * P, OM = 3 * P + 3;
    static constexpr int NSB = (P + BY - 2) / BY + 2, NSC = (P + BZ - 2) / BZ + 2;   // block tiles a window can meet
    static_assert(P % 8 == 0 && (REC % 2) == 0, "layout");
};

template <int P, bool SPREAD>
struct alignas(16) Stage {
    typedef Cfg<P> C;
    double rec[CAP + 1][C::REC];             // [CAP] stays all-zero: the padding record
    double U[SPREAD ? 1 : CAP][C::NCW][3];   // G2P: per-warp partial sums of the round
    int pidx[CAP];                           // sorted index of the candidate (G2P slot write-out)
    int s, na;                               // step (anchor plane, unwrapped) and candidate count
};

template <int P, bool SPREAD>
struct alignas(16) Smem {
    typedef Cfg<P> C;
    Stage<P, SPREAD> st[NST];
    uint64_t full[NST], empty[NST];
    unsigned char wlist[C::NCW][CAP + 8];
};

__device__ __forceinline__ int modM(int v, int M) { v %= M; return v < 0 ? v + M : v; }

// does the window [0, P) (indices mod M) meet columns T0 .. T0 + n - 1, given l0 = (T0 - anchor) mod M ?
__device__ __forceinline__ bool meets(int l0, int n, int M, int P) { return n > 0 && (l0 < P || l0 + n - 1 >= M); }

// window value W[(l0 + i) mod M] of a record row, zero outside the support
__device__ __forceinline__ double wval(const double *w, int l0, int i, int M, int P)
{
    int l = l0 + i; if (l >= M) l -= M;
    return l < P ? w[l] : 0.0;
}

template <int P, bool SPREAD>
__global__ void __launch_bounds__((NWY * NWZ + 1) * 32, 1)
k_mma(SeGeom g, const double *__restrict__ recs, const int *__restrict__ bin_start, double *__restrict__ grid,
      double *__restrict__ uFpart)
{
    typedef Cfg<P> C;
    constexpr int NCW = C::NCW, BY = C::BY, BZ = C::BZ, MT = C::MT, REC = C::REC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem<P, SPREAD> &S = *reinterpret_cast<Smem<P, SPREAD> *>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int M = g.M, nzb = g.nbin;
    const int ntY = (M + BY - 1) / BY, ntZ = (M + BZ - 1) / BZ;
    const int tz = blockIdx.x % ntZ, ty = (blockIdx.x / ntZ) % ntY, chunk = blockIdx.x / (ntZ * ntY);
    const int nchunk = SPREAD ? g.nchunk : g.nchunk_g2p;
    const int CL = (M + nchunk - 1) / nchunk;
    const int X0 = chunk * CL;
    const int CLen = min(CL, M - X0);
    if (CLen <= 0) return;
    const int Y0 = ty * BY, Z0 = tz * BZ;
    const int s_begin = SPREAD ? X0 - (P - 1) : X0, s_end = X0 + CLen;

    for (int e = tid; e < NST * REC; e += C::NT) S.st[e / REC].rec[CAP][e % REC] = 0.0;
    if (tid == 0)
        for (int i = 0; i < NST; ++i) { mbar_init(&S.full[i], 1); mbar_init(&S.empty[i], NCW); }
    __syncthreads();

    if (warp == NCW) {
        // =================================== PRODUCER ==========================================================
        // candidate rows / z-bins of this block tile (anchors): cyclic [Y0-(P-1), Y0+BY-1], [Z0-(P-1), Z0+BZ-1]
        const int leny = min(BY + P - 1, M);
        const int ylo = modM(Y0 - (P - 1), M);
        int zb0, nzbins;
        {
            const int len = BZ + P - 1;
            if (len + ZBW > M) { zb0 = 0; nzbins = nzb; }
            else {
                const int lo = modM(Z0 - (P - 1), M), hi = modM(Z0 + BZ - 1, M);
                zb0 = lo / ZBW;
                nzbins = hi / ZBW - zb0; if (nzbins < 0) nzbins += nzb;
                nzbins += 1;
            }
        }
        // Runs of one step: (z-bin k, row-range piece) -> 16 lanes per step, two steps per walk iteration
        // (at most 7 z-bins: BZ + P - 1 + ZBW - 1 <= 8 * 7, and grids with M < BZ + P - 1 + ZBW have <= 7 bins).
        static_assert((BZ + P - 1 + ZBW - 2) / ZBW + 1 <= 8, "runs per step");
        const int nrun = 2 * nzbins;
        const int sl = lane >> 4, rl = lane & 15;
        int rcount = 0;                                              // rounds issued so far

        // G2P: add the consumers' partial sums of the round that last used stage `sg`, one slot per block tile
        auto writeout = [&](Stage<P, SPREAD> &T) {
            if (SPREAD) return;
            const int n3 = T.na * 3;
            for (int it = lane; it < n3; it += 32) {
                const int a = it / 3, c = it - 3 * a;
                const int2 an = *reinterpret_cast<const int2 *>(&T.rec[a][C::OM]);
                const int ly = modM(Y0 - an.x, M), lz = modM(Z0 - an.y, M);
                const bool hit = meets(ly, min(BY, M - Y0), M, P) && meets(lz, min(BZ, M - Z0), M, P);
                const int rb = modM(ty - an.x / BY, ntY), rc = modM(tz - an.y / BZ, ntZ);
                if (hit && rb < C::NSB && rc < C::NSC) {
                    double sum = 0.0;
#pragma unroll
                    for (int w = 0; w < NCW; ++w) sum += T.U[a][w][c];
                    uFpart[((size_t)(rb * C::NSC + rc) * g.N + T.pidx[a]) * 3 + c] = sum;
                }
            }
        };
        // wait until the consumers have released stage sg (if it was used), flush its sums, make it ours again
        auto acquire = [&](int r) {
            const int sg = r & (NST - 1);
            if (r >= NST) {
                mbar_wait(&S.empty[sg], ((r / NST) - 1) & 1);
                writeout(S.st[sg]);
                __syncwarp();
            }
        };

        {
            for (int sb = s_begin; sb < s_end; sb += 2) {
                const int s = sb + sl;
                int beg = 0, len = 0;
                if (s < s_end && rl < nrun) {
                    const int k = rl >> 1, piece = rl & 1;
                    int zb = zb0 + k; if (zb >= nzb) zb -= nzb;
                    const int base = (modM(s, M) * nzb + zb) * M;
                    int r0, r1;                                      // rows [r0, r1)
                    if (piece == 0) { r0 = ylo; r1 = min(ylo + leny, M); }
                    else { r0 = 0; r1 = max(ylo + leny - M, 0); }
                    beg = __ldg(&bin_start[base + r0]);
                    len = __ldg(&bin_start[base + r1]) - beg;
                }
                // exclusive prefix of len over the 16 lanes of the step
                int inc = len;
#pragma unroll
                for (int o = 1; o < 16; o <<= 1) {
                    const int y = __shfl_up_sync(0xffffffffu, inc, o, 16);
                    if (rl >= o) inc += y;
                }
                const int ofs = inc - len;
                for (int k = 0; k < 2 && sb + k < s_end; ++k) {
                    const int total = __shfl_sync(0xffffffffu, inc, 16 * k + 15);
                    for (int first = 0; first < total; first += CAP, ++rcount) {
                        const int na = min(CAP, total - first);
                        acquire(rcount);
                        Stage<P, SPREAD> &T = S.st[rcount & (NST - 1)];
                        uint64_t *bar = &S.full[rcount & (NST - 1)];
                        if (lane == 0) {
                            T.s = sb + k; T.na = na;
                            mbar_arrive_expect_tx(bar, (unsigned)(na * REC * 8));
                        }
                        __syncwarp();
                        if (sl == k) {
                            const int lo = max(first, ofs), hi = min(first + na, ofs + len);
                            if (lo < hi) {
                                const int src = beg + (lo - ofs);
                                bulk_g2s(T.rec[lo - first], recs + (size_t)src * REC, (unsigned)((hi - lo) * REC * 8), bar);
                                if (!SPREAD)
                                    for (int v = lo; v < hi; ++v) T.pidx[v - first] = src + (v - lo);
                            }
                        }
                    }
                }
            }
        }
        // terminal round: lets the consumers finish the sweep
        {
            acquire(rcount);
            Stage<P, SPREAD> &T = S.st[rcount & (NST - 1)];
            if (lane == 0) { T.s = s_end; T.na = 0; mbar_arrive(&S.full[rcount & (NST - 1)]); }
            ++rcount;
        }
        // G2P: slots of the rounds still in flight
        if (!SPREAD)
            for (int r = max(rcount - NST, 0); r < rcount; ++r) {
                const int sg = r & (NST - 1);
                mbar_wait(&S.empty[sg], (r / NST) & 1);
                writeout(S.st[sg]);
                __syncwarp();
            }
        return;
    }

    // ======================================= CONSUMER ==============================================================
    const int gq = lane >> 2, tq = lane & 3;
    const int wy0 = 4 * (warp / NWZ), wz0 = 4 * (warp % NWZ);       // warp patch inside the block tile
    const int Yw = Y0 + wy0, Zw = Z0 + wz0;
    const int nyw = min(4, M - Yw), nzw = min(4, M - Zw);           // valid rows / columns of the patch
    const size_t MM = (size_t)M * M, M3 = MM * M;

    // ring: P2G  acc[mt][c][j]  = C fragment of n-tile j (rows 2j, 2j+1 of the patch; columns 2(tq&1), +1)
    //       G2P  acc[mt][c][ky] = A fragments (row ky of the patch, column tq), two k-steps per double pair
    double acc[MT][3][2][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int j = 0; j < 2; ++j) acc[mt][c][j][0] = acc[mt][c][j][1] = 0.0;

    // ---- P2G: this lane's C columns: n = 2 tq, 2 tq + 1 -> y = 2j + (tq >> 1), z = 2 (tq & 1) + {0, 1}
    const int cyl = tq >> 1, czl = 2 * (tq & 1);
    const bool cz_ok = czl < nzw;                                    // M, Zw even: the pair is valid together
    const size_t colS = (size_t)(Yw + cyl) * M + (Zw + czl);
    auto flush_mt = [&](auto mtc, int X, bool valid) {
        constexpr int mt = decltype(mtc)::value;
        const size_t off = (size_t)modM(X, M) * MM + colS;
        const double cw = g.cw;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (valid && 2 * j + cyl < nyw)
                    *reinterpret_cast<double2 *>(&grid[c * M3 + off + (size_t)(2 * j) * M]) =
                        make_double2(cw * acc[mt][c][j][0], cw * acc[mt][c][j][1]);
                acc[mt][c][j][0] = acc[mt][c][j][1] = 0.0;
            }
    };
    auto flush = [&](int X) {
        const int r = modM(X, P);
        if (gq != (r & 7)) return;
        const bool valid = cz_ok && X >= X0;
        switch (r >> 3) {
        case 0: flush_mt(std::integral_constant<int, 0>{}, X, valid); break;
        case 1: flush_mt(std::integral_constant<int, 1>{}, X, valid); break;
        case 2: if constexpr (MT > 2) flush_mt(std::integral_constant<int, 2>{}, X, valid); break;
        case 3: if constexpr (MT > 3) flush_mt(std::integral_constant<int, 3>{}, X, valid); break;
        }
    };
    // ---- G2P: this lane's A elements: plane row gq, k = tq -> column z = tq of patch row ky
    const bool gz_ok = tq < nzw;
    const size_t colG = (size_t)Yw * M + (Zw + tq);
    double pre[3][4];                                                // plane prefetched one step ahead
    int pre_X = INT_MIN;
    auto fetch_plane = [&](int X) {                                  // issue the loads of plane X into `pre`
        pre_X = X;
        if (gq != (modM(X, P) & 7)) return;
        const size_t off = (size_t)modM(X, M) * MM + colG;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int ky = 0; ky < 4; ++ky)
                pre[c][ky] = (gz_ok && ky < nyw) ? __ldg(&grid[c * M3 + off + (size_t)ky * M]) : 0.0;
    };
    auto commit_mt = [&](auto mtc) {
        constexpr int mt = decltype(mtc)::value;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            acc[mt][c][0][0] = pre[c][0]; acc[mt][c][0][1] = pre[c][1];
            acc[mt][c][1][0] = pre[c][2]; acc[mt][c][1][1] = pre[c][3];
        }
    };
    auto commit_plane = [&]() {                                      // move `pre` into its residue of the ring
        const int r = modM(pre_X, P);
        if (gq != (r & 7)) return;
        switch (r >> 3) {
        case 0: commit_mt(std::integral_constant<int, 0>{}); break;
        case 1: commit_mt(std::integral_constant<int, 1>{}); break;
        case 2: if constexpr (MT > 2) commit_mt(std::integral_constant<int, 2>{}); break;
        case 3: if constexpr (MT > 3) commit_mt(std::integral_constant<int, 3>{}); break;
        }
    };

    int cur = s_begin;            // P2G: first plane not yet flushed; G2P: first plane not yet in the ring
    for (int r = 0;; ++r) {
        const int sg = r & (NST - 1);
        Stage<P, SPREAD> &T = S.st[sg];
        mbar_wait(&S.full[sg], (r / NST) & 1);
        const int s = T.s, na = T.na;
        if (s >= s_end) {                                            // terminal round
            if (SPREAD) while (cur < s_end) { flush(cur); ++cur; }
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.empty[sg]);
            break;
        }
        if (SPREAD) {
            while (cur < s) { flush(cur); ++cur; }
        } else {
            // planes s .. s+P-1 must be in the ring; plane cur-1 may be waiting in `pre`
            if (cur < s) { cur = s; pre_X = INT_MIN; }               // planes nobody gathers from are skipped
            while (cur < s + P) {
                if (pre_X != cur) fetch_plane(cur);
                commit_plane();
                ++cur;
            }
            if (pre_X != s + P) fetch_plane(s + P);                  // next step's new plane, consumed next round
        }

        // ---- this warp's candidates, padded to whole K-groups with the zero record -------------------------
        int cnt = 0;
        for (int a0 = 0; a0 < na; a0 += 32) {
            const int a = a0 + lane;
            bool hit = false;
            if (a < na) {
                const int2 an = *reinterpret_cast<const int2 *>(&T.rec[a][C::OM]);
                int ly = Yw - an.x; if (ly < 0) ly += M;
                int lz = Zw - an.y; if (lz < 0) lz += M;
                hit = meets(ly, nyw, M, P) && meets(lz, nzw, M, P);
                if (!SPREAD && !hit) { T.U[a][warp][0] = 0.0; T.U[a][warp][1] = 0.0; T.U[a][warp][2] = 0.0; }
            }
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) S.wlist[warp][cnt + __popc(m & ((1u << lane) - 1u))] = (unsigned char)a;
            cnt += __popc(m);
        }
        constexpr int GRP = SPREAD ? 4 : 8;
        const int padded = (cnt + GRP - 1) & ~(GRP - 1);
        if (lane < padded - cnt) S.wlist[warp][cnt + lane] = (unsigned char)CAP;
        __syncwarp();

        // Wx index of this lane's ring rows: plane s + l <-> residue (s + l) mod P
        const int rs = modM(s, P);
        int lx[MT];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) { int l = 8 * mt + gq - rs; lx[mt] = l < 0 ? l + P : l; }

        if (SPREAD) {
            // B[k = tq][n = gq]: particle tq of the group, column n -> y = 2j + (gq >> 2), z = gq & 3
            const int byl = gq >> 2, bzl = gq & 3;
            for (int q = 0; q < padded; q += 4) {
                const double *rp = T.rec[S.wlist[warp][q + tq]];
                const double2 f01 = *reinterpret_cast<const double2 *>(&rp[C::OF]);
                const double2 f2m = *reinterpret_cast<const double2 *>(&rp[C::OF + 2]);
                const long long an = __double_as_longlong(f2m.y);                // (a_y, a_z)
                int ly = Yw - (int)(an & 0xffffffffll); if (ly < 0) ly += M;
                int lz = Zw - (int)(an >> 32); if (lz < 0) lz += M;
                const double wzv = wval(rp + C::OZ, lz, bzl, M, P);
                const double b0 = wval(rp + C::OY, ly, byl, M, P) * wzv;
                const double b1 = wval(rp + C::OY, ly, byl + 2, M, P) * wzv;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const double wx = rp[lx[mt]];
                    const double a0 = f01.x * wx, a1 = f01.y * wx, a2 = f2m.x * wx;
                    dmma(acc[mt][0][0], a0, b0); dmma(acc[mt][0][1], a0, b1);
                    dmma(acc[mt][1][0], a1, b0); dmma(acc[mt][1][1], a1, b1);
                    dmma(acc[mt][2][0], a2, b0); dmma(acc[mt][2][1], a2, b1);
                }
            }
        } else {
            // B[k = tq][n = gq]: column z = tq of patch row ky, particle gq of the group
            for (int q = 0; q < padded; q += 8) {
                const double *rp = T.rec[S.wlist[warp][q + gq]];
                const int2 an = *reinterpret_cast<const int2 *>(&rp[C::OM]);
                int ly = Yw - an.x; if (ly < 0) ly += M;
                int lz = Zw - an.y; if (lz < 0) lz += M;
                const double wzv = wval(rp + C::OZ, lz, tq, M, P);
                double b[4];
#pragma unroll
                for (int ky = 0; ky < 4; ++ky) b[ky] = wval(rp + C::OY, ly, ky, M, P) * wzv;
                const int a0 = S.wlist[warp][q + 2 * tq], a1 = S.wlist[warp][q + 2 * tq + 1];
                double p0[3] = {0.0, 0.0, 0.0}, p1[3] = {0.0, 0.0, 0.0};
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const double wx0 = T.rec[a0][lx[mt]], wx1 = T.rec[a1][lx[mt]];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double d[2] = {0.0, 0.0};
                        dmma(d, acc[mt][c][0][0], b[0]); dmma(d, acc[mt][c][0][1], b[1]);
                        dmma(d, acc[mt][c][1][0], b[2]); dmma(d, acc[mt][c][1][1], b[3]);
                        p0[c] = fma(d[0], wx0, p0[c]);
                        p1[c] = fma(d[1], wx1, p1[c]);
                    }
                }
                // sum over the 8 row-lanes (lane bits 2..4); lanes gq = 0 end with particle 2 tq, gq = 4 with 2 tq + 1
                const bool hi = lane & 16;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double snd = hi ? p0[c] : p1[c];
                    double v = hi ? p1[c] : p0[c];
                    v += __shfl_xor_sync(0xffffffffu, snd, 16);
                    v += __shfl_xor_sync(0xffffffffu, v, 8);
                    v += __shfl_xor_sync(0xffffffffu, v, 4);
                    p0[c] = v;
                }
                if ((lane & 12) == 0) {
                    const int aa = hi ? a1 : a0;
                    if (aa < CAP) { T.U[aa][warp][0] = p0[0]; T.U[aa][warp][1] = p0[1]; T.U[aa][warp][2] = p0[2]; }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.empty[sg]);
    }
}

// u^F (grid-sorted order) = fixed-order sum of the slots the particle's window actually meets
template <int P>
__global__ void k_reduce_slots(SeGeom g, const short4 *__restrict__ anchor, const double *__restrict__ part,
                               double *__restrict__ uF)
{
    typedef Cfg<P> C;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    const int M = g.M;
    const int ntY = (M + C::BY - 1) / C::BY, ntZ = (M + C::BZ - 1) / C::BZ;
    const short4 a = anchor[i];
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int rb = 0; rb < C::NSB && rb < ntY; ++rb) {
        const int ty = (a.y / C::BY + rb) % ntY, Y0 = ty * C::BY;
        if (!meets(modM(Y0 - a.y, M), min(C::BY, M - Y0), M, P)) continue;
        for (int rc = 0; rc < C::NSC && rc < ntZ; ++rc) {
            const int tz = (a.z / C::BZ + rc) % ntZ, Z0 = tz * C::BZ;
            if (!meets(modM(Z0 - a.z, M), min(C::BZ, M - Z0), M, P)) continue;
            const double *q = part + ((size_t)(rb * C::NSC + rc) * g.N + i) * 3;
            s0 += q[0]; s1 += q[1]; s2 += q[2];
        }
    }
    uF[3 * i + 0] = s0; uF[3 * i + 1] = s1; uF[3 * i + 2] = s2;
}

template <int P, bool SPREAD>
cudaError_t launch(se_plan *p, cudaStream_t s)
{
    typedef Cfg<P> C;
    const SeGeom &g = p->g;
    static bool attr_set = false;
    const size_t smem = sizeof(Smem<P, SPREAD>);
    auto kern = k_mma<P, SPREAD>;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int ntY = (g.M + C::BY - 1) / C::BY, ntZ = (g.M + C::BZ - 1) / C::BZ;
    const int nchunk = SPREAD ? g.nchunk : g.nchunk_g2p;
    kern<<<(unsigned)(nchunk * ntY * ntZ), C::NT, smem, s>>>(g, (const double *)p->wtab, p->bin_start,
                                                             (double *)p->grid, (double *)p->uFpart);
    p->launches += 1;
    if (!SPREAD) {
        k_reduce_slots<P><<<(unsigned)((g.N + 255) / 256), 256, 0, s>>>(g, p->anchor, (const double *)p->uFpart,
                                                                        (double *)p->uF);
        p->launches += 1;
    }
    return cudaGetLastError();
}

template <bool SPREAD>
cudaError_t dispatch(se_plan *p, cudaStream_t s)
{
    switch (p->g.P) {
    case 24: return launch<24, SPREAD>(p, s);
    case 16: return launch<16, SPREAD>(p, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace

bool se_mma_supported(int P, int precision) { return precision == SE_FP64 && (P == 24 || P == 16); }
int se_mma_slots(int P) { return P == 24 ? Cfg<24>::NSB * Cfg<24>::NSC : Cfg<16>::NSB * Cfg<16>::NSC; }
cudaError_t se_launch_mma_p2g(se_plan *p, cudaStream_t s) { return dispatch<true>(p, s); }
cudaError_t se_launch_mma_g2p(se_plan *p, cudaStream_t s) { return dispatch<false>(p, s); }
