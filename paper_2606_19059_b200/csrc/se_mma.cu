// K3 P2G (eq. (2.5)) and K5 G2P (eq. (2.7)) in FP64 as an x-SWEEP whose inner
// product runs on the FP64 tensor-core instruction (mma.sync m8n8k4 f64 -> DMMA), for every even 4 <= P <= 24 in fp64
// plans and 4 <= P <= 16 in fp32 plans (float grid, double records and accumulators); supports that are not a
// multiple of 8 (P2G) / 4 (G2P) run on the next ring size with zero rows in the records.
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
// Gathering is the transpose: the ring holds the grid planes as B-fragments (k = 4 planes, n = 8 columns),
// A = Wx of 8 particles, E[particle, (yz)] accumulates over the P/4 k-steps and is contracted with Wy Wz
// in a short epilogue (4 FMA per component, 2 shuffles over the 4 column-lanes); per-(particle, block tile)
// partial sums go to their own slot and are added in a fixed order afterwards (bit-reproducible, no atomics).
//
// Staging.  K1 writes 16-byte aligned RECORDS per particle in sorted order (se_common.cuh):
//   spread: c_w f_c Wx[P] (c = x, y, z) | Wy[P] | Wz[P] | (a_y, a_z)     (992 bytes at P = 24)
//   gather: Wx[P] | Wy[P] | Wz[P] | (a_y, a_z)                            (608 bytes at P = 24)
// so that every DMMA operand except the Wy Wz product comes out of shared memory ready-made: an FP64
// multiply in front of a DMMA queues behind the DMMAs in flight on the shared FP64 datapath.
// The candidates of a (block tile, step) are at most 14 contiguous runs of the sorted order, so ONE
// producer warp stages them with one bulk asynchronous copy (cp.async.bulk, the TMA engine) per run,
// completing on the stage's `full` mbarrier; 12 consumer warps (152 registers each after setmaxnreg) test
// the raw records against their own patch, keep a packed hit list (candidate, window index of the patch origin
// in y and z) and read the window values under the patch straight from the staged records (zero outside the
// support); they release the stage through its `empty` mbarrier.  In G2P the other
// three warps of the producer warpgroup add the consumers' per-warp partial sums in fixed order and write
// the slot before the stage is refilled.
#include <climits>
#include <type_traits>

#include "se_common.cuh"

namespace {

#ifndef SE_CAP
#define SE_CAP 48
#endif
#ifndef SE_NST_P2G
#define SE_NST_P2G 3
#endif
#ifndef SE_NST_G2P
#define SE_NST_G2P 5
#endif
constexpr int CAP = SE_CAP;          // candidates per round (one step's candidates, split if more)
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

template <int P, bool SPREAD>
struct Cfg {
    static constexpr int NCW = NWY * NWZ;                      // consumer warps (3 warpgroups)
    static constexpr int NT = (NCW + 4) * 32;                  // + the producer warpgroup
    static constexpr int BY = 4 * NWY, BZ = 4 * NWZ;           // block tile (columns)
    static constexpr int MT = P / 8;                           // m-tiles in the ring
    static constexpr int REC = SPREAD ? SE_MMA_RECS(P) : SE_MMA_RECG(P);   // doubles per record
    static constexpr int OY = SPREAD ? 3 * P : P, OZ = OY + P, OM = OZ + P; // offsets of Wy, Wz, (a_y, a_z)
    static constexpr int NST = SPREAD ? SE_NST_P2G : SE_NST_G2P;   // stages (measured: P2G 4 = 3, G2P 5 > 4)
    static constexpr int GRP = SPREAD ? 4 : 8;                 // candidates per K-group (P2G: k = 4; G2P: n = 8)
    static constexpr int NSB = (P + BY - 2) / BY + 2, NSC = (P + BZ - 2) / BZ + 2;   // block tiles a window can meet
    static_assert(P % 4 == 0 && (!SPREAD || P % 8 == 0) && (REC % 2) == 0 && NCW % 4 == 0 && CAP % GRP == 0, "layout");
};
// registers per thread after the warpgroups re-split the register file (setmaxnreg): per scheduler
// 3 consumer warps + 1 producer-group warp share 512 registers per lane
constexpr int REGS_CONSUMER = 152, REGS_PRODUCER = 56;

template <int P, bool SPREAD>
struct alignas(16) Stage {
    typedef Cfg<P, SPREAD> C;
    double rec[CAP + 1][C::REC];             // [CAP] stays all-zero: the padding record
    double U[SPREAD ? 1 : CAP][C::NCW][3];   // G2P: per-warp partial sums of the round
    int pidx[SPREAD ? 1 : CAP];              // G2P: sorted index of the candidate (slot write-out)
    unsigned char hit[SPREAD ? 1 : CAP][SPREAD ? 4 : 16];   // G2P: did consumer warp w gather from candidate a?
    int s, na, rs, pad;                      // step (anchor plane, unwrapped), candidate count, s mod P
};

// Per-warp scratch of a round: the packed hit list.
template <int P, bool SPREAD>
struct alignas(16) WarpScratch {
    unsigned wl[CAP + 8];            // hit list: candidate a | l_y << 8 | l_z << 20 (window index of the patch origin)
};

template <int P, bool SPREAD>
struct alignas(16) Smem {
    typedef Cfg<P, SPREAD> C;
    Stage<P, SPREAD> st[C::NST];
    WarpScratch<P, SPREAD> ws[C::NCW];
    uint64_t full[C::NST], empty[C::NST], drained[C::NST];
};

__device__ __forceinline__ int modM(int v, int M) { v %= M; return v < 0 ? v + M : v; }

// does the window [0, P) (indices mod M) meet columns T0 .. T0 + n - 1, given l0 = (T0 - anchor) mod M ?
__device__ __forceinline__ bool meets(int l0, int n, int M, int P) { return n > 0 && (l0 < P || l0 + n - 1 >= M); }

// grid values <-> double pairs (the grid is stored in the plan's precision; all arithmetic here is double)
template <typename GR> struct GV;
template <> struct GV<double> {
    static __device__ __forceinline__ void st2(double *p, double a, double b) { *reinterpret_cast<double2 *>(p) = make_double2(a, b); }
    static __device__ __forceinline__ double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
};
template <> struct GV<float> {
    static __device__ __forceinline__ void st2(float *p, double a, double b) { *reinterpret_cast<float2 *>(p) = make_float2((float)a, (float)b); }
    static __device__ __forceinline__ double2 ld2(const float *p) { const float2 v = *reinterpret_cast<const float2 *>(p); return make_double2((double)v.x, (double)v.y); }
};

// P: ring size = row stride of the records (a multiple of 8 for P2G, of 4 for G2P); W <= P: window support (the
// record rows are zero beyond W); GR: grid storage type.
// SLAB: the grid has g.Mx planes along x instead of M (slab plans, se.h se_plan_desc); a compile-time switch, so that the
// whole-grid kernels keep one grid size in registers (the extra live value cost G2P 7 %)
// what k_mma needs of the plan's geometry: a compact by-value parameter (see the note at SeGeom)
struct MmaGeom {
    int64_t N;
    int M, Mx, nbin, nchunk, nchunk_g2p, nfull, nsplit;
};

template <int P, bool SPREAD, int W, typename GR, bool SLAB>
__global__ void __launch_bounds__((NWY * NWZ + 4) * 32, 1)
k_mma(MmaGeom g, const double *__restrict__ recs, const int *__restrict__ bin_start, GR *__restrict__ grid,
      double *__restrict__ uFpart)
{
    static_assert(W <= P && W > P - (SPREAD ? 8 : 4), "window / ring");
    typedef Cfg<P, SPREAD> C;
    constexpr int NCW = C::NCW, BY = C::BY, BZ = C::BZ, MT = C::MT, REC = C::REC, NST = C::NST, GRP = C::GRP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem<P, SPREAD> &S = *reinterpret_cast<Smem<P, SPREAD> *>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int M = g.M, Mx = SLAB ? g.Mx : g.M, nzb = g.nbin;      // Mx planes along x (the sweep direction), M along y and z
    const int ntY = (M + BY - 1) / BY, ntZ = (M + BZ - 1) / BZ;
    int tile = blockIdx.x % (ntZ * ntY), chunk = blockIdx.x / (ntZ * ntY);
    int nchunk = SPREAD ? g.nchunk : g.nchunk_g2p;
    if (SPREAD && g.nsplit > 1) {
        // whole sweeps first (one block per tile), then the tiles of the last wave in nsplit pieces each
        if ((int)blockIdx.x < g.nfull) { tile = blockIdx.x; chunk = 0; nchunk = 1; }
        else { const int bb = blockIdx.x - g.nfull; tile = g.nfull + bb / g.nsplit; chunk = bb % g.nsplit; nchunk = g.nsplit; }
    }
    const int tz = tile % ntZ, ty = tile / ntZ;
    const int CL = (Mx + nchunk - 1) / nchunk;
    const int X0 = chunk * CL;
    const int CLen = min(CL, Mx - X0);
    if (CLen <= 0) return;
    const int Y0 = ty * BY, Z0 = tz * BZ;
    // P2G: a chunk re-spreads the P - 1 anchor planes in front of it (warm-up) -- except when one chunk covers the
    // whole periodic axis: then the sweep starts at plane 0 and the P - 1 planes left in the ring at the end are the
    // wrapped contributions to planes 0 .. P - 2, which the same thread adds to what it wrote there (no warm-up).
    const bool wrap_add = SPREAD && nchunk == 1;
    const int s_begin = (SPREAD && !wrap_add) ? X0 - (W - 1) : X0, s_end = X0 + CLen;

    for (int e = tid; e < NST * REC; e += C::NT) S.st[e / REC].rec[CAP][e % REC] = 0.0;
    if (tid == 0)
        for (int i = 0; i < NST; ++i) {
            mbar_init(&S.full[i], 1); mbar_init(&S.empty[i], NCW); mbar_init(&S.drained[i], 3);
        }
    __syncthreads();

    if (warp >= NCW) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS_PRODUCER));
        if (warp > NCW) {
            // ============================ G2P WRITE-OUT WARPS ===================================================
            // add the consumers' partial sums of every round in fixed order, one slot per (particle, block tile)
            if (SPREAD) return;
            const int wl = (warp - NCW - 1) * 32 + lane;             // 0 .. 95
            for (int r = 0;; ++r) {
                const int sg = r % NST;
                Stage<P, SPREAD> &T = S.st[sg];
                mbar_wait(&S.full[sg], (r / NST) & 1);
                if (T.s >= s_end) return;
                mbar_wait(&S.empty[sg], (r / NST) & 1);
                const int n3 = T.na * 3;
                for (int it = wl; it < n3; it += 96) {
                    const int a = it / 3, c = it - 3 * a;
                    const int2 an = *reinterpret_cast<const int2 *>(&T.rec[a][C::OM]);
                    const int ly = modM(Y0 - an.x, M), lz = modM(Z0 - an.y, M);
                    const bool hit = meets(ly, min(BY, M - Y0), M, W) && meets(lz, min(BZ, M - Z0), M, W);
                    const int rb = modM(ty - an.x / BY, ntY), rc = modM(tz - an.y / BZ, ntZ);
                    if (hit && rb < C::NSB && rc < C::NSC) {
                        double sum = 0.0;
#pragma unroll
                        for (int w = 0; w < NCW; ++w) sum += T.hit[a][w] ? T.U[a][w][c] : 0.0;
                        uFpart[((size_t)(rb * C::NSC + rc) * g.N + T.pidx[a]) * 3 + c] = sum;
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&S.drained[sg]);
            }
        }
        // =================================== PRODUCER ==========================================================
        // candidate rows / z-bins of this block tile (anchors): cyclic [Y0-(P-1), Y0+BY-1], [Z0-(P-1), Z0+BZ-1]
        const int leny = min(BY + W - 1, M);
        const int ylo = modM(Y0 - (W - 1), M);
        int zb0, nzbins;
        {
            const int len = BZ + W - 1;
            if (len + ZBW > M) { zb0 = 0; nzbins = nzb; }
            else {
                const int lo = modM(Z0 - (W - 1), M), hi = modM(Z0 + BZ - 1, M);
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
        // this lane's run of step s: [beg, beg + len) in the sorted order
        int r0 = 0, r1 = 0, zoff = 0;
        if (rl < nrun) {
            const int k = rl >> 1, piece = rl & 1;
            int zb = zb0 + k; if (zb >= nzb) zb -= nzb;
            zoff = zb * M;
            if (piece == 0) { r0 = ylo; r1 = min(ylo + leny, M); }
            else { r0 = 0; r1 = max(ylo + leny - M, 0); }
        }
        auto run_of = [&](int s, int &beg, int &len) {
            beg = 0; len = 0;
            if (s < s_end && r1 > r0) {
                const int base = modM(s, Mx) * nzb * M + zoff;
                beg = __ldg(&bin_start[base + r0]);
                len = __ldg(&bin_start[base + r1]) - beg;
            }
        };
        // wait until stage r % NST has been released (P2G: by the consumers; G2P: by the write-out warps)
        auto acquire = [&](int r) {
            const int sg = r % NST;
            if (r >= NST) mbar_wait(SPREAD ? &S.empty[sg] : &S.drained[sg], ((r / NST) - 1) & 1);
        };

        int nbeg, nlen;
        run_of(s_begin + sl, nbeg, nlen);
        for (int sb = s_begin; sb < s_end; sb += 2) {
            const int beg = nbeg, len = nlen;
            run_of(sb + 2 + sl, nbeg, nlen);                         // next iteration's offsets: latency overlaps this one
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
                    Stage<P, SPREAD> &T = S.st[rcount % NST];
                    uint64_t *bar = &S.full[rcount % NST];
                    if (lane == 0) {
                        T.s = sb + k; T.na = na; T.rs = modM(sb + k, P);
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
        // terminal round: lets the consumers (and the write-out warps) finish
        acquire(rcount);
        if (lane == 0) {
            Stage<P, SPREAD> &T = S.st[rcount % NST];
            T.s = s_end; T.na = 0; T.rs = 0;
            mbar_arrive(&S.full[rcount % NST]);
        }
        return;
    }

    // ======================================= CONSUMER ==============================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS_CONSUMER));
    const int gq = lane >> 2, tq = lane & 3;
    const int wy0 = 4 * (warp / NWZ), wz0 = 4 * (warp % NWZ);       // warp patch inside the block tile
    const int Yw = Y0 + wy0, Zw = Z0 + wz0;
    const int nyw = min(4, M - Yw), nzw = min(4, M - Zw);           // valid rows / columns of the patch
    const size_t MM = (size_t)M * M, M3 = MM * Mx;
    WarpScratch<P, SPREAD> &WS = S.ws[warp];
    // Both kernels see the patch as two n-tiles of 8 columns: column n of n-tile j is row 2j + (n >> 2),
    // z-column n & 3 of the patch.

    // cur: P2G first plane not yet flushed; G2P first plane not yet in the ring.  curP = cur mod P, curM = cur mod M.
    int cur = s_begin, curP = modM(s_begin, P), curM = modM(s_begin, Mx);
    auto advance = [&]() {
        ++cur;
        if (++curP == P) curP = 0;
        if (++curM == Mx) curM = 0;
    };

    // this warp's hits of a round: packed list (candidate, window index of the patch origin in y and z), padded
    // to whole K-groups with the all-zero record.  The DMMA operands are read from the staged records
    // directly (window value W[(l0 + i) mod M], zero outside the support): no per-warp copy of the windows.
    auto build_hits = [&](Stage<P, SPREAD> &T, int na) -> int {
        int cnt = 0;
        for (int a0 = 0; a0 < na; a0 += 32) {
            const int a = a0 + lane;
            bool hit = false;
            int ly = 0, lz = 0;
            if (a < na) {
                const int2 an = *reinterpret_cast<const int2 *>(&T.rec[a][C::OM]);
                ly = Yw - an.x; if (ly < 0) ly += M;
                lz = Zw - an.y; if (lz < 0) lz += M;
                hit = meets(ly, nyw, M, W) && meets(lz, nzw, M, W);
                if (!SPREAD) T.hit[a][warp] = (unsigned char)hit;
            }
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) WS.wl[cnt + __popc(m & ((1u << lane) - 1u))] = (unsigned)a | ((unsigned)ly << 8) | ((unsigned)lz << 20);
            cnt += __popc(m);
        }
        const int padded = (cnt + GRP - 1) & ~(GRP - 1);
        if (lane < padded - cnt) WS.wl[cnt + lane] = (unsigned)CAP;
        __syncwarp();
        return padded;
    };
    // window value W[(l0 + i) mod M] of a staged record row, zero outside the support (l0 + i < 2 M)
    auto wrec = [&](const double *w, int l) -> double {
        if (l >= M) l -= M;
        return l < W ? w[l] : 0.0;
    };

    if constexpr (SPREAD) {
        // ---------------------------------------- P2G ---------------------------------------------------------
        // C[row = plane residue][n] += A[row][k = hit] B[k][n]:  A = c_w f_c Wx straight from the record,
        // B = Wy Wz.  Ring acc[mt][c][j]: C fragment of m-tile mt, component c, n-tile j; this lane holds
        // columns n = 2 tq, 2 tq + 1 -> patch row 2j + (tq >> 1), z-columns 2 (tq & 1), + 1.
        double acc[MT][3][2][2];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int j = 0; j < 2; ++j) acc[mt][c][j][0] = acc[mt][c][j][1] = 0.0;
        const int cyl = tq >> 1, czl = 2 * (tq & 1);
        const bool cz_ok = czl < nzw;                                // M, Zw even: the pair is valid together
        const size_t colS = (size_t)(Yw + cyl) * M + (Zw + czl);
        auto flush_mt = [&](auto mtc, int XM, bool valid) {
            constexpr int mt = decltype(mtc)::value;
            const size_t off = (size_t)XM * MM + colS;
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    if (valid && 2 * j + cyl < nyw)
                        GV<GR>::st2(&grid[c * M3 + off + (size_t)(2 * j) * M], acc[mt][c][j][0], acc[mt][c][j][1]);
                    acc[mt][c][j][0] = acc[mt][c][j][1] = 0.0;
                }
        };
        auto flush = [&]() {                                         // plane cur is complete: write it, clear its residue
            if (gq == (curP & 7)) {
                const bool valid = cz_ok && cur >= X0;
                switch (curP >> 3) {
                case 0: flush_mt(std::integral_constant<int, 0>{}, curM, valid); break;
                case 1: flush_mt(std::integral_constant<int, 1>{}, curM, valid); break;
                case 2: if constexpr (MT > 2) flush_mt(std::integral_constant<int, 2>{}, curM, valid); break;
                case 3: if constexpr (MT > 3) flush_mt(std::integral_constant<int, 3>{}, curM, valid); break;
                }
            }
        };
        for (int r = 0;; ++r) {
            const int sg = r % NST;
            Stage<P, SPREAD> &T = S.st[sg];
            mbar_wait(&S.full[sg], (r / NST) & 1);
            const int s = T.s, na = T.na, rs = T.rs;
            if (s >= s_end) {                                        // terminal round
                while (cur < s_end) { flush(); advance(); }
                if (wrap_add) {
                    // ring residue 8 mt + gq now holds plane s_end + t, t = (8 mt + gq - s_end) mod P, i.e. grid
                    // plane t of the next period: all loads first, then add and store
                    double2 o[MT][3][2];
                    int tt[MT];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        int t = 8 * mt + gq - curP; if (t < 0) t += P;
                        tt[mt] = t;
#pragma unroll
                        for (int c = 0; c < 3; ++c)
#pragma unroll
                            for (int j = 0; j < 2; ++j)
                                if (cz_ok && t < W - 1 && 2 * j + cyl < nyw)
                                    o[mt][c][j] = GV<GR>::ld2(&grid[c * M3 + (size_t)t * MM + colS + (size_t)(2 * j) * M]);
                    }
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                        for (int c = 0; c < 3; ++c)
#pragma unroll
                            for (int j = 0; j < 2; ++j)
                                if (cz_ok && tt[mt] < W - 1 && 2 * j + cyl < nyw)
                                    GV<GR>::st2(&grid[c * M3 + (size_t)tt[mt] * MM + colS + (size_t)(2 * j) * M],
                                                o[mt][c][j].x + acc[mt][c][j][0], o[mt][c][j].y + acc[mt][c][j][1]);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&S.empty[sg]);
                break;
            }
            while (cur < s) { flush(); advance(); }
            const int padded = build_hits(T, na);
            // Wx index of this lane's ring rows: plane s + l <-> residue (s + l) mod P
            int lx[MT];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) { int l = 8 * mt + gq - rs; lx[mt] = l < 0 ? l + P : l; }
            // B[k = tq][n = gq] = Wy Wz of hit tq at column n of the two n-tiles (rows gq >> 2 and + 2, z-column
            // gq & 3).  No FP64 arithmetic feeds a DMMA of the same group: the two B products of group q + 1
            // are formed while group q issues.
            const int by = gq >> 2, bz = gq & 3;
            auto bprod = [&](unsigned w, double &p0, double &p1) {
                const double *rp = T.rec[w & 0xffu];
                const int ly = (int)((w >> 8) & 0xfffu) + by, lz = (int)(w >> 20) + bz;
                const double wz = wrec(rp + C::OZ, lz);
                p0 = wrec(rp + C::OY, ly) * wz; p1 = wrec(rp + C::OY, ly + 2) * wz;
            };
            unsigned wcur = 0;
            double b0 = 0.0, b1 = 0.0;
            if (padded > 0) { wcur = WS.wl[tq]; bprod(wcur, b0, b1); }
            for (int q = 0; q < padded; q += 4) {
                const double *rp = T.rec[wcur & 0xffu];
                double a[MT][3];
#pragma unroll
                for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                    for (int c = 0; c < 3; ++c) a[mt][c] = rp[c * P + lx[mt]];
                const double c0 = b0, c1 = b1;
                if (q + 4 < padded) { wcur = WS.wl[q + 4 + tq]; bprod(wcur, b0, b1); }
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    dmma(acc[mt][0][0], a[mt][0], c0); dmma(acc[mt][0][1], a[mt][0], c1);
                    dmma(acc[mt][1][0], a[mt][1], c0); dmma(acc[mt][1][1], a[mt][1], c1);
                    dmma(acc[mt][2][0], a[mt][2], c0); dmma(acc[mt][2][1], a[mt][2], c1);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.empty[sg]);
        }
    } else {
        // ---------------------------------------- G2P ---------------------------------------------------------
        // E[hit][n] = sum_planes A[hit][k = plane] B[k][n]:  A = Wx of 8 hits straight from the record, B = the
        // ring of grid planes, rg[ks][c][j] = plane residue 4 ks + tq, column n = gq of n-tile j, component c.
        // All P/4 k-steps of a group accumulate in 6 independent chains (c, j); the epilogue multiplies by
        // Wy Wz of the hit, sums this lane's two columns of both n-tiles and reduces over the 4 tq lanes.
        constexpr int KS = P / 4;
        double rg[KS][3][2];
#pragma unroll
        for (int ks = 0; ks < KS; ++ks)
#pragma unroll
            for (int c = 0; c < 3; ++c) rg[ks][c][0] = rg[ks][c][1] = 0.0;
        const int gyl = gq >> 2, gzl = gq & 3;                       // this lane's column of an n-tile
        const bool gz_ok = gzl < nzw;
        const size_t colG = (size_t)(Yw + gyl) * M + (Zw + gzl);
        double pre[3][2];                                            // plane prefetched one step ahead
        int pre_X = INT_MIN, preP = 0;
        auto fetch_plane = [&](int X, int XP, int XM) {              // issue the loads of plane X into `pre`
            pre_X = X; preP = XP;
            if (tq != (XP & 3)) return;
            const size_t off = (size_t)XM * MM + colG;
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int j = 0; j < 2; ++j)
                    pre[c][j] = (gz_ok && 2 * j + gyl < nyw) ? (double)__ldg(&grid[c * M3 + off + (size_t)(2 * j) * M]) : 0.0;
        };
        auto commit_plane = [&]() {                                  // move `pre` into its residue of the ring
            // warp-uniform switch over the k-step, predicated moves inside (a divergent early-out in front of the
            // switch made the compiler shuffle the whole ring through moves)
            const bool mine = tq == (preP & 3);
            const int ksel = __shfl_sync(0xffffffffu, preP >> 2, 0);
#define SE_COMMIT(ks)                                                                  \
    case ks:                                                                           \
        if constexpr (ks < KS) {                                                       \
            _Pragma("unroll") for (int c = 0; c < 3; ++c) {                            \
                if (mine) { rg[ks < KS ? ks : 0][c][0] = pre[c][0]; rg[ks < KS ? ks : 0][c][1] = pre[c][1]; } \
            }                                                                          \
        }                                                                              \
        break;
            switch (ksel) {
                SE_COMMIT(0) SE_COMMIT(1) SE_COMMIT(2) SE_COMMIT(3) SE_COMMIT(4) SE_COMMIT(5) SE_COMMIT(6) SE_COMMIT(7)
            }
#undef SE_COMMIT
        };
        for (int r = 0;; ++r) {
            const int sg = r % NST;
            Stage<P, SPREAD> &T = S.st[sg];
            mbar_wait(&S.full[sg], (r / NST) & 1);
            const int s = T.s, na = T.na, rs = T.rs;
            if (s >= s_end) {                                        // terminal round
                __syncwarp();
                if (lane == 0) mbar_arrive(&S.empty[sg]);
                break;
            }
            // planes s .. s+P-1 must be in the ring; plane cur may be waiting in `pre`
            if (cur < s) { cur = s; curP = rs; curM = modM(s, Mx); pre_X = INT_MIN; }  // planes nobody gathers from
            if (s + P - cur > 2) {
                // (re)fill after a chunk start or a jump: all missing planes of this lane's k-columns at once (one
                // memory latency instead of one per plane); residue 4 ks + tq holds plane s + ((4 ks + tq - rs) mod P)
                const int sM = modM(s, Mx);
#pragma unroll
                for (int ks = 0; ks < KS; ++ks) {
                    int l = 4 * ks + tq - rs; if (l < 0) l += P;
                    if (s + l < cur) continue;                       // still valid in the ring
                    int XM = sM + l; if (XM >= Mx) XM -= Mx;
                    const size_t off = (size_t)XM * MM + colG;
#pragma unroll
                    for (int c = 0; c < 3; ++c)
#pragma unroll
                        for (int j = 0; j < 2; ++j)
                            rg[ks][c][j] = (gz_ok && 2 * j + gyl < nyw) ? (double)__ldg(&grid[c * M3 + off + (size_t)(2 * j) * M]) : 0.0;
                }
                cur = s + P; curP = rs; curM = modM(cur, Mx); pre_X = INT_MIN;
            }
            while (cur < s + P) {
                if (pre_X != cur) fetch_plane(cur, curP, curM);
                commit_plane();
                advance();
            }
            if (pre_X != cur) fetch_plane(cur, curP, curM);          // plane s + P: consumed at the next step
            const int padded = build_hits(T, na);
            // Wx index of this lane's k-column: residue 4 ks + tq <-> plane s + l
            int lx[KS];
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) { int l = 4 * ks + tq - rs; lx[ks] = l < 0 ? l + P : l; }
            // epilogue weights of hit gq at this lane's D columns n = 2 tq, 2 tq + 1 of n-tile j:
            // row 2j + (tq >> 1), z-columns 2 (tq & 1), + 1
            const int ey = tq >> 1, ez = 2 * (tq & 1);
            // the hit word of group q + 1 is read before the epilogue of group q (whose shared-memory stores would
            // otherwise order the dependent chain hit word -> record loads behind it)
            unsigned wn = padded > 0 ? WS.wl[gq] : (unsigned)CAP;
            for (int q = 0; q < padded; q += 8) {
                const unsigned w = wn;
                const int a = (int)(w & 0xffu);
                const double *rp = T.rec[a];
                double wx[KS];
#pragma unroll
                for (int ks = 0; ks < KS; ++ks) wx[ks] = rp[lx[ks]];
                const int ly = (int)((w >> 8) & 0xfffu) + ey, lz = (int)(w >> 20) + ez;
                const double wy0 = wrec(rp + C::OY, ly), wy1 = wrec(rp + C::OY, ly + 2);
                const double wz0 = wrec(rp + C::OZ, lz), wz1 = wrec(rp + C::OZ, lz + 1);
                const double w00 = wy0 * wz0, w01 = wy0 * wz1, w10 = wy1 * wz0, w11 = wy1 * wz1;
                if (q + 8 < padded) wn = WS.wl[q + 8 + gq];
                // one component at a time (8 accumulator registers live instead of 24), the epilogue of component c
                // placed behind the DMMAs of component c + 1 so that it does not wait for their results in line
                double pc[3];
                double e0[2], e1[2];
                auto burst = [&](int c, double (&d0)[2], double (&d1)[2]) {
                    d0[0] = d0[1] = d1[0] = d1[1] = 0.0;
#pragma unroll
                    for (int ks = 0; ks < KS; ++ks) { dmma(d0, wx[ks], rg[ks][c][0]); dmma(d1, wx[ks], rg[ks][c][1]); }
                };
                auto fold = [&](const double (&d0)[2], const double (&d1)[2]) -> double {
                    double v = d0[0] * w00;
                    v = fma(d0[1], w01, v); v = fma(d1[0], w10, v); v = fma(d1[1], w11, v);
                    v += __shfl_xor_sync(0xffffffffu, v, 1);
                    v += __shfl_xor_sync(0xffffffffu, v, 2);
                    return v;
                };
                {
                    double f0[2], f1[2];
                    burst(0, e0, e1);
                    burst(1, f0, f1);
                    pc[0] = fold(e0, e1);
                    burst(2, e0, e1);
                    pc[1] = fold(f0, f1);
                    pc[2] = fold(e0, e1);
                }
                if (tq == 0 && a < CAP) { T.U[a][warp][0] = pc[0]; T.U[a][warp][1] = pc[1]; T.U[a][warp][2] = pc[2]; }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.empty[sg]);
        }
    }
}

// u^F (grid-sorted order) = fixed-order sum of the slots the particle's window actually meets
template <int P, int W, typename GR>
__global__ void k_reduce_slots(SeGeom g, const short4 *__restrict__ anchor, const double *__restrict__ part,
                               GR *__restrict__ uF)
{
    typedef Cfg<P, false> C;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.N) return;
    const int M = g.M;
    const int ntY = (M + C::BY - 1) / C::BY, ntZ = (M + C::BZ - 1) / C::BZ;
    const short4 a = anchor[i];
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int rb = 0; rb < C::NSB && rb < ntY; ++rb) {
        const int ty = (a.y / C::BY + rb) % ntY, Y0 = ty * C::BY;
        if (!meets(modM(Y0 - a.y, M), min(C::BY, M - Y0), M, W)) continue;
        for (int rc = 0; rc < C::NSC && rc < ntZ; ++rc) {
            const int tz = (a.z / C::BZ + rc) % ntZ, Z0 = tz * C::BZ;
            if (!meets(modM(Z0 - a.z, M), min(C::BZ, M - Z0), M, W)) continue;
            const double *q = part + ((size_t)(rb * C::NSC + rc) * g.N + i) * 3;
            s0 += q[0]; s1 += q[1]; s2 += q[2];
        }
    }
    uF[3 * i + 0] = (GR)s0; uF[3 * i + 1] = (GR)s1; uF[3 * i + 2] = (GR)s2;
}

// prepare == true: only opt this plan's device in to the kernel's dynamic shared memory (once per plan, at creation)
template <int P, bool SPREAD, int W, typename GR, bool SLAB>
cudaError_t launch_k(se_plan *p, cudaStream_t s, bool prepare)
{
    typedef Cfg<P, SPREAD> C;
    SeGeom g = p->g;
    const SeSet &Q = SPREAD ? p->S : p->T;                     // P2G spreads the sources, G2P gathers at the targets
    g.N = Q.n;
    constexpr size_t smem = sizeof(Smem<P, SPREAD>);
    static_assert(smem <= 227 * 1024, "shared memory per block");
    auto kern = k_mma<P, SPREAD, W, GR, SLAB>;
    if (prepare) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int ntY = (g.M + C::BY - 1) / C::BY, ntZ = (g.M + C::BZ - 1) / C::BZ;
    const int nchunk = SPREAD ? g.nchunk : g.nchunk_g2p;
    const int nblocks = (SPREAD && g.nsplit > 1) ? g.nfull + g.nsplit * (ntY * ntZ - g.nfull) : nchunk * ntY * ntZ;
    const MmaGeom mg{g.N, g.M, g.Mx, g.nbin, g.nchunk, g.nchunk_g2p, g.nfull, g.nsplit};
    kern<<<(unsigned)nblocks, C::NT, smem, s>>>(mg, (const double *)(SPREAD ? Q.wtab : Q.recg), Q.bin_start,
                                                             (GR *)p->grid, (double *)p->uFpart);
    p->launches += 1;
    if (!SPREAD) {
        k_reduce_slots<P, W, GR><<<(unsigned)((g.N + 255) / 256), 256, 0, s>>>(g, Q.anchor, (const double *)p->uFpart,
                                                                            (GR *)p->uF);
        p->launches += 1;
    }
    return cudaGetLastError();
}

template <int P, bool SPREAD, int W, typename GR>
cudaError_t launch(se_plan *p, cudaStream_t s, bool prepare)
{
    return p->slab ? launch_k<P, SPREAD, W, GR, true>(p, s, prepare) : launch_k<P, SPREAD, W, GR, false>(p, s, prepare);
}

template <bool SPREAD>
cudaError_t dispatch(se_plan *p, cudaStream_t s, bool prepare = false)
{
    // ring (row stride of the records; the rows are zero beyond the window): P rounded up to a multiple of 8 for P2G
    // (m-tiles of 8 planes), of 4 for G2P (k-steps of 4 planes); fp32 plans: float grid, double records / accumulators
#define SE_MMA_CASE(W, GR) \
    case W: return launch<SPREAD ? (W + 7) / 8 * 8 : (W + 3) / 4 * 4, SPREAD, W, GR>(p, s, prepare);
    if (p->precision == SE_FP64) {
        switch (p->g.P) {
            SE_MMA_CASE(4, double) SE_MMA_CASE(6, double) SE_MMA_CASE(8, double) SE_MMA_CASE(10, double)
            SE_MMA_CASE(12, double) SE_MMA_CASE(14, double) SE_MMA_CASE(16, double) SE_MMA_CASE(18, double)
            SE_MMA_CASE(20, double) SE_MMA_CASE(22, double) SE_MMA_CASE(24, double)
        default: return cudaErrorInvalidValue;
        }
    }
    switch (p->g.P) {
        SE_MMA_CASE(4, float) SE_MMA_CASE(6, float) SE_MMA_CASE(8, float) SE_MMA_CASE(10, float)
        SE_MMA_CASE(12, float) SE_MMA_CASE(14, float) SE_MMA_CASE(16, float)
    default: return cudaErrorInvalidValue;
    }
#undef SE_MMA_CASE
}

}  // namespace

bool se_mma_supported(int P, int precision)
{
    return P >= 4 && !(P & 1) && P <= (precision == SE_FP64 ? 24 : 16);
}
int se_mma_ring(int P) { return (P + 7) / 8 * 8; }     // row stride of the spread records
int se_mma_ring_g(int P) { return (P + 3) / 4 * 4; }   // row stride of the gather records
int se_mma_slots(int P)                                // slots of a particle in uFpart: block tiles its window can meet
{
    switch (se_mma_ring_g(P)) {
    case 24: return Cfg<24, false>::NSB * Cfg<24, false>::NSC;
    case 20: return Cfg<20, false>::NSB * Cfg<20, false>::NSC;
    case 16: return Cfg<16, false>::NSB * Cfg<16, false>::NSC;
    case 12: return Cfg<12, false>::NSB * Cfg<12, false>::NSC;
    case 8: return Cfg<8, false>::NSB * Cfg<8, false>::NSC;
    default: return Cfg<4, false>::NSB * Cfg<4, false>::NSC;
    }
}
cudaError_t se_launch_mma_p2g(se_plan *p, cudaStream_t s) { return dispatch<true>(p, s); }
cudaError_t se_launch_mma_g2p(se_plan *p, cudaStream_t s) { return dispatch<false>(p, s); }
cudaError_t se_prepare_mma(se_plan *p)
{
    cudaError_t e = dispatch<true>(p, nullptr, true);
    return e != cudaSuccess ? e : dispatch<false>(p, nullptr, true);
}
