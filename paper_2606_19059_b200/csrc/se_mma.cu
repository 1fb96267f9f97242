// K3 P2G (eq. (2.5)) and K5 G2P (eq. (2.7)) in FP64 as an x-SWEEP whose inner
// product runs on the FP64 tensor-core path (mma.sync m8n8k4 f64 -> DMMA), for P = 16 and 24.
//
// Why.  With a Gaussian window at P = 24 both gridding steps are FP64-arithmetic bound: 3 P^3 = 41,472
// FMA per particle against ~1 KB of compulsory traffic.  On B200 the DFMA pipe
// and DMMA deliver the same peak (36.7 vs 33.0 TFLOP/s measured), but one DFMA warp instruction is 32
// FMAs and needs an issue slot every 2 cycles per scheduler, while one DMMA is 256 FMAs and occupies the
// pipe for 16 cycles: the tensor form leaves ~15 of every 16 issue slots for the bookkeeping that
// output-stationary gridding needs (candidate lists, table staging, ring rotation).  tcgen05 has no
// FP64 kind, so mma.sync is the only tensor path for this precision.
//
// The contraction.  Spreading is  H_c[x,y,z] += sum_n (f_nc Wx_n[x]) * (Wy_n[y] Wz_n[z]); for one y it is a
// GEMM  C[(x), (z)] += A[(x), n] B[n, (z)]  with K = particles.  A warp owns J = 2 y-rows x 8 z-columns and
// sweeps x: its accumulators are a RING of the P planes currently under the window (plane X lives in
// residue X mod P, P/8 m-tiles of 8 rows) x 3 components x J, i.e. 9 J C-fragments (36 doubles per thread
// at P = 24).  Particles are sorted by (anchor plane a_x, a_z / 16, a_y); all particles of one step have
// the same a_x, touch every residue exactly once, and are consumed 4 at a time (the K of m8n8k4).  When the
// sweep leaves a plane it is complete and is written once with plain 16-byte stores: no atomics, no
// zero-fill, deterministic.  Efficiency of issued FMAs: 1 in x (no tile overlap in the sweep direction),
// P/(P+J-1) in y, P/(P+7) in z.
// Gathering is the transpose: the ring holds the grid planes as A-fragments (rows = planes, k = z),
// B = Wy Wz of 8 particles, D[(plane), particle] is contracted with Wx in a short epilogue and reduced over
// the 8 row-lanes with a packed butterfly; per-(particle, block tile) partial sums go to their own slot and
// are added in a fixed order afterwards (bit-reproducible, no atomics).
//
// Block = NWY x NWZ CONSUMER warps (the contraction above) + 4 PRODUCER warps.  Each producer warp walks
// the sweep on its own, and for every NPW-th round (<= CAP candidates of one step) finds the candidate runs
// in the sorted order, reads the anchors, and stages the records (Wx[P], the block tile's slices of Wy and
// Wz zero-padded outside the support, f) from the global window tables into its own shared-memory stage;
// full/empty mbarriers hand the stages over, so table staging (three dependent global latencies) overlaps
// the tensor work of the previous rounds.  In G2P the producer also adds the consumers' per-warp partial
// sums in fixed order and writes the slot before it refills a stage.
#include <type_traits>

#include "se_common.cuh"

namespace {

constexpr int CAP = 48;              // candidates per round (one step's candidates, split if more)
constexpr int NPW = 4;               // producer warps = stages
constexpr int ZBW = SE_MMA_ZBIN;     // z-bin width of the sort key

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

// 8-byte async copy global -> shared; !pred writes zeros (src-size 0)
__device__ __forceinline__ void cp_async8(void *dst, const void *src, bool pred)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(pred ? 8 : 0)
                 : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <int P, int NWY, int NWZ>
struct Cfg {
    static constexpr int NCW = NWY * NWZ;                      // consumer warps
    static constexpr int NT = (NCW + NPW) * 32;
    static constexpr int BY = 2 * NWY, BZ = 8 * NWZ;           // block tile (columns)
    static constexpr int MT = P / 8;                           // m-tiles in the ring
    static constexpr int OY = P, OZ = P + BY, OF = P + BY + BZ;  // record offsets: wx | wy | wz | f
    static constexpr int REC = OF + 4;
    static constexpr int NSB = (P - 2) / BY + 3, NSC = (P - 2) / BZ + 3;   // block tiles a window can meet
    static constexpr int NCP = P / 2 + BY + BZ + 3;            // async copies per record: wx in 16-byte pieces
    static_assert(P % 8 == 0 && (REC % 2) == 0 && NCP <= 64, "layout");
};

template <int P, int NWY, int NWZ, bool SPREAD>
struct alignas(16) Stage {
    typedef Cfg<P, NWY, NWZ> C;
    double rec[CAP + 1][C::REC];             // [CAP] stays all-zero: the padding record
    double U[SPREAD ? 1 : CAP][C::NCW][3];   // G2P: per-warp partial sums of the round
    int pidx[CAP];
    short ly0[CAP], lz0[CAP];                // window index of the block tile's first column, in [0, M)
    short sid[CAP];                          // G2P: slot of (particle, this block tile); -1: does not touch
    int s, na;                               // step (anchor plane, unwrapped) and candidate count
};

template <int P, int NWY, int NWZ, bool SPREAD>
struct alignas(16) Smem {
    typedef Cfg<P, NWY, NWZ> C;
    Stage<P, NWY, NWZ, SPREAD> st[NPW];
    uint64_t full[NPW], empty[NPW];
    unsigned char wlist[C::NCW][CAP + 8];
};

__device__ __forceinline__ int modM(int v, int M) { v %= M; return v < 0 ? v + M : v; }

// does the window [0, P) (indices mod M) meet columns T0 .. T0 + n - 1, given l0 = (T0 - anchor) mod M ?
__device__ __forceinline__ bool meets(int l0, int n, int M, int P) { return n > 0 && (l0 < P || l0 + n - 1 >= M); }

template <int P, int NWY, int NWZ, bool SPREAD>
__global__ void __launch_bounds__((NWY * NWZ + NPW) * 32, 1)
k_mma(SeGeom g, const short4 *__restrict__ anchor, const double *__restrict__ wtab,
      const double *__restrict__ fs, const int *__restrict__ bin_start, double *__restrict__ grid,
      double *__restrict__ uFpart)
{
    typedef Cfg<P, NWY, NWZ> C;
    constexpr int NCW = C::NCW, BY = C::BY, BZ = C::BZ, MT = C::MT, REC = C::REC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem<P, NWY, NWZ, SPREAD> &S = *reinterpret_cast<Smem<P, NWY, NWZ, SPREAD> *>(smem_raw);

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

    for (int e = tid; e < NPW * REC; e += C::NT) S.st[e / REC].rec[CAP][e % REC] = 0.0;
    if (tid == 0)
        for (int i = 0; i < NPW; ++i) { mbar_init(&S.full[i], 1); mbar_init(&S.empty[i], NCW); }
    __syncthreads();

    if (warp >= NCW) {
        // =================================== PRODUCER ==========================================================
        const int pw = warp - NCW;
        Stage<P, NWY, NWZ, SPREAD> &T = S.st[pw];
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
        const int nrun = 2 * nzbins;                                 // <= 10 (z-bin, row-range piece) runs per step
        const int sl = lane >> 4, rl = lane & 15;                    // 2 steps x 16 runs per walk iteration
        int uses = 0;                                                // times this warp has filled its stage
        int rcount = 0;                                              // rounds issued so far (all producers agree)

        // G2P: add the consumers' partial sums of the finished round in fixed order, one slot per block tile
        auto writeout = [&]() {
            if (SPREAD) return;
            const int n3 = T.na * 3;
            for (int it = lane; it < n3; it += 32) {
                const int a = it / 3, c = it - 3 * a;
                const int sid = T.sid[a];
                if (sid >= 0) {
                    double sum = 0.0;
#pragma unroll
                    for (int w = 0; w < NCW; ++w) sum += T.U[a][w][c];
                    uFpart[((size_t)sid * g.N + T.pidx[a]) * 3 + c] = sum;
                }
            }
        };
        // wait until the consumers have released the stage, then make it ours again
        auto acquire = [&]() {
            if (uses > 0) {
                mbar_wait(&S.empty[pw], (uses - 1) & 1);
                writeout();
                __syncwarp();
            }
        };
        auto publish = [&](int s, int na) {
            if (lane == 0) { T.s = s; T.na = na; }
            cp_async_wait_all();
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.full[pw]);
            ++uses;
        };

        for (int sb = s_begin; sb < s_end; sb += 2) {
            const int s = sb + sl;
            int beg = 0, len = 0;
            if (s < s_end && rl < nrun) {
                const int k = rl >> 1, piece = rl & 1;
                int zb = zb0 + k; if (zb >= nzb) zb -= nzb;
                const int base = (modM(s, M) * nzb + zb) * M;
                int r0, r1;                                          // rows [r0, r1)
                if (piece == 0) { r0 = ylo; r1 = min(ylo + leny, M); }
                else { r0 = 0; r1 = max(ylo + leny - M, 0); }
                beg = bin_start[base + r0];
                len = bin_start[base + r1] - beg;
            }
            int tot = len;
            tot += __shfl_xor_sync(0xffffffffu, tot, 1);
            tot += __shfl_xor_sync(0xffffffffu, tot, 2);
            tot += __shfl_xor_sync(0xffffffffu, tot, 4);
            tot += __shfl_xor_sync(0xffffffffu, tot, 8);
            for (int k = 0; k < 2 && sb + k < s_end; ++k) {
                const int total = __shfl_sync(0xffffffffu, tot, 16 * k);
                for (int first = 0; first < total; first += CAP, ++rcount) {
                    if ((rcount & (NPW - 1)) != pw) continue;
                    const int na = min(CAP, total - first);
                    acquire();
                    // ---- identify the candidates: sorted index, anchor -> window offsets of the block tile ------
                    for (int a0 = 0; a0 < na; a0 += 32) {
                        const int a = a0 + lane, v = first + a;
                        int pi = -1, ofs = 0;
#pragma unroll
                        for (int r = 0; r < 10; ++r) {
                            const int b = __shfl_sync(0xffffffffu, beg, 16 * k + r);
                            const int n = __shfl_sync(0xffffffffu, len, 16 * k + r);
                            if (pi < 0 && v < ofs + n) pi = b + (v - ofs);
                            ofs += n;
                        }
                        if (a < na) {
                            const short4 an = anchor[pi];
                            const int ly = modM(Y0 - an.y, M), lz = modM(Z0 - an.z, M);
                            T.pidx[a] = pi;
                            T.ly0[a] = (short)ly; T.lz0[a] = (short)lz;
                            if (!SPREAD) {
                                const bool hit = meets(ly, min(BY, M - Y0), M, P) && meets(lz, min(BZ, M - Z0), M, P);
                                const int rb = modM(ty - an.y / BY, ntY), rc = modM(tz - an.z / BZ, ntZ);
                                T.sid[a] = (short)((hit && rb < C::NSB && rc < C::NSC) ? rb * C::NSC + rc : -1);
                            }
                        }
                    }
                    __syncwarp();
                    // ---- stage the records: asynchronous copies, zero-filled outside the support ------------------
                    const int ncp = na * 64;
                    for (int it = lane; it < ncp; it += 32) {
                        const int a = it >> 6, e = it & 63;
                        if (e >= C::NCP) continue;
                        const int pi = T.pidx[a];
                        const double *w = wtab + (size_t)pi * 3 * P;
                        double *dst = T.rec[a];
                        if (e < P / 2) cp_async16(dst + 2 * e, w + 2 * e);
                        else if (e < P / 2 + BY) {
                            const int j = e - P / 2;
                            int l = T.ly0[a] + j; if (l >= M) l -= M;
                            const bool in = l < P && Y0 + j < M;
                            cp_async8(dst + C::OY + j, w + P + (in ? l : 0), in);
                        } else if (e < P / 2 + BY + BZ) {
                            const int j = e - P / 2 - BY;
                            int l = T.lz0[a] + j; if (l >= M) l -= M;
                            const bool in = l < P && Z0 + j < M;
                            cp_async8(dst + C::OZ + j, w + 2 * P + (in ? l : 0), in);
                        } else {
                            const int c = e - P / 2 - BY - BZ;
                            cp_async8(dst + C::OF + c, fs + (size_t)pi * 3 + c, true);
                        }
                    }
                    if (!SPREAD)
                        for (int it = lane; it < na * NCW * 3; it += 32) (&T.U[0][0][0])[it] = 0.0;
                    publish(sb + k, na);
                }
            }
        }
        // terminal round: lets the consumers finish the sweep
        if ((rcount & (NPW - 1)) == pw) { acquire(); publish(s_end, 0); }
        acquire();                                                   // G2P: slots of this warp's last round
        return;
    }

    // ======================================= CONSUMER ==============================================================
    const int gq = lane >> 2, tq = lane & 3;
    const int wy0 = 2 * (warp / NWZ), wz0 = 8 * (warp % NWZ);       // warp tile inside the block tile
    const int nyw = min(2, M - (Y0 + wy0)), nzw = min(8, M - (Z0 + wz0));
    // this lane's two adjacent z-columns (C-fragment columns in P2G, A-fragment k-columns in G2P)
    const int cy = Y0 + wy0, cz = Z0 + wz0 + 2 * tq;
    const bool col_ok = (cy < M) && (cz < M);                        // M, cy, cz even: pairs are valid together
    const size_t MM = (size_t)M * M, M3 = MM * M;
    const size_t col = (size_t)cy * M + cz;

    // ring: acc[mt][c][j] is a 2-double fragment (P2G: C tile; G2P: A fragments for zh = 0, 1)
    double acc[MT][3][2][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int j = 0; j < 2; ++j) acc[mt][c][j][0] = acc[mt][c][j][1] = 0.0;

    // P2G: plane X (residue X mod P) is complete once every step <= X has been consumed.  The m-tile is
    // selected with a switch over compile-time indices so that the ring stays in registers.
    auto flush_mt = [&](auto mtc, int X, bool valid) {
        constexpr int mt = decltype(mtc)::value;
        const size_t off = (size_t)modM(X, M) * MM + col;
        const double cw = g.cw;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (valid)
                    *reinterpret_cast<double2 *>(&grid[c * M3 + off + (size_t)j * M]) =
                        make_double2(cw * acc[mt][c][j][0], cw * acc[mt][c][j][1]);
                acc[mt][c][j][0] = acc[mt][c][j][1] = 0.0;
            }
    };
    auto flush = [&](int X) {
        const int r = modM(X, P);
        if (gq != (r & 7)) return;
        const bool valid = col_ok && X >= X0;
        switch (r >> 3) {
        case 0: flush_mt(std::integral_constant<int, 0>{}, X, valid); break;
        case 1: flush_mt(std::integral_constant<int, 1>{}, X, valid); break;
        case 2: if constexpr (MT > 2) flush_mt(std::integral_constant<int, 2>{}, X, valid); break;
        case 3: if constexpr (MT > 3) flush_mt(std::integral_constant<int, 3>{}, X, valid); break;
        }
    };
    // G2P: bring plane X into its residue
    auto load_mt = [&](auto mtc, int X) {
        constexpr int mt = decltype(mtc)::value;
        const size_t off = (size_t)modM(X, M) * MM + col;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const double2 v = *reinterpret_cast<const double2 *>(&grid[c * M3 + off + (size_t)j * M]);
                acc[mt][c][j][0] = v.x; acc[mt][c][j][1] = v.y;
            }
    };
    auto load_plane = [&](int X) {
        const int r = modM(X, P);
        if (gq != (r & 7) || !col_ok) return;
        switch (r >> 3) {
        case 0: load_mt(std::integral_constant<int, 0>{}, X); break;
        case 1: load_mt(std::integral_constant<int, 1>{}, X); break;
        case 2: if constexpr (MT > 2) load_mt(std::integral_constant<int, 2>{}, X); break;
        case 3: if constexpr (MT > 3) load_mt(std::integral_constant<int, 3>{}, X); break;
        }
    };

    int cur = s_begin;                       // P2G: first plane not yet flushed; G2P: first plane not yet loaded
    for (int r = 0;; ++r) {
        const int sg = r & (NPW - 1);
        Stage<P, NWY, NWZ, SPREAD> &T = S.st[sg];
        mbar_wait(&S.full[sg], (r / NPW) & 1);
        const int s = T.s, na = T.na;
        if (SPREAD) {
            while (cur < s) { flush(cur); ++cur; }
        } else if (na > 0) {
            cur = max(cur, s);                                       // planes nobody gathers from are skipped
            while (cur < s + P) { load_plane(cur); ++cur; }
        }
        if (s >= s_end) {                                            // terminal round
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.empty[sg]);
            break;
        }

        // ---- this warp's candidates, padded to whole K-groups with the zero record -------------------------
        int cnt = 0;
        for (int a0 = 0; a0 < na; a0 += 32) {
            const int a = a0 + lane;
            bool hit = false;
            if (a < na) {
                int ly = T.ly0[a] + wy0; if (ly >= M) ly -= M;
                int lz = T.lz0[a] + wz0; if (lz >= M) lz -= M;
                hit = meets(ly, nyw, M, P) && meets(lz, nzw, M, P);
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
            for (int q = 0; q < padded; q += 4) {
                const double *rp = T.rec[S.wlist[warp][q + tq]];
                const double f0 = rp[C::OF], f1 = rp[C::OF + 1], f2 = rp[C::OF + 2];
                const double2 wyv = *reinterpret_cast<const double2 *>(&rp[C::OY + wy0]);
                const double wzv = rp[C::OZ + wz0 + gq];
                const double b0 = wyv.x * wzv, b1 = wyv.y * wzv;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const double wx = rp[lx[mt]];
                    const double a0 = f0 * wx, a1 = f1 * wx, a2 = f2 * wx;
                    dmma(acc[mt][0][0], a0, b0); dmma(acc[mt][0][1], a0, b1);
                    dmma(acc[mt][1][0], a1, b0); dmma(acc[mt][1][1], a1, b1);
                    dmma(acc[mt][2][0], a2, b0); dmma(acc[mt][2][1], a2, b1);
                }
            }
        } else {
            for (int q = 0; q < padded; q += 8) {
                const double *rp = T.rec[S.wlist[warp][q + gq]];
                const double2 wyv = *reinterpret_cast<const double2 *>(&rp[C::OY + wy0]);
                const double2 wzv = *reinterpret_cast<const double2 *>(&rp[C::OZ + wz0 + 2 * tq]);
                const double b00 = wyv.x * wzv.x, b01 = wyv.x * wzv.y, b10 = wyv.y * wzv.x, b11 = wyv.y * wzv.y;
                const int a0 = S.wlist[warp][q + 2 * tq], a1 = S.wlist[warp][q + 2 * tq + 1];
                double p0[3] = {0.0, 0.0, 0.0}, p1[3] = {0.0, 0.0, 0.0};
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const double wx0 = T.rec[a0][lx[mt]], wx1 = T.rec[a1][lx[mt]];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double d[2] = {0.0, 0.0};
                        dmma(d, acc[mt][c][0][0], b00); dmma(d, acc[mt][c][0][1], b01);
                        dmma(d, acc[mt][c][1][0], b10); dmma(d, acc[mt][c][1][1], b11);
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
template <int P, int NWY, int NWZ>
__global__ void k_reduce_slots(SeGeom g, const short4 *__restrict__ anchor, const double *__restrict__ part,
                               double *__restrict__ uF)
{
    typedef Cfg<P, NWY, NWZ> C;
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

template <int P, int NWY, int NWZ, bool SPREAD>
cudaError_t launch(se_plan *p, cudaStream_t s)
{
    typedef Cfg<P, NWY, NWZ> C;
    const SeGeom &g = p->g;
    static bool attr_set = false;
    const size_t smem = sizeof(Smem<P, NWY, NWZ, SPREAD>);
    auto kern = k_mma<P, NWY, NWZ, SPREAD>;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int ntY = (g.M + C::BY - 1) / C::BY, ntZ = (g.M + C::BZ - 1) / C::BZ;
    const int nchunk = SPREAD ? g.nchunk : g.nchunk_g2p;
    kern<<<(unsigned)(nchunk * ntY * ntZ), C::NT, smem, s>>>(g, p->anchor, (const double *)p->wtab,
                                                             (const double *)p->fs_grid, p->bin_start,
                                                             (double *)p->grid, (double *)p->uFpart);
    p->launches += 1;
    if (!SPREAD) {
        k_reduce_slots<P, NWY, NWZ><<<(unsigned)((g.N + 255) / 256), 256, 0, s>>>(
            g, p->anchor, (const double *)p->uFpart, (double *)p->uF);
        p->launches += 1;
    }
    return cudaGetLastError();
}

template <bool SPREAD>
cudaError_t dispatch(se_plan *p, cudaStream_t s)
{
    switch (p->g.P) {
    case 24: return launch<24, SE_MMA_NWY, SE_MMA_NWZ, SPREAD>(p, s);
    case 16: return launch<16, SE_MMA_NWY, SE_MMA_NWZ, SPREAD>(p, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace

bool se_mma_supported(int P, int precision) { return precision == SE_FP64 && (P == 24 || P == 16); }
int se_mma_slots(int P)
{
    return P == 24 ? Cfg<24, SE_MMA_NWY, SE_MMA_NWZ>::NSB * Cfg<24, SE_MMA_NWY, SE_MMA_NWZ>::NSC
                   : Cfg<16, SE_MMA_NWY, SE_MMA_NWZ>::NSB * Cfg<16, SE_MMA_NWY, SE_MMA_NWZ>::NSC;
}
cudaError_t se_launch_mma_p2g(se_plan *p, cudaStream_t s) { return dispatch<true>(p, s); }
cudaError_t se_launch_mma_g2p(se_plan *p, cudaStream_t s) { return dispatch<false>(p, s); }
