// K2: near-field P2P,  u^N_i = sum_j sum_p [0 < |r| <= rc] G^N(r) f_j,  r = x_i - x_j + p
// (eq. (2.2), eq. (2.3)), over the 27 colleague cells.
//
// Design.  Only ~15% of the candidates in the 27 colleague cells are inside the cutoff sphere, so the paper's
// thread-per-target loop runs the expensive erfc/exp code at ~15% lane utilisation, and on
// B200 the FP64 pipe (64 lanes per SM) is the scarce resource.  Here a LANE owns a target (32 consecutive
// targets of the near-sorted order per warp) and the work is split by pipe:
//   phase A (filter; packed FP16, two sources per instruction; sources fetched 32 at a time as 16 pair records, one
//            coalesced 16-byte load per lane one chunk ahead, and broadcast from a shared-memory line): the warp walks
//            the sources of the colleague cells; every lane forms r^2 to its own target from the FP16 pair records
//            `xp` K1 wrote (coordinates relative to the particle's cell in units of the cell width, so periodic images
//            cost nothing): 3 HADD2, HMUL2, 2 HFMA2 and one packed compare per PAIR of sources, whose two predicates
//            guard the appends of the source indices to the lane's OWN ring queue in shared memory (predicated
//            stores; no ballot, no compaction; ~10 instructions per 32 pair tests).  The threshold carries a margin
//            that bounds the FP16 rounding (p2p_impl below), so no in-range pair is lost; the ~2 % extra ones are
//            rejected exactly in phase B.  (P2P_HALF2 = 0 selects the first design, the same test in FP32 from `xq`:
//            15 instructions per 32 tests.)
//   phase B (heavy; FP64 pipe, FP32 for fp32 plans): in a round every lane pops one pair of its own queue:
//            exact r from the full-precision coordinates in the form of eq. (2.2), x_i - (x_j + p), the exact
//            test 0 < r^2 <= rc^2 (reading S6), and G^N evaluated in registers as
//              C1 = A - B,  C2 = (A + B)/r^2,  A = erfc(xi r)/r = 1/r - xi erf(x)/x (x = xi r),  B = 2 xi e^{-x^2}/sqrt(pi),
//            erf(x)/x being the rational p(x^2)/q(x^2) of PAPER.md:429-431 (degree 12 over 12 in double, 6 over 6 in
//            single precision; se_erf_rational.h), 1/r a hardware seed with one correction, e^{-x^2} a degree-11
//            polynomial (expf in single precision): no libm calls, no table look-ups.  (A table-driven erfcx, the first
//            design, is kept behind P2P_F64_RATIONAL = 0 / P2P_F32_RATIONAL = 0: same accuracy, 11 shared-memory loads
//            per pair more, and K2 is bound by shared-memory wavefronts before FP64 issue, profiles/r02a.)  Rounds run
//            only when the fullest queue of the warp needs room, so that all lanes stay busy; the lane adds into its
//            own three accumulators (no reduction; double for every plan, an fp32 plan adding one float partial sum
//            per round) and writes u^N_i itself.
// A warp whose targets span several cells processes them in passes: the targets of one z-row of cells whose
// cell index is within P2P_ZSPAN of the first; a lane only accepts sources of its own 27 colleague cells.
// A queue entry is 16 bits: (virtual cell << 9) | offset, a virtual cell being <= 512 consecutive sources of one
// colleague cell; a per-warp table maps it to the first source index and to the periodic image shift p of that
// cell (three reals, written once when the virtual cell is opened).  fp32 plans use cell-relative positions in
// phase B too, so that r keeps full float precision across images (the fresh single-precision path of north_star: the
// rational erf(x)/x, no libm erfc).
#include <cmath>

#include <cuda_fp16.h>

#include "se_common.cuh"
#include "se_erf_rational.h"

namespace {

constexpr int P2P_WARPS = 4;
constexpr int P2P_QC = 128;         // ring-queue slots per lane (power of two), 16-bit entries
constexpr int P2P_CHUNK = 32;       // sources scanned between two queue-room checks
constexpr int P2P_VBITS = 9;        // a queue entry = (virtual cell << VBITS) | offset: virtual cells of <= 512 sources
constexpr int P2P_NV = 64;          // virtual-cell table entries per warp ((NV << VBITS) = 2^15)
#ifndef P2P_TWO
#define P2P_TWO 4
#endif
#ifndef P2P_TWO_F32
#define P2P_TWO_F32 6
#endif
#ifndef P2P_FU
#define P2P_FU 16           /* filter group (sources loaded ahead of the queue stores), fp64 plans */
#endif
#ifndef P2P_FU_F32
#define P2P_FU_F32 8        /* the same for fp32 plans */
#endif
#ifndef P2P_BLOCKS
#define P2P_BLOCKS 4
#endif
#ifndef P2P_BFAN
#define P2P_BFAN 2          /* mode B: pairs per lane and cooperative round, fp64 plans */
#endif
#ifndef P2P_BFAN_F32
#define P2P_BFAN_F32 1      /* the same for fp32 plans */
#endif
#ifndef P2P_BT
#define P2P_BT 8            /* mode B only if the fullest queue could feed this many lanes more than there are non-empty queues */
#endif
#ifndef P2P_A2Q
#define P2P_A2Q 2          /* mode A2 when at least this many quarters of the non-empty queues hold KP pairs */
#endif
#ifndef P2P_HALF2
#define P2P_HALF2 1         /* 1: the filter tests two sources per instruction in packed FP16; 0: one per instruction in FP32 */
#endif
constexpr int P2P_ZSPAN = 6;        // cells along z a pass may span (<= 29: one lane per source cell)

// ---- function tables (built on the host in long double at plan creation) --------------------------------------
// erfcx(x) = e^{x^2} erfc(x) on [0, 8]: 33 pieces centred at i/4 (half-width 1/8), each a polynomial in the local
// variable v = x - i/4 (interpolation at Chebyshev nodes, converted to monomials): degree 10 in double (measured
// relative error < 4e-16), degree 5 in float (< 2e-8 before rounding).  The piece index comes out of the
// round-to-nearest shifter trick (no float <-> int conversion instructions).  Row stride 11 doubles = 22 words: 16
// consecutive rows start in 16 different bank pairs.  For x >= 8 the argument is clamped; e^{-x^2} < 2e-28 there.
// e^t on [-ln2/2, ln2/2]: degree-11 polynomial (Chebyshev interpolant, relative error < 1e-17), kept in constant
// memory so that its coefficients are FMA operands, not loads.
constexpr int MT_NP = 33, MT_DEG = 10, MT_ROW = MT_DEG + 1;
constexpr int MT_DEGF = 5, MT_ROWF = MT_DEGF + 1;
constexpr int MT_F32 = MT_NP * MT_ROW;                           // offset of the float table, in doubles
constexpr int MT_SIZE = MT_F32 + (MT_NP * MT_ROWF + 1) / 2;      // doubles in p->mtab
constexpr int MT_EXPDEG = 11;
__constant__ double c_exp[MT_EXPDEG + 1];
// erf(x)/x ~ p(t)/q(t), t = x^2/36 (se_erf_rational.h, written by gen_erf_rational.py): degree 6 over 6
// for fp32 plans, 12 over 12 for fp64 plans; in constant memory, so that the coefficients are FMA operands, not loads
__constant__ float c_erfr_p32[SE_ERFR_DEG_F32 + 1], c_erfr_q32[SE_ERFR_DEG_F32 + 1];
__constant__ double c_erfr_p64[SE_ERFR_DEG_F64 + 1], c_erfr_q64[SE_ERFR_DEG_F64 + 1];
#ifndef P2P_F32_RATIONAL
#define P2P_F32_RATIONAL 1      /* 1: the rational erf(x)/x of PAPER.md:429-431; 0: the degree-5 erfcx table */
#endif
#ifndef P2P_F64_RATIONAL
#define P2P_F64_RATIONAL 1      /* 1: rational erf(x)/x (no table look-ups: K2 is bound by shared-memory wavefronts); 0: erfcx table */
#endif

template <typename Real> struct NearMath;

template <> struct NearMath<double> {
    static constexpr int TAB = P2P_F64_RATIONAL ? 1 : MT_NP * MT_ROW;     // table entries in shared memory
    static __device__ __forceinline__ void load(double *mt, const double *mtab, int tid, int nt)
    {
        for (int e = tid; e < TAB; e += nt) mt[e] = mtab[e];
    }
    // e^{-y}, y >= 0
    template <bool CLAMP> static __device__ __forceinline__ double exp_neg(double y)
    {
        if (CLAMP) y = fmin(y, 700.0);
        const double SH = 6755399441055744.0;                    // 1.5 * 2^52: round-to-nearest integer shifter
        const double t = fma(y, -1.4426950408889634074, SH);
        const int n = __double2loint(t);                         // n = rint(-y log2 e) <= 0
        const double nf = t - SH;
        double r = fma(nf, -6.93147180369123816490e-01, -y);     // r = -y - n ln2 (ln2 split hi + lo)
        r = fma(nf, -1.90821492927058770002e-10, r);
        double p = c_exp[MT_EXPDEG];
#pragma unroll
        for (int k = MT_EXPDEG - 1; k >= 0; --k) p = fma(p, r, c_exp[k]);
        return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
    }
    template <bool CLAMP> static __device__ __forceinline__ double erfcx_tab(double x, const double *mt)
    {
        const double SH = 6755399441055744.0;
        const double xm = CLAMP ? fmin(x, 8.0) : x;
        const double t = fma(xm, 4.0, SH);                       // piece i = rint(4 x), v = x - i/4
        const double v = fma(t - SH, -0.25, xm);
        const double *c = mt + __double2loint(t) * MT_ROW;
        double p = c[MT_DEG];
#pragma unroll
        for (int k = MT_DEG - 1; k >= 0; --k) p = fma(p, v, c[k]);
        return p;
    }
    // 1/sqrt(x), x > 0 finite: hardware seed (2^-22) and one third-order correction, no special cases
    static __device__ __forceinline__ double rsq(double x)
    {
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        const double e = fma(-(x * y), y, 1.0);
        return fma(y * e, fma(0.375, e, 0.5), y);
    }
    // 1/x, x in [1, 1e6]: hardware seed (2^-23) and two Newton steps
    static __device__ __forceinline__ double rcp(double x)
    {
        double y;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        y = fma(y, fma(-x, y, 1.0), y);
        return fma(y, fma(-x, y, 1.0), y);
    }
    template <bool CLAMP>
    static __device__ __forceinline__ void coeffs(double r2, double xi, double c2, const double *mt, double &C1, double &C2)
    {
        const double rinv = rsq(r2);
        const double x2 = xi * xi * r2;
        const double e = exp_neg<CLAMP>(x2);
#if P2P_F64_RATIONAL
        // erfc(xi r)/r = 1/r - xi erf(x)/x, x = xi r: p and q by Horner (2 x 12 FMA, all coefficients
        // positive: no cancellation), q >= 1; the quotient gets one residual correction.  The difference cancels for
        // large x, which costs nothing: its error, ~1e-16 / r, is that of the two terms, i.e. of every near pair.
        const double t = fmin(x2, 36.0) * (1.0 / 36.0);
        double pn = c_erfr_p64[SE_ERFR_DEG_F64], qn = c_erfr_q64[SE_ERFR_DEG_F64];
#pragma unroll
        for (int k = SE_ERFR_DEG_F64 - 1; k >= 0; --k) { pn = fma(pn, t, c_erfr_p64[k]); qn = fma(qn, t, c_erfr_q64[k]); }
        const double y = rcp(qn);
        double R = pn * y;
        R = fma(fma(-qn, R, pn), y, R);
        double A = fma(-xi, R, rinv);
        if (CLAMP && x2 > 36.0) A = 0.0;
#else
        const double A = e * erfcx_tab<CLAMP>(xi * (r2 * rinv), mt) * rinv;
#endif
        const double B = c2 * e;
        C1 = A - B;
        C2 = (A + B) * (rinv * rinv);
    }
};

template <> struct NearMath<float> {
    static constexpr int TAB = P2P_F32_RATIONAL ? 1 : MT_NP * MT_ROWF;
    static __device__ __forceinline__ void load(float *mt, const double *mtab, int tid, int nt)
    {
        const float *src = reinterpret_cast<const float *>(mtab + MT_F32);
        for (int e = tid; e < TAB; e += nt) mt[e] = src[e];
    }
    template <bool CLAMP> static __device__ __forceinline__ float erfcx_tab(float x, const float *mt)
    {
        const float SH = 12582912.0f;                            // 1.5 * 2^23
        const float xm = CLAMP ? fminf(x, 8.0f) : x;
        const float t = fmaf(xm, 4.0f, SH);
        const float v = fmaf(t - SH, -0.25f, xm);
        const float *c = mt + (__float_as_int(t) - __float_as_int(SH)) * MT_ROWF;
        float p = c[MT_DEGF];
#pragma unroll
        for (int k = MT_DEGF - 1; k >= 0; --k) p = fmaf(p, v, c[k]);
        return p;
    }
    template <bool CLAMP>
    static __device__ __forceinline__ void coeffs(float r2, float xi, float c2, const float *mt, float &C1, float &C2)
    {
        float rinv = rsqrtf(r2);
        float x2 = xi * xi * r2;
        float e = expf(-x2);
#if P2P_F32_RATIONAL
        // erfc(xi r)/r = 1/r - xi erf(x)/x, x = xi r: p and q by Horner (2 x 6 FMA, all coefficients
        // positive), one fast division; beyond x = 6 erf(x)/x = 1/x to rounding, i.e. the term vanishes
        const float t = fminf(x2, 36.f) * (1.f / 36.f);
        float pn = c_erfr_p32[SE_ERFR_DEG_F32], qn = c_erfr_q32[SE_ERFR_DEG_F32];
#pragma unroll
        for (int k = SE_ERFR_DEG_F32 - 1; k >= 0; --k) { pn = fmaf(pn, t, c_erfr_p32[k]); qn = fmaf(qn, t, c_erfr_q32[k]); }
        float A = fmaf(-xi, __fdividef(pn, qn), rinv);
        if (CLAMP && x2 > 36.f) A = 0.f;
#else
        float A = e * erfcx_tab<CLAMP>(xi * (r2 * rinv), mt) * rinv;
#endif
        float B = c2 * e;
        C1 = A - B;
        C2 = (A + B) * (rinv * rinv);
    }
};

// CLAMP: xi rc is so large that the arguments of the function approximations must be clamped (other plans never leave
// their range: every evaluated pair has r <= rc, a rejected one is evaluated at r = rc)
// what k_p2p needs of the plan's geometry: a compact by-value parameter (see the note at SeGeom)
struct P2PGeom {
    int64_t N;
    int ncell, pad_;
    double L, xi, rc, wcell;
};

template <typename Real, bool CLAMP>
__global__ void __launch_bounds__(P2P_WARPS * 32, P2P_BLOCKS)
k_p2p(P2PGeom g, const float4 *__restrict__ xq, const uint4 *__restrict__ xp, int64_t ns, const Real *__restrict__ src,
      const int *__restrict__ cell_start,
      const float4 *__restrict__ xq_t, const Real *__restrict__ src_t, const int *__restrict__ cellp,
      const double *__restrict__ mtab, Real *__restrict__ uN, float rc2m)
{
    // sources: xq, src, cell_start (near order of the source set); targets (g.N of them): xq_t, src_t, cellp (near order
    // of the target set -- the same arrays when the targets are the sources)
    __shared__ Real mt[NearMath<Real>::TAB];
    NearMath<Real>::load(mt, mtab, threadIdx.x, P2P_WARPS * 32);
    __syncthreads();
    __shared__ unsigned short qsm[P2P_WARPS][P2P_QC][32];
    __shared__ int vtab[P2P_WARPS][P2P_NV];                      // virtual cell -> sorted index of its first source
    __shared__ Real vshift[P2P_WARPS][P2P_NV][3];                // virtual cell -> periodic image shift of its sources
    __shared__ int vzcell[P2P_WARPS][P2P_NV];                    // cell-relative plans: unwrapped z cell of the sources
    __shared__ float4 sbuf[P2P_WARPS][P2P_CHUNK];                // the chunk of sources being tested (broadcast reads)

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int nc = g.ncell;
    const Real rc2 = (Real)(g.rc * g.rc);
    const Real xi = (Real)g.xi;
    const Real c2 = (Real)(2.0 * g.xi / sqrt(SE_PI));
    const Real Lr = (Real)g.L, wc = (Real)g.wcell;
#if !P2P_HALF2
    const float wf = (float)g.wcell;
    constexpr float FAR = 1.0e18f;                               // coordinate of a lane that must not match
#endif
    char *const Qb = reinterpret_cast<char *>(&qsm[w][0][lane]); // this lane's queue column, slot stride 64 B
    constexpr int QSTRIDE = 64, QBYTES = P2P_QC * QSTRIDE;
    int *const VT = vtab[w];
    Real (*const VS)[3] = vshift[w];
    int *const VZ = vzcell[w];
    constexpr bool REL = sizeof(Real) == 4;                      // fp32 plans: cell-relative coordinates (g.rel_coords)
    float4 *const SB = sbuf[w];
    int nv = 0, nv_drained = 0;                                  // virtual cells opened / opened at the last full drain

    const int64_t i = ((int64_t)blockIdx.x * P2P_WARPS + w) * 32 + lane;
    const bool valid = i < g.N;
    const int64_t ic = valid ? i : g.N - 1;
    const float4 qi = xq_t[ic];
#if P2P_HALF2
    const float inv_wf = (float)(1.0 / g.wcell);
    const float ux = qi.x * inv_wf, uy = qi.y * inv_wf, uz = qi.z * inv_wf;      // target, in units of the cell width
    const __half2 thr2 = __halves2half2(__float2half_ru(rc2m), __float2half_ru(rc2m));
    const unsigned qb_s = (unsigned)__cvta_generic_to_shared(Qb);
    const uint4 *const xpo = xp + SE_XP_LEN(ns);                  // the odd-pair array
    constexpr float FAR_T = 200.f;                               // target coordinate of a lane that must not match
    const unsigned far2 = 0xd640d640u;                           // (-100, -100) in FP16: a source that is never in range
#endif
    const int pci = cellp[ic];
    const int cz = pci & 1023;
    const Real X0 = src_t[6 * ic + 0], X1 = src_t[6 * ic + 1], X2 = src_t[6 * ic + 2];
    // accumulators are double for every plan: an fp32 plan sums the pairs of one round in float and adds that partial sum
    // here, so that the error of u^N does not grow with the number of neighbours
    double a0 = 0, a1 = 0, a2 = 0;
    int woff = 0, roff = 0;                                      // ring write / read offsets (bytes); empty when equal

    auto queued = [&]() { return ((woff - roff) & (QBYTES - 1)) / QSTRIDE; };
    // One round of phase B.  Mode A (balanced): every lane with a queued pair pops and evaluates one of its own.
    // Mode B (imbalanced: at least P2P_BT fewer non-empty queues than the fullest one could feed; a measured threshold: with
    // fewer idle lanes a plain round is cheaper than the reduction): the 32 lanes evaluate pairs of the fullest queue together
    // and a butterfly sum hands the result to its owner.  The choice is a pure
    // function of the queue lengths, so the summation order stays deterministic.
    // one pair: queue entry at byte offset qo of this lane's (or, mode B, the owner's) column -> contribution d
    // keep = false: evaluate but contribute nothing; d0..d2 are ADDED to (fused into the last FMAs)
    auto pair = [&](int qo, bool keep, Real T0, Real T1, Real T2, int tcz, Real &d0, Real &d1, Real &d2) {
        const int e = *reinterpret_cast<const unsigned short *>(Qb + qo);
        const int j = VT[e >> P2P_VBITS] + (e & ((1 << P2P_VBITS) - 1));
        const Real *sp = src + 6 * (int64_t)j;
        Real xj, yj, zj, f0, f1, f2;
        if (sizeof(Real) == 8) {
            const double2 p0 = __ldg(reinterpret_cast<const double2 *>(sp));
            const double2 p1 = __ldg(reinterpret_cast<const double2 *>(sp + 2));
            const double2 p2 = __ldg(reinterpret_cast<const double2 *>(sp + 4));
            xj = (Real)p0.x; yj = (Real)p0.y; zj = (Real)p1.x; f0 = (Real)p1.y; f1 = (Real)p2.x; f2 = (Real)p2.y;
        } else {
            const float2 p0 = __ldg(reinterpret_cast<const float2 *>(sp));
            const float2 p1 = __ldg(reinterpret_cast<const float2 *>(sp + 2));
            const float2 p2 = __ldg(reinterpret_cast<const float2 *>(sp + 4));
            xj = (Real)p0.x; yj = (Real)p0.y; zj = (Real)p1.x; f0 = (Real)p1.y; f1 = (Real)p2.x; f2 = (Real)p2.y;
        }
        // periodic image of the source as this target sees it: the virtual cell's shift (absolute coordinates:
        // a multiple of L per axis; cell-relative coordinates: the cell offset, in z the INTEGER cell difference to
        // the target's own cell times the cell width, so that the shift carries one rounding, like x and y)
        const Real *vs = VS[e >> P2P_VBITS];
        const Real sx = vs[0], sy = vs[1];
        const Real sz = REL ? (Real)(VZ[e >> P2P_VBITS] - tcz) * wc : vs[2];
        const Real rx = T0 - (xj + sx), ry = T1 - (yj + sy), rz = T2 - (zj + sz);
        Real r2 = rx * rx + ry * ry + rz * rz;
        const bool ok = keep && (r2 <= rc2) && (r2 > (Real)0);
        if (!ok) r2 = rc2;                                       // stays inside the function tables
        Real C1, C2;
        NearMath<Real>::template coeffs<CLAMP>(r2, xi, c2, mt, C1, C2);
        if (!ok) { C1 = (Real)0; C2 = (Real)0; }
        const Real rf = C2 * (rx * f0 + ry * f1 + rz * f2);
        d0 = fma(rf, rx, fma(C1, f0, d0));
        d1 = fma(rf, ry, fma(C1, f1, d1));
        d2 = fma(rf, rz, fma(C1, f2, d2));
    };
    constexpr int KP = sizeof(Real) == 8 ? P2P_TWO : P2P_TWO_F32;   // pairs per lane and round in mode A2
    auto round = [&]() {
        const int c = queued();
        const unsigned m1 = __ballot_sync(0xffffffffu, c > 0);
        const int cmax = __reduce_max_sync(0xffffffffu, c);
        const int cB = min(cmax, 32);
        if (cB > __popc(m1) + P2P_BT) {                          // mode B (warp-uniform)
            const int o = __ffs(__ballot_sync(0xffffffffu, c == cmax)) - 1;
            const Real T0 = __shfl_sync(0xffffffffu, X0, o), T1 = __shfl_sync(0xffffffffu, X1, o);
            const Real T2 = __shfl_sync(0xffffffffu, X2, o);
            const int tcz = __shfl_sync(0xffffffffu, cz, o);
            // up to KB pairs per lane (entries lane, lane + 32, ... of the owner's queue), evaluated side by side like the
            // pairs of mode A2, then ONE butterfly: independent dependency chains, and the reduction is paid once per
            // 32 KB pairs (config 5 spends half of its pairs here).  A lane past the end re-evaluates the owner's last entry
            // and drops it.
            constexpr int KB = sizeof(Real) == 8 ? P2P_BFAN : P2P_BFAN_F32;
            const int nB = cmax >= 32 ? min(cmax & ~31, 32 * KB) : cmax;      // whole waves of 32 pairs, or the rest
            const int ro0 = __shfl_sync(0xffffffffu, roff, o);
            Real d0 = 0, d1 = 0, d2 = 0;
#pragma unroll
            for (int k = 0; k < KB; ++k) {
                if (32 * k < nB) {                               // warp-uniform
                    const int idx = lane + 32 * k;
                    const int qo = (ro0 + min(idx, nB - 1) * QSTRIDE) & (QBYTES - 1);
                    pair((o - lane) * 2 + qo, idx < nB, T0, T1, T2, tcz, d0, d1, d2);
                }
            }
#pragma unroll
            for (int sh = 16; sh > 0; sh >>= 1) {
                d0 += __shfl_xor_sync(0xffffffffu, d0, sh);
                d1 += __shfl_xor_sync(0xffffffffu, d1, sh);
                d2 += __shfl_xor_sync(0xffffffffu, d2, sh);
            }
            if (lane == o) { a0 += (double)d0; a1 += (double)d1; a2 += (double)d2; roff = (roff + nB * QSTRIDE) & (QBYTES - 1); }
        } else if (KP > 1 && __popc(__ballot_sync(0xffffffffu, c >= KP)) * 4 >= __popc(m1) * P2P_A2Q) {
            // mode A2: at least P2P_A2Q quarters of the non-empty queues hold KP pairs: every lane pops up to that many of its own, evaluated side
            // by side (independent dependency chains); a lane with fewer re-evaluates its last one and drops it
            if (c > 0) {
                int ro = roff;
                if (sizeof(Real) == 8) {
                    Real t0 = (Real)a0, t1 = (Real)a1, t2 = (Real)a2;        // fp64: the accumulators themselves
#pragma unroll
                    for (int k = 0; k < KP; ++k) {
                        pair(ro, k < c, X0, X1, X2, cz, t0, t1, t2);
                        if (k + 1 < c) ro = (ro + QSTRIDE) & (QBYTES - 1);
                    }
                    a0 = t0; a1 = t1; a2 = t2;
                } else {
                    Real t0 = 0, t1 = 0, t2 = 0;
#pragma unroll
                    for (int k = 0; k < KP; ++k) {
                        pair(ro, k < c, X0, X1, X2, cz, t0, t1, t2);
                        if (k + 1 < c) ro = (ro + QSTRIDE) & (QBYTES - 1);
                    }
                    a0 += (double)t0; a1 += (double)t1; a2 += (double)t2;
                }
                roff = (roff + min(c, KP) * QSTRIDE) & (QBYTES - 1);
            }
        } else if (c > 0) {                                      // mode A: every lane pops one pair of its own
            if (sizeof(Real) == 8) {
                Real t0 = (Real)a0, t1 = (Real)a1, t2 = (Real)a2;
                pair(roff, true, X0, X1, X2, cz, t0, t1, t2);
                a0 = t0; a1 = t1; a2 = t2;
            } else {
                Real t0 = 0, t1 = 0, t2 = 0;
                pair(roff, true, X0, X1, X2, cz, t0, t1, t2);
                a0 += (double)t0; a1 += (double)t1; a2 += (double)t2;
            }
            roff = (roff + QSTRIDE) & (QBYTES - 1);
        }
    };

    unsigned remaining = __ballot_sync(0xffffffffu, valid);
    while (remaining) {
        // ---- pass: the targets of the first remaining lane's z-row whose cell is at most P2P_ZSPAN further ----
        const int leader = __ffs(remaining) - 1;
        const int pl = __shfl_sync(0xffffffffu, pci, leader);
        const int cxl = pl >> 20, cyl = (pl >> 10) & 1023, czl = pl & 1023;
        const int dzl = cz - czl;                                // this lane's cell, in cells from the leader's
        const bool member = valid && (pci >> 10) == (pl >> 10) && dzl >= 0 && dzl <= P2P_ZSPAN;
        const unsigned act = __ballot_sync(0xffffffffu, member) & remaining;
        const int span = __reduce_max_sync(0xffffffffu, member ? dzl : 0);
        const int ncl = span + 3;                                // source cells k = 0 .. ncl-1 <-> cell czl - 1 + k
#if !P2P_HALF2
        const float tx0 = ((act >> lane) & 1u) ? qi.x : FAR;
#endif

        // colleague rows in centre-out order, alternating sides, and the cells of a row centre-out as well: every
        // lane then receives its hits at a roughly steady rate, which keeps all 32 queues non-empty
#pragma unroll 1
        for (int rr = 0; rr < 9; ++rr) {
            const int dx = ((0x22161 >> (2 * rr)) & 3) - 1, dy = ((0x0a215 >> (2 * rr)) & 3) - 1;
            int nx = cxl + dx, ny = cyl + dy;
            if (nx < 0) nx += nc; else if (nx >= nc) nx -= nc;
            if (ny < 0) ny += nc; else if (ny >= nc) ny -= nc;
#if P2P_HALF2
            const __half2 hx2 = __float2half2_rn((((act >> lane) & 1u) ? ux : FAR_T) - (float)dx);
            const __half2 hy2 = __float2half2_rn(uy - (float)dy);
#else
            const float tx = tx0 - (float)dx * wf, ty = qi.y - (float)dy * wf;
#endif
            // lane k holds the CSR range of source cell k of this row
            int cb = 0, ce = 0;
            if (lane < ncl) {
                int zc = czl - 1 + lane;
                zc %= nc; if (zc < 0) zc += nc;
                const int *cs = cell_start + (size_t)(nx * nc + ny) * nc + zc;
                cb = __ldg(cs); ce = __ldg(cs + 1);
            }
            const int mid = ncl >> 1;
#pragma unroll 1
            for (int kk = 0; kk < ncl; ++kk) {
                const int k = mid + ((kk & 1) ? -((kk + 1) >> 1) : (kk >> 1));
                const int jb = __shfl_sync(0xffffffffu, cb, k), je = __shfl_sync(0xffffffffu, ce, k);
                // a lane accepts the cell only if it is one of its own three colleague cells of this row
                const int dk = k - 1 - dzl;
#if P2P_HALF2
                const __half2 hz2 = __float2half2_rn((dk >= -1 && dk <= 1) ? uz - (float)dk : FAR_T);
#else
                const float tz = (dk >= -1 && dk <= 1) ? qi.z - (float)dk * wf : FAR;
#endif
#pragma unroll 1
                for (int v0 = jb; v0 < je; v0 += (1 << P2P_VBITS)) {
                    // open a virtual cell; its table slot may still be referenced by queued entries of the
                    // virtual cell P2P_NV earlier: drain everything before wrapping around
                    if (nv - nv_drained >= P2P_NV) {
                        while (__any_sync(0xffffffffu, woff != roff)) round();
                        nv_drained = nv;
                    }
                    const int vslot = nv & (P2P_NV - 1);
                    ++nv;
                    __syncwarp();
                    if (lane < 3) {
                        // lane a writes the shift along axis a (x, y, z)
                        const int zu = czl - 1 + k;              // unwrapped z cell of the sources
                        const int cu = lane == 0 ? cxl + dx : (lane == 1 ? cyl + dy : zu);
                        Real sh;
                        if (REL) sh = (Real)(lane == 0 ? dx : (lane == 1 ? dy : 0)) * wc;
                        else sh = cu < 0 ? -Lr : (cu >= nc ? Lr : (Real)0);
                        VS[vslot][lane] = sh;
                        if (lane == 0) VT[vslot] = v0;
                        if (lane == 2) VZ[vslot] = zu;
                    }
                    __syncwarp();
                    const int ve = min(je, v0 + (1 << P2P_VBITS));
#if P2P_HALF2
                    // The 32 sources of a chunk are 16 FP16 pair records (K1: relative to the cell, in units of its width):
                    // lanes 0..15 fetch one each, one chunk ahead, and the warp reads them back as broadcasts.  A cell pairs
                    // its sources up from its first one (even or odd pair array by the parity of that index); a half past
                    // the cell's end is replaced by a coordinate that is never in range.
                    const uint4 *const xpc = (v0 & 1) ? xpo : xp;
                    auto load_pair = [&](int j0) {
                        uint4 r = make_uint4(far2, far2, far2, 0u);
                        const int s0 = j0 + 2 * lane;
                        if (lane < 16 && s0 < ve) {
                            r = __ldg(xpc + (s0 >> 1));
                            if (s0 + 1 >= ve) { r.x = (r.x & 0xffffu) | (far2 << 16); r.y = (r.y & 0xffffu) | (far2 << 16); r.z = (r.z & 0xffffu) | (far2 << 16); }
                        }
                        return r;
                    };
                    uint4 nxt = load_pair(v0);
                    uint4 *const SB2 = reinterpret_cast<uint4 *>(SB);
#pragma unroll 1
                    for (int j0 = v0; j0 < ve; j0 += P2P_CHUNK) {
                        const uint4 cur = nxt;
                        nxt = load_pair(j0 + P2P_CHUNK);
                        while (__any_sync(0xffffffffu, queued() > P2P_QC - 1 - P2P_CHUNK)) round();
                        const int n2 = (min(P2P_CHUNK, ve - j0) + 1) >> 1;       // pairs in this chunk
                        if (lane < 16) SB2[lane] = cur;
                        __syncwarp();
                        const int ebase = (vslot << P2P_VBITS) + (j0 - v0);
                        // groups of FU2 pairs: all broadcast loads of a group first; per pair 3 HADD2, 1 HMUL2, 2 HFMA2 and one
                        // packed compare whose two predicates guard the two queue pushes
                        constexpr int FU2 = 8;
#pragma unroll 1
                        for (int pb = 0; pb < n2; pb += FU2) {
                            uint4 q[FU2];
#pragma unroll
                            for (int u = 0; u < FU2; ++u) q[u] = SB2[pb + u];
#pragma unroll
                            for (int u = 0; u < FU2; ++u) {
                                const __half2 rx = __hsub2(hx2, *reinterpret_cast<const __half2 *>(&q[u].x));
                                const __half2 ry = __hsub2(hy2, *reinterpret_cast<const __half2 *>(&q[u].y));
                                const __half2 rz = __hsub2(hz2, *reinterpret_cast<const __half2 *>(&q[u].z));
                                const __half2 r2 = __hfma2(rz, rz, __hfma2(ry, ry, __hmul2(rx, rx)));
                                const unsigned short e0 = (unsigned short)(ebase + 2 * (pb + u)), e1 = (unsigned short)(e0 + 1);
                                asm volatile("{\n"
                                             ".reg .pred p, q;\n"
                                             ".reg .b32 a;\n"
                                             "setp.le.f16x2 p|q, %1, %2;\n"
                                             "add.u32 a, %3, %0;\n"
                                             "@p st.shared.u16 [a], %4;\n"
                                             "@p add.u32 %0, %0, 64;\n"
                                             "@p and.b32 %0, %0, %6;\n"
                                             "add.u32 a, %3, %0;\n"
                                             "@q st.shared.u16 [a], %5;\n"
                                             "@q add.u32 %0, %0, 64;\n"
                                             "@q and.b32 %0, %0, %6;\n"
                                             "}"
                                             : "+r"(woff)
                                             : "r"(*reinterpret_cast<const unsigned *>(&r2)), "r"(*reinterpret_cast<const unsigned *>(&thr2)),
                                               "r"(qb_s), "h"(e0), "h"(e1), "r"(QBYTES - 1)
                                             : "memory");
                            }
                        }
#else
                    // the 32 sources of a chunk are fetched with one coalesced 16-byte load per lane, one chunk
                    // ahead (the load of chunk k + 1 is in flight while chunk k is tested), and broadcast through
                    // a per-warp shared-memory line
                    float4 nxt = make_float4(FAR, FAR, FAR, 0.f);
                    if (v0 + lane < ve) nxt = __ldg(xq + v0 + lane);
#pragma unroll 1
                    for (int j0 = v0; j0 < ve; j0 += P2P_CHUNK) {
                        const float4 cur = nxt;
                        nxt = make_float4(FAR, FAR, FAR, 0.f);
                        if (j0 + P2P_CHUNK + lane < ve) nxt = __ldg(xq + j0 + P2P_CHUNK + lane);
                        while (__any_sync(0xffffffffu, queued() > P2P_QC - 1 - P2P_CHUNK)) round();
                        const int n = min(P2P_CHUNK, ve - j0);
                        SB[lane] = cur;                          // entries past the cell's end are FAR: never in range
                        __syncwarp();
                        const int ebase = (vslot << P2P_VBITS) + (j0 - v0);
                        // groups of P2P_FU sources: all broadcast loads of a group first (the queue stores that
                        // follow are shared-memory stores the compiler must order against later loads)
                        constexpr int FU = sizeof(Real) == 8 ? P2P_FU : P2P_FU_F32;
#pragma unroll 1
                        for (int jb = 0; jb < n; jb += FU) {
                            float4 q[FU];
#pragma unroll
                            for (int u = 0; u < FU; ++u) q[u] = SB[jb + u];
#pragma unroll
                            for (int u = 0; u < FU; ++u) {
                                const float rx = tx - q[u].x, ry = ty - q[u].y, rz = tz - q[u].z;
                                if (rx * rx + ry * ry + rz * rz <= rc2m) {
                                    *reinterpret_cast<unsigned short *>(Qb + woff) = (unsigned short)(ebase + jb + u);
                                    woff = (woff + QSTRIDE) & (QBYTES - 1);
                                }
                            }
                        }
#endif
                        __syncwarp();
                    }
                }
            }
        }
        remaining &= ~act;
    }
    while (__any_sync(0xffffffffu, woff != roff)) round();
    if (valid) { uN[3 * i + 0] = (Real)a0; uN[3 * i + 1] = (Real)a1; uN[3 * i + 2] = (Real)a2; }
}

// Diagnostics for bench.py's K2 roofline (not on the evaluation path): candidates (sources in the 27 colleague cells) and
// in-range pairs (0 < r <= rc) summed over all targets, from the FP32 cell-relative copies, one thread per target.
__global__ void __launch_bounds__(256)
k_count_pairs(SeGeom g, const float4 *__restrict__ xq, const int *__restrict__ cell_start, const float4 *__restrict__ xq_t,
              const int *__restrict__ cellp, unsigned long long *__restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long cand = 0, hit = 0;
    if (i < g.N) {
        const float4 qi = xq_t[i];
        const int pc = cellp[i], nc = g.ncell;
        const int cx = pc >> 20, cy = (pc >> 10) & 1023, cz = pc & 1023;
        const float wf = (float)g.wcell, rc2 = (float)(g.rc * g.rc);
        for (int dx = -1; dx <= 1; ++dx)
        for (int dy = -1; dy <= 1; ++dy)
        for (int dz = -1; dz <= 1; ++dz) {
            const int nx = (cx + dx + nc) % nc, ny = (cy + dy + nc) % nc, nz = (cz + dz + nc) % nc;
            const int *cs = cell_start + (size_t)(nx * nc + ny) * nc + nz;
            const int jb = cs[0], je = cs[1];
            cand += (unsigned long long)(je - jb);
            for (int j = jb; j < je; ++j) {
                const float4 q = __ldg(xq + j);
                const float rx = qi.x - q.x - dx * wf, ry = qi.y - q.y - dy * wf, rz = qi.z - q.z - dz * wf;
                const float r2 = rx * rx + ry * ry + rz * rz;
                hit += (r2 <= rc2 && r2 > 0.f) ? 1u : 0u;
            }
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        cand += __shfl_down_sync(0xffffffffu, cand, o);
        hit += __shfl_down_sync(0xffffffffu, hit, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(out, cand); atomicAdd(out + 1, hit); }
}

template <typename Real>
cudaError_t p2p_impl(se_plan *p, cudaStream_t s)
{
    SeGeom g = p->g;
    g.N = p->T.n;                                                // a lane per target
    const SeSet &S = p->S, &T = p->T;
    int64_t per_block = (int64_t)P2P_WARPS * 32;
    unsigned nblk = (unsigned)((g.N + per_block - 1) / per_block);
#if P2P_HALF2
    // Filter threshold on r^2 in units of the cell width w (rho = rc / w <= 1), in FP16 arithmetic.  Rounding moves a source
    // (s in [0, 1)) by at most 2^-12, a target (|t| < 2) by 2^-11 and their difference (|d| <= 1 for a pair in range) by
    // 2^-11 per component: |d - r_c| <= 1.22e-3, so sum d^2 <= rho^2 + 4.3e-3 rho + 4.5e-6; the three roundings of the sum
    // add at most 3 x 2^-11 of it.  The threshold is rounded up to FP16; ~1.7 % of the candidates it lets through are out
    // of range and rejected exactly in phase B.
    const double rho = g.rc / g.wcell;
    const double rc2m = (rho * rho + 4.3e-3 * rho + 4.5e-6) * (1.0 + 1.5e-3) + 1e-4;
#else
    // FP32 filter margin: the cell-relative coordinates are < 2 wcell in magnitude, each rounded to 6e-8
    // relative, so |dr| < 1e-6 wcell per component and |d r^2| < 2 sqrt(3) rc 1e-6 wcell
    const double rc2m = g.rc * g.rc * (1.0 + 1e-5) + 4e-6 * g.rc * g.wcell;
#endif
    // CLAMP instantiation: plans whose arguments can leave the range of the function approximations (x = xi r <= 6 for
    // the rational erf(x)/x, 7.8 for the erfcx tables); every evaluated pair has r <= rc
    const bool rational = p->precision == SE_FP64 ? P2P_F64_RATIONAL != 0 : P2P_F32_RATIONAL != 0;
    const P2PGeom pg{g.N, g.ncell, 0, g.L, g.xi, g.rc, g.wcell};
    if (g.xi * g.rc > (rational ? 5.99 : 7.8))
        k_p2p<Real, true><<<nblk, P2P_WARPS * 32, 0, s>>>(pg, (const float4 *)S.xq, (const uint4 *)S.xp, S.n, (const Real *)S.src_near, S.cell_start,
                                                         (const float4 *)T.xq, (const Real *)T.src_near, T.cell_sorted,
                                                         p->mtab, (Real *)p->uN, (float)rc2m);
    else
        k_p2p<Real, false><<<nblk, P2P_WARPS * 32, 0, s>>>(pg, (const float4 *)S.xq, (const uint4 *)S.xp, S.n, (const Real *)S.src_near, S.cell_start,
                                                          (const float4 *)T.xq, (const Real *)T.src_near, T.cell_sorted,
                                                          p->mtab, (Real *)p->uN, (float)rc2m);
    p->launches += 1;
    return cudaGetLastError();
}

}  // namespace

// Host side of the function tables: interpolate at Chebyshev nodes in long double, convert to monomials.
void se_cheb_fit(long double (*fn)(long double, const void *), const void *ctx, long double c, long double hw, int deg,
                 double *out)
{
    const int n = deg + 1;
    const long double PI = 3.14159265358979323846264338327950288L;
    long double fv[24], ch[24], T[24][24] = {}, mono[24] = {};
    for (int k = 0; k < n; ++k) fv[k] = fn(c + hw * cosl(PI * (k + 0.5L) / n), ctx);
    for (int j = 0; j < n; ++j) {
        long double a = 0;
        for (int k = 0; k < n; ++k) a += fv[k] * cosl(PI * j * (k + 0.5L) / n);
        ch[j] = (j == 0 ? 1.0L : 2.0L) * a / n;
    }
    T[0][0] = 1; if (n > 1) T[1][1] = 1;
    for (int j = 2; j < n; ++j)
        for (int i = 0; i <= j; ++i) T[j][i] = (i > 0 ? 2 * T[j - 1][i - 1] : 0) - T[j - 2][i];
    for (int j = 0; j < n; ++j)
        for (int i = 0; i <= j; ++i) mono[i] += ch[j] * T[j][i];
    for (int i = 0; i < n; ++i) out[i] = (double)mono[i];
}
static long double erfcx_l(long double x, const void *) { return expl(x * x) * erfcl(x); }
static long double exp_l(long double x, const void *) { return expl(x); }

cudaError_t se_build_mtab(se_plan *p)
{
    static_assert(MT_DEG < 24 && MT_EXPDEG < 24, "cheb_fit scratch");
    double h[MT_SIZE] = {};
    float *hf = reinterpret_cast<float *>(h + MT_F32);
    for (int i = 0; i < MT_NP; ++i) {
        // pieces centred at i/4, half-width 1/8; monomials in v = x - i/4: divide by (1/8)^k (exact)
        double row[MT_ROW], rowf[MT_ROWF];
        se_cheb_fit(erfcx_l, nullptr, 0.25L * i, 0.125L, MT_DEG, row);
        se_cheb_fit(erfcx_l, nullptr, 0.25L * i, 0.125L, MT_DEGF, rowf);
        double s = 1.0;
        for (int k = 0; k <= MT_DEG; ++k) { h[i * MT_ROW + k] = row[k] * s; s *= 8.0; }
        s = 1.0;
        for (int k = 0; k <= MT_DEGF; ++k) { hf[i * MT_ROWF + k] = (float)(rowf[k] * s); s *= 8.0; }
    }
    // e^t: the polynomial is evaluated in t itself, not in t / hw: rescale the monomials
    double e[MT_EXPDEG + 1], ec[MT_EXPDEG + 1];
    const long double hw = 0.34657359027997265470861606072908828L * 1.0001L;   // ln2 / 2 and a little slack
    se_cheb_fit(exp_l, nullptr, 0.0L, hw, MT_EXPDEG, e);
    long double s = 1;
    for (int k = 0; k <= MT_EXPDEG; ++k) { ec[k] = (double)(e[k] / s); s *= hw; }
    cudaError_t err = cudaMemcpyToSymbol(c_exp, ec, sizeof(ec));
    if (err != cudaSuccess) return err;
    float rp[SE_ERFR_DEG_F32 + 1], rq[SE_ERFR_DEG_F32 + 1];
    for (int k = 0; k <= SE_ERFR_DEG_F32; ++k) { rp[k] = (float)se_erfr_p32[k]; rq[k] = (float)se_erfr_q32[k]; }
    err = cudaMemcpyToSymbol(c_erfr_p32, rp, sizeof(rp));
    if (err != cudaSuccess) return err;
    err = cudaMemcpyToSymbol(c_erfr_q32, rq, sizeof(rq));
    if (err != cudaSuccess) return err;
    err = cudaMemcpyToSymbol(c_erfr_p64, se_erfr_p64, sizeof(se_erfr_p64));
    if (err != cudaSuccess) return err;
    err = cudaMemcpyToSymbol(c_erfr_q64, se_erfr_q64, sizeof(se_erfr_q64));
    if (err != cudaSuccess) return err;
    err = cudaMalloc(&p->mtab, sizeof(h));
    if (err != cudaSuccess) return err;
    p->workspace_bytes += sizeof(h);
    return cudaMemcpy(p->mtab, h, sizeof(h), cudaMemcpyHostToDevice);
}

cudaError_t se_launch_p2p(se_plan *p, cudaStream_t s)
{
    return p->precision == SE_FP64 ? p2p_impl<double>(p, s) : p2p_impl<float>(p, s);
}

// se.h: counts of the last sorted configuration (synchronises the stream it runs on; allocates 16 bytes)
extern "C" se_status se_count_pairs(se_plan *p, int64_t *candidates, int64_t *in_range)
{
    if (!p || !candidates || !in_range) return SE_EINVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) { cudaGetLastError(); return SE_EINVAL; }
    unsigned long long *d = nullptr, h[2] = {0, 0};
    if (cudaMalloc(&d, sizeof(h)) != cudaSuccess) { cudaGetLastError(); return SE_ENOMEM; }
    cudaMemset(d, 0, sizeof(h));
    SeGeom g = p->g;
    g.N = p->T.n;
    k_count_pairs<<<(unsigned)((g.N + 255) / 256), 256>>>(g, (const float4 *)p->S.xq, p->S.cell_start, (const float4 *)p->T.xq,
                                                         p->T.cell_sorted, d);
    cudaError_t e = cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) { cudaGetLastError(); return SE_ECUDA; }
    *candidates = (int64_t)h[0];
    *in_range = (int64_t)h[1];
    return SE_OK;
}
