// K4: Fourier-space scaling (CNV), eq. (2.6) with G^F_hat of PAPER.md:69 eq. (2.4b)
// and the window's transform w_hat(k) = w_hat0(k1) w_hat0(k2) w_hat0(k3):
//   H~hat(k) = s(k) [k^2 Hhat - k (k.Hhat)],
//   s(k) = (1/M^3) 8 pi k^-4 (1 + k^2/4xi^2) e(k1) e(k2) e(k3),   e(k_d) = exp(-k_d^2/4xi^2) / w_hat0(k_d)^2
// (Gaussian window, reading S4: w_hat0 = exp(-eta k_d^2 / 8 xi^2), e = exp(-(1-eta) k_d^2/4xi^2); Kaiser-Bessel:
// the closed-form transform, reading S20; the table of e per 1-D index is built on the host in se_window.cu),
// zero at k = 0 (reading S2) and on the Nyquist planes (reading S8).  One thread per stored
// mode of the R2C half-spectrum (conjugate symmetry).  The exponential factors
// as a product of three 1-D tables built once per plan, so the kernel is pure HBM streaming:
// 3 complex in, 3 complex out per mode.
// Also in this file, for se_eval's fused path ("Own 2-D transforms"): k_xfft_scale (transform over x + K4 +
// inverse transform over x in one kernel), k_zr2c / k_zc2r / k_yfft (the 2-D transforms of the x-planes), and
// se_scale_noalloc (K4 without a plan or an allocation, table in a static device array).
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "se_common.cuh"

namespace {

template <typename Real> struct Cplx;
template <> struct Cplx<double> { typedef double2 type; };
template <> struct Cplx<float> { typedef float2 type; };

// one mode of eq. (2.6): (h0, h1, h2) <- s(k) [k^2 h - k (k . h)]; e = e(k1) e(k2) e(k3) from the table
template <typename Real, typename C>
__device__ __forceinline__ void scale_mode(int M, int ix, int iy, int iz, Real kx, Real ky, Real kz, Real e, Real pref,
                                           Real inv4xi2, C &h0, C &h1, C &h2)
{
    const Real k2 = kx * kx + ky * ky + kz * kz;
    const bool nyq = (2 * ix == M) || (2 * iy == M) || (2 * iz == M);
    Real s = 0;
    if (!nyq && k2 > (Real)0) s = pref * ((Real)1 + k2 * inv4xi2) * e / (k2 * k2);
    const Real kr = kx * h0.x + ky * h1.x + kz * h2.x;
    const Real ki = kx * h0.y + ky * h1.y + kz * h2.y;
    C o0, o1, o2;
    o0.x = s * (k2 * h0.x - kx * kr); o0.y = s * (k2 * h0.y - kx * ki);
    o1.x = s * (k2 * h1.x - ky * kr); o1.y = s * (k2 * h1.y - ky * ki);
    o2.x = s * (k2 * h2.x - kz * kr); o2.y = s * (k2 * h2.y - kz * ki);
    h0 = o0; h1 = o1; h2 = o2;
}

// 1 / x for x > 0 finite, to rounding: hardware seed and two Newton steps (no IEEE division sequence)
__device__ __forceinline__ double fast_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    y = fma(y, fma(-x, y, 1.0), y);
    return fma(y, fma(-x, y, 1.0), y);
}
__device__ __forceinline__ float fast_rcp(float x) { return __frcp_rn(x); }

// the same for K4x: the Nyquist planes are zeros of the table factor e (set by the caller), 1 / k^4 by fast_rcp
template <typename Real, typename C>
__device__ __forceinline__ void scale_mode_x(Real kx, Real ky, Real kz, Real e, Real pref, Real inv4xi2, C &h0, C &h1, C &h2)
{
    const Real k2 = kx * kx + ky * ky + kz * kz;
    Real s = 0;
    if (k2 > (Real)0) s = pref * ((Real)1 + k2 * inv4xi2) * e * fast_rcp(k2 * k2);
    const Real kr = kx * h0.x + ky * h1.x + kz * h2.x;
    const Real ki = kx * h0.y + ky * h1.y + kz * h2.y;
    C o0, o1, o2;
    o0.x = s * (k2 * h0.x - kx * kr); o0.y = s * (k2 * h0.y - kx * ki);
    o1.x = s * (k2 * h1.x - ky * kr); o1.y = s * (k2 * h1.y - ky * ki);
    o2.x = s * (k2 * h2.x - kz * kr); o2.y = s * (k2 * h2.y - kz * ki);
    h0 = o0; h1 = o1; h2 = o2;
}

// ktab layout: [0..M) k value of index i, [M..2M) e(k_i)
template <typename Real>
__global__ void __launch_bounds__(256)
k_scale(int M, int Mh, int y0, int ny, Real pref, Real inv4xi2, const Real *__restrict__ ktab,
        typename Cplx<Real>::type *__restrict__ spec)
{
    // spec: [3][M][ny][Mh], the modes with second index y0 .. y0 + ny - 1 (the whole spectrum: y0 = 0, ny = M)
    typedef typename Cplx<Real>::type C;
    const int iz = blockIdx.x * blockDim.x + threadIdx.x;
    const int iy = y0 + blockIdx.y, ix = blockIdx.z;
    if (iz >= Mh) return;
    const size_t nm = (size_t)M * ny * Mh;
    const size_t idx = ((size_t)ix * ny + blockIdx.y) * Mh + iz;
    C h0 = spec[idx], h1 = spec[nm + idx], h2 = spec[2 * nm + idx];
    scale_mode<Real>(M, ix, iy, iz, ktab[ix], ktab[iy], ktab[iz], ktab[M + ix] * ktab[M + iy] * ktab[M + iz], pref, inv4xi2, h0, h1, h2);
    spec[idx] = h0; spec[nm + idx] = h1; spec[2 * nm + idx] = h2;
}


// ================================================================================================================
// K4x: the transform over x, K4 and the inverse transform over x in ONE kernel (se_eval's path when the plan's
// `xf_ok` is set).  A 3-D transform is a 2-D transform over (y, z) of every x-plane followed by 1-D transforms
// over x; K4 is diagonal in k, and the 1-D transforms over x of different (ky, kz) are independent.  So
//   H --2-D R2C of every x-plane--> [this kernel] --2-D C2R of every x-plane--> H~      (own kernels below, or cuFFT batch 3 M)
// where a block of this kernel owns TZ consecutive kz of one ky for all three components (K4 mixes the
// components, eq. (2.6)): it loads the 3 TZ x-columns (length M, stride M (M/2+1)) into shared memory
// with 16-byte asynchronous copies, runs them through an in-place mixed-radix decimation-in-frequency transform
// (radices 16, 9, 8, 7, 5, 4, 3, 2 in registers, twiddles from a shared table), applies K4 in the digit-reversed
// order the transform leaves (index table per plan), runs the mirror-image decimation-in-time inverse (which
// takes that order and returns the natural one, unnormalised like cuFFT's) and writes the columns back in place.
// Against cuFFT's third pass + k_scale + cuFFT's first inverse pass that is one read and one write of the
// half-spectrum instead of three of each; the arithmetic is the same.  HBM-bound: 2 x 16 (8) bytes per mode.
// Layout in shared memory: element x of column f (= component * TZ + tz) at [x][f], so that the threads of a
// quarter-warp touch 128 contiguous bytes whatever the stride of the stage.
__constant__ double c_cs[17][16][2];      // (cos, sin)(2 pi j / R) for R <= 16, j < R
__constant__ float c_csf[17][16][2];

template <typename Real> struct XfT;
template <> struct XfT<double> {
    typedef double2 C;
    static __device__ __forceinline__ double cs(int R, int j, int k) { return c_cs[R][j][k]; }
};
template <> struct XfT<float> {
    typedef float2 C;
    static __device__ __forceinline__ float cs(int R, int j, int k) { return c_csf[R][j][k]; }
};

template <typename C> __device__ __forceinline__ C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
// a * (wr + i wi)
template <typename C, typename Real> __device__ __forceinline__ C cmulw(C a, Real wr, Real wi)
{
    C r;
    r.x = fma(-a.y, wi, a.x * wr);
    r.y = fma(a.y, wr, a.x * wi);
    return r;
}

template <typename Real, int R, bool INV> struct Dft;

template <typename Real, bool INV> struct Dft<Real, 2, INV> {
    typedef typename XfT<Real>::C C;
    static __device__ __forceinline__ void run(C (&v)[2])
    {
        const C a = cadd(v[0], v[1]), b = csub(v[0], v[1]);
        v[0] = a; v[1] = b;
    }
};
template <typename Real, bool INV> struct Dft<Real, 4, INV> {
    typedef typename XfT<Real>::C C;
    static __device__ __forceinline__ void run(C (&v)[4])
    {
        const C a = cadd(v[0], v[2]), b = csub(v[0], v[2]), c = cadd(v[1], v[3]), d = csub(v[1], v[3]);
        C md;                                   // -i d (forward), +i d (inverse)
        md.x = INV ? -d.y : d.y; md.y = INV ? d.x : -d.x;
        v[0] = cadd(a, c); v[1] = cadd(b, md); v[2] = csub(a, c); v[3] = csub(b, md);
    }
};
// odd prime R: X_p = v0 + sum_q cos(2 pi p q / R) (v_q + v_{R-q}) -/+ i sum_q sin(2 pi p q / R) (v_q - v_{R-q})
template <typename Real, int R, bool INV> struct DftPrime {
    typedef typename XfT<Real>::C C;
    static __device__ __forceinline__ void run(C (&v)[R])
    {
        constexpr int H = (R - 1) / 2;
        C s[H + 1], d[H + 1];
#pragma unroll
        for (int q = 1; q <= H; ++q) { s[q] = cadd(v[q], v[R - q]); d[q] = csub(v[q], v[R - q]); }
        const C x0 = v[0];
        C sum = x0;
#pragma unroll
        for (int q = 1; q <= H; ++q) sum = cadd(sum, s[q]);
#pragma unroll
        for (int p = 1; p <= H; ++p) {
            Real ar = x0.x, ai = x0.y, br = (Real)0, bi = (Real)0;
#pragma unroll
            for (int q = 1; q <= H; ++q) {
                const Real cj = XfT<Real>::cs(R, (p * q) % R, 0), sj = XfT<Real>::cs(R, (p * q) % R, 1);
                ar = fma(cj, s[q].x, ar); ai = fma(cj, s[q].y, ai);
                br = fma(sj, d[q].x, br); bi = fma(sj, d[q].y, bi);
            }
            C lo, hi;                           // a - i b, a + i b
            lo.x = ar + bi; lo.y = ai - br; hi.x = ar - bi; hi.y = ai + br;
            v[p] = INV ? hi : lo; v[R - p] = INV ? lo : hi;
        }
        v[0] = sum;
    }
};
template <typename Real, bool INV> struct Dft<Real, 3, INV> : DftPrime<Real, 3, INV> {};
template <typename Real, bool INV> struct Dft<Real, 5, INV> : DftPrime<Real, 5, INV> {};
template <typename Real, bool INV> struct Dft<Real, 7, INV> : DftPrime<Real, 7, INV> {};
// R = A B in registers: n = n1 + A n2, k = B k1 + k2:  X[B k1 + k2] = sum_n1 w_A^{n1 k1} w_R^{n1 k2} sum_n2 x[n1 + A n2] w_B^{n2 k2}
template <typename Real, int A, int B, bool INV> struct DftCT {
    typedef typename XfT<Real>::C C;
    static __device__ __forceinline__ void run(C (&v)[A * B])
    {
        constexpr int R = A * B;
        C t[A][B];
#pragma unroll
        for (int n1 = 0; n1 < A; ++n1) {
            C u[B];
#pragma unroll
            for (int n2 = 0; n2 < B; ++n2) u[n2] = v[n1 + A * n2];
            Dft<Real, B, INV>::run(u);
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) {
                const int j = n1 * k2;
                if (j == 0) t[n1][k2] = u[k2];
                else t[n1][k2] = cmulw(u[k2], XfT<Real>::cs(R, j, 0), INV ? XfT<Real>::cs(R, j, 1) : -XfT<Real>::cs(R, j, 1));
            }
        }
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) {
            C u[A];
#pragma unroll
            for (int n1 = 0; n1 < A; ++n1) u[n1] = t[n1][k2];
            Dft<Real, A, INV>::run(u);
#pragma unroll
            for (int k1 = 0; k1 < A; ++k1) v[B * k1 + k2] = u[k1];
        }
    }
};
template <typename Real, bool INV> struct Dft<Real, 8, INV> : DftCT<Real, 2, 4, INV> {};
template <typename Real, bool INV> struct Dft<Real, 9, INV> : DftCT<Real, 3, 3, INV> {};
template <typename Real, bool INV> struct Dft<Real, 16, INV> : DftCT<Real, 4, 4, INV> {};

constexpr int XF_MAXST = 12;
struct XfStages {
    int nst;
    int radix[XF_MAXST];
    unsigned magic[XF_MAXST];      // ceil(2^32 / m), m = sub-transform length / radix of the stage (unused when m == 1)
};

// One in-place stage on this thread's column f: sub-transforms of length L = R m.  Forward (decimation in frequency):
// R-point transform of x[b L + j + q m], q < R, times w_L^{j p}, written to the same places; inverse (decimation in
// time): the same backwards.  GLOBAL == 1: the forward stage reads its inputs from the spectrum in global memory instead
// of shared memory, the inverse stage writes its outputs there (first / last stage of the kernel: no staging pass);
// GLOBAL == 2: the stage writes its outputs to global memory whatever its direction.
template <typename Real, int R, bool INV, int NF, int GLOBAL>
__device__ __forceinline__ void xf_stage(typename XfT<Real>::C *sm, typename XfT<Real>::C *gcol, size_t gstride, bool gvalid,
                                         const typename XfT<Real>::C *__restrict__ tw, int M, int L, unsigned magic, int w, int BW, int f)
{
    typedef typename XfT<Real>::C C;
    const int m = L / R, tstep = M / L, nb = M / R;
    for (int bf = w; bf < nb; bf += BW) {
        const int b = m == 1 ? bf : (int)__umulhi((unsigned)bf, magic), j = bf - b * m;
        const int e0 = b * L + j;
        C v[R];
        if (!INV && GLOBAL == 1) {
#pragma unroll
            for (int q = 0; q < R; ++q) {
                if (gvalid) v[q] = __ldcs(gcol + (size_t)(e0 + q * m) * gstride);
                else { v[q].x = (Real)0; v[q].y = (Real)0; }
            }
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = sm[(e0 + q * m) * NF + f];
        }
        if (!INV) Dft<Real, R, false>::run(v);
        if (j != 0) {
#pragma unroll
            for (int p = 1; p < R; ++p) {
                const C t = __ldg(tw + tstep * j * p);            // w_L^{j p}, forward sign
                v[p] = cmulw(v[p], t.x, INV ? -t.y : t.y);
            }
        }
        if (INV) Dft<Real, R, true>::run(v);
        if ((INV && GLOBAL == 1) || GLOBAL == 2) {
            if (gvalid) {
#pragma unroll
                for (int q = 0; q < R; ++q) __stcs(gcol + (size_t)(e0 + q * m) * gstride, v[q]);
            }
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) sm[(e0 + q * m) * NF + f] = v[q];
        }
    }
}

template <typename Real, bool INV, int NF, int GLOBAL, bool R16>
__device__ __forceinline__ void xf_stage_any(int R, typename XfT<Real>::C *sm, typename XfT<Real>::C *gcol, size_t gstride, bool gvalid,
                                             const typename XfT<Real>::C *__restrict__ tw, int M, int L, unsigned magic, int w, int BW, int f)
{
#define XF_CASE(RR) case RR: xf_stage<Real, RR, INV, NF, GLOBAL>(sm, gcol, gstride, gvalid, tw, M, L, magic, w, BW, f); break;
    switch (R) {
    case 16: if constexpr (R16) xf_stage<Real, 16, INV, NF, GLOBAL>(sm, gcol, gstride, gvalid, tw, M, L, magic, w, BW, f); break;
        XF_CASE(9) XF_CASE(8) XF_CASE(7) XF_CASE(5) XF_CASE(4) XF_CASE(3)
    default: xf_stage<Real, 2, INV, NF, GLOBAL>(sm, gcol, gstride, gvalid, tw, M, L, magic, w, BW, f); break;
    }
#undef XF_CASE
}

// The innermost stage (L = R: contiguous groups of R positions), K4 and the same stage of the inverse in registers, for
// the three components of one kz at a time (K4 mixes the components): saves two passes over shared memory and the K4 pass.
template <typename Real, int R, int TZ>
__device__ __forceinline__ void xf_centre(typename XfT<Real>::C *sm, int M, Real ky, Real kz, Real eyz, bool valid,
                                          const typename XfT<Real>::C *__restrict__ xkk, Real pref, Real inv4xi2, int w, int BW, int tz)
{
    typedef typename XfT<Real>::C C;
    constexpr int NF = 3 * TZ;
    if (!valid) return;                                          // a kz beyond the half-spectrum (ragged last tile): zeros stay zeros
    for (int bf = w; bf < M / R; bf += BW) {
        C kk[R];                                                 // (k_x, e_x) of the R positions: loads in flight during the transforms
#pragma unroll
        for (int q = 0; q < R; ++q) kk[q] = __ldg(xkk + bf * R + q);
        C v[3][R];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
#pragma unroll
            for (int q = 0; q < R; ++q) v[c][q] = sm[(bf * R + q) * NF + c * TZ + tz];
            Dft<Real, R, false>::run(v[c]);
        }
#pragma unroll
        for (int q = 0; q < R; ++q) scale_mode_x<Real>(kk[q].x, ky, kz, kk[q].y * eyz, pref, inv4xi2, v[0][q], v[1][q], v[2][q]);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Dft<Real, R, true>::run(v[c]);
#pragma unroll
            for (int q = 0; q < R; ++q) sm[(bf * R + q) * NF + c * TZ + tz] = v[c][q];
        }
    }
}

// blockDim.x = NF * BW: thread (w, f) works on column f = component * TZ + tz, butterflies w, w + BW, ...
template <int BYTES> __device__ __forceinline__ void cp_async(void *dst, const void *src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src) : "memory");
}

#ifndef XF_MINB
#define XF_MINB 2
#endif
template <typename Real, int TZ, bool R16>
__global__ void __launch_bounds__(256, R16 ? 1 : XF_MINB)
k_xfft_scale(int M, int Mh, XfStages xs, Real pref, Real inv4xi2, const Real *__restrict__ ktab,
             const typename XfT<Real>::C *__restrict__ xkk, const typename XfT<Real>::C *__restrict__ ykk,
             const typename XfT<Real>::C *__restrict__ tw, typename XfT<Real>::C *__restrict__ spec)
{
    // ykk != nullptr: the second axis of the spectrum is in the digit-reversed order k_yfft leaves, (k_y, e_y) per position
    typedef typename XfT<Real>::C C;
    constexpr int NF = 3 * TZ;
    extern __shared__ __align__(16) unsigned char xf_raw[];
    C *sm = reinterpret_cast<C *>(xf_raw);                 // [M][NF]
    const int tid = threadIdx.x, NT = blockDim.x;
    const int iy = blockIdx.y, iz0 = blockIdx.x * TZ;
    const size_t plane = (size_t)M * Mh;
    const int f = tid % NF, w = tid / NF, BW = NT / NF;
    const int fc = f / TZ, ftz = f - fc * TZ;
    const bool gvalid = iz0 + ftz < Mh;
    C *gcol = spec + (size_t)fc * M * plane + (size_t)iy * Mh + iz0 + ftz;      // element x of this thread's column at + x * plane
    const int nst = xs.nst;
    const bool gfirst = nst >= 2;                          // the outermost inverse stage writes global memory directly

    // all columns of the block by asynchronous 16-byte (fp32: 8-byte) copies: every load of the block is in flight at once,
    // and the other blocks of the SM compute meanwhile
    for (int ix = w; ix < M; ix += BW) {
        if (gvalid) cp_async<sizeof(C)>(&sm[ix * NF + f], gcol + (size_t)ix * plane);
        else { sm[ix * NF + f].x = (Real)0; sm[ix * NF + f].y = (Real)0; }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
    int L = M;
    for (int st = 0; st < nst - 1; ++st) {
        xf_stage_any<Real, false, NF, false, R16>(xs.radix[st], sm, gcol, plane, gvalid, tw, M, L, xs.magic[st], w, BW, f);
        L /= xs.radix[st];
        __syncthreads();
    }
    {
        // innermost stage (L == its radix), K4, and back
        const int R = xs.radix[nst - 1];
        const int tz = tid % TZ, w3 = tid / TZ, BW3 = NT / TZ;
        const bool valid = iz0 + tz < Mh;
        const int iz = min(iz0 + tz, Mh - 1);
        // k_y, k_z and e_y e_z of this thread's modes; zero on the Nyquist planes (reading S8), like e_x in the table
        Real ky, ey;
        if (ykk) { const C t = __ldg(ykk + iy); ky = t.x; ey = t.y; }
        else { ky = __ldg(ktab + iy); ey = 2 * iy == M ? (Real)0 : __ldg(ktab + M + iy); }
        const Real kz = __ldg(ktab + iz);
        const Real eyz = 2 * iz == M ? (Real)0 : ey * __ldg(ktab + M + iz);
        if (R <= 5) {
            switch (R) {
            case 5: xf_centre<Real, 5, TZ>(sm, M, ky, kz, eyz, valid, xkk, pref, inv4xi2, w3, BW3, tz); break;
            case 4: xf_centre<Real, 4, TZ>(sm, M, ky, kz, eyz, valid, xkk, pref, inv4xi2, w3, BW3, tz); break;
            case 3: xf_centre<Real, 3, TZ>(sm, M, ky, kz, eyz, valid, xkk, pref, inv4xi2, w3, BW3, tz); break;
            default: xf_centre<Real, 2, TZ>(sm, M, ky, kz, eyz, valid, xkk, pref, inv4xi2, w3, BW3, tz); break;
            }
        } else {
            xf_stage_any<Real, false, NF, false, R16>(R, sm, gcol, plane, gvalid, tw, M, L, xs.magic[nst - 1], w, BW, f);
            __syncthreads();
            if (valid) {
                for (int pos = w3; pos < M; pos += BW3) {
                    const C kk = __ldg(xkk + pos);
                    C *q = sm + pos * NF + tz;
                    scale_mode_x<Real>(kk.x, ky, kz, kk.y * eyz, pref, inv4xi2, q[0], q[TZ], q[2 * TZ]);
                }
            }
            __syncthreads();
            xf_stage_any<Real, true, NF, false, R16>(R, sm, gcol, plane, gvalid, tw, M, L, xs.magic[nst - 1], w, BW, f);
        }
        __syncthreads();
    }
    for (int st = nst - 2; st >= 0; --st) {
        L *= xs.radix[st];
        if (st == 0 && gfirst) xf_stage_any<Real, true, NF, true, R16>(xs.radix[st], sm, gcol, plane, gvalid, tw, M, L, xs.magic[st], w, BW, f);
        else xf_stage_any<Real, true, NF, false, R16>(xs.radix[st], sm, gcol, plane, gvalid, tw, M, L, xs.magic[st], w, BW, f);
        if (st > 0) __syncthreads();
    }
    if (!gfirst) {
        __syncthreads();
        for (int ix = w; ix < M; ix += BW)
            if (gvalid) gcol[(size_t)ix * plane] = sm[ix * NF + f];
    }
}

// ================================================================================================================
// Own 2-D transforms of the x-planes (the fused path's SE_STAGE_FFT / SE_STAGE_IFFT): a real-to-complex pass over z
// with M/2-point complex transforms (k_zr2c / k_zc2r) and a complex pass over y (k_yfft), built from the same
// register butterflies as K4x.  cuFFT's 2-D plan runs its pass over z at 2.3 TB/s (blocks of 60 threads); these
// passes stream whole contiguous chunks of rows / 8 (fp32: 16) adjacent columns through shared memory.
// The pass over y leaves the ky index in the digit-reversed order of its decimation-in-frequency stages (position p of
// the second axis holds mode ky = rev(p)); K4x takes k_y and e_y from a table per position, and the inverse pass
// (decimation in time) takes that order and returns the natural one.  Nothing else reads the spectrum on this path.

// one in-place stage of a length-N transform on a column whose element `pos` is at col[pos] (shared memory);
// twiddle w_N^t = tw[tws * t] (the plan's table of w_M^t, M = tws N)
template <typename Real, int R, bool INV>
__device__ __forceinline__ void zf_stage(typename XfT<Real>::C *col, const typename XfT<Real>::C *__restrict__ tw, int tws, int N,
                                         int L, unsigned magic, int w, int BW)
{
    typedef typename XfT<Real>::C C;
    const int m = L / R, tstep = (N / L) * tws, nb = N / R;
    for (int bf = w; bf < nb; bf += BW) {
        const int b = m == 1 ? bf : (int)__umulhi((unsigned)bf, magic), j = bf - b * m;
        C *base = col + b * L + j;
        C v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = base[q * m];
        if (!INV) Dft<Real, R, false>::run(v);
        if (j != 0) {
#pragma unroll
            for (int p = 1; p < R; ++p) {
                const C t = __ldg(tw + tstep * j * p);
                v[p] = cmulw(v[p], t.x, INV ? -t.y : t.y);
            }
        }
        if (INV) Dft<Real, R, true>::run(v);
#pragma unroll
        for (int q = 0; q < R; ++q) base[q * m] = v[q];
    }
}

template <typename Real, bool INV, bool R16>
__device__ __forceinline__ void zf_stage_any(int R, typename XfT<Real>::C *col, const typename XfT<Real>::C *__restrict__ tw, int tws,
                                             int N, int L, unsigned magic, int w, int BW)
{
#define ZF_CASE(RR) case RR: zf_stage<Real, RR, INV>(col, tw, tws, N, L, magic, w, BW); break;
    switch (R) {
    case 16: if constexpr (R16) zf_stage<Real, 16, INV>(col, tw, tws, N, L, magic, w, BW); break;
        ZF_CASE(9) ZF_CASE(8) ZF_CASE(7) ZF_CASE(5) ZF_CASE(4) ZF_CASE(3)
    default: zf_stage<Real, 2, INV>(col, tw, tws, N, L, magic, w, BW); break;
    }
#undef ZF_CASE
}

// Real-to-complex over z.  A block takes RB consecutive rows (M reals each = N2 = M/2 complex numbers z_j = x_2j + i x_2j+1,
// one contiguous chunk of the grid), row r at sm[r * RS ...] with RS = 1 mod 8 (16) complex numbers so that the RB lanes of
// a butterfly step hit different banks; thread (w, f): row f, butterflies w, w + BW, ...  After the N2-point transform Z
// (digit-reversed: Z_k at position zpos[k]):  X_k = E_k + w_M^k O_k, E_k = (Z_k + conj Z_{N2-k}) / 2, O_k = -i (Z_k - conj Z_{N2-k}) / 2,
// k = 0 .. N2, written straight to the spectrum rows (M/2 + 1 complex numbers, again one contiguous chunk).
template <typename Real, bool R16>
__global__ void __launch_bounds__(256)
k_zr2c(int M, int RS, int RB, long long nrows, XfStages xs, const typename XfT<Real>::C *__restrict__ tw, const int *__restrict__ zpos,
       const Real *__restrict__ grid, typename XfT<Real>::C *__restrict__ spec)
{
    typedef typename XfT<Real>::C C;
    extern __shared__ __align__(16) unsigned char xf_raw[];
    C *sm = reinterpret_cast<C *>(xf_raw);
    const int tid = threadIdx.x, NT = blockDim.x, N2 = M / 2, Mh = N2 + 1;
    const long long row0 = (long long)blockIdx.x * RB;
    const int nr = (int)min((long long)RB, nrows - row0);
    const C *src = reinterpret_cast<const C *>(grid) + row0 * N2;
    const unsigned mg = 0xffffffffu / (unsigned)N2 + 1u;                               // e / N2 for e < 2^16
    for (int e = tid; e < nr * N2; e += NT) {
        const int r = (int)__umulhi((unsigned)e, mg);
        cp_async<sizeof(C)>(&sm[r * RS + (e - r * N2)], src + e);
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
    const int f = tid % RB, w = tid / RB, BW = NT / RB;
    C *col = sm + f * RS;
    int L = N2;
    for (int st = 0; st < xs.nst; ++st) {
        if (f < nr) zf_stage_any<Real, false, R16>(xs.radix[st], col, tw, 2, N2, L, xs.magic[st], w, BW);
        L /= xs.radix[st];
        __syncthreads();
    }
    // lanes run over the rows first (the same position of RB rows: conflict-free; consecutive k of one row sit 20 or more
    // positions apart, i.e. in two bank groups), each row gets 32 / RB consecutive k of a warp
    C *dst = spec + row0 * Mh + (long long)f * Mh;
    for (int k = w; k < Mh && f < nr; k += BW) {
        const int ka = k == N2 ? 0 : k, kb = k == 0 ? 0 : N2 - k;
        const C a = col[__ldg(zpos + ka)], bq = col[__ldg(zpos + kb)];
        // E = (a + conj b) / 2, O = -i (a - conj b) / 2
        const Real er = (Real)0.5 * (a.x + bq.x), ei = (Real)0.5 * (a.y - bq.y);
        const Real dr = (Real)0.5 * (a.x - bq.x), di = (Real)0.5 * (a.y + bq.y);      // (a - conj b) / 2
        const Real orr = di, oi = -dr;                                                // times -i
        const C t = __ldg(tw + k);                                                    // w_M^k
        C o;
        o.x = er + (orr * t.x - oi * t.y);
        o.y = ei + (orr * t.y + oi * t.x);
        dst[k] = o;
    }
}

// Complex-to-real over z, unnormalised like cuFFT's: Z_k = E_k + i O_k with E_k = X_k + conj X_{N2-k}, O_k = (X_k - conj X_{N2-k}) w_M^{-k},
// k = 0 .. N2 - 1 (the imaginary parts of X_0 and X_{N2} are ignored, as by cuFFT), placed at position zpos[k]; the inverse
// (decimation-in-time) stages return z_j = x_2j + i x_2j+1 in natural order, i.e. the grid rows.
template <typename Real, bool R16>
__global__ void __launch_bounds__(256)
k_zc2r(int M, int RS, int RB, long long nrows, XfStages xs, const typename XfT<Real>::C *__restrict__ tw, const int *__restrict__ zpos,
       const typename XfT<Real>::C *__restrict__ spec, Real *__restrict__ grid)
{
    typedef typename XfT<Real>::C C;
    extern __shared__ __align__(16) unsigned char xf_raw[];
    C *sm = reinterpret_cast<C *>(xf_raw);
    const int tid = threadIdx.x, NT = blockDim.x, N2 = M / 2, Mh = N2 + 1;
    const long long row0 = (long long)blockIdx.x * RB;
    const int nr = (int)min((long long)RB, nrows - row0);
    const int f = tid % RB, w = tid / RB, BW = NT / RB;
    C *col = sm + f * RS;
    // lanes along k: coalesced loads of the spectrum rows (every entry is read twice, the second time from L1); the stores
    // into the digit-reversed positions conflict two- to four-way, which measured cheaper than staging the rows in shared
    // memory (half the blocks per SM) or loading with the lanes over the rows (64-byte pieces)
    const C *src = spec + row0 * Mh;
    const unsigned mg = 0xffffffffu / (unsigned)N2 + 1u;                               // e / N2 for e < 2^16
    for (int e = tid; e < nr * N2; e += NT) {
        const int r = (int)__umulhi((unsigned)e, mg), k = e - r * N2;
        C a = __ldg(src + (long long)r * Mh + k), bq = __ldg(src + (long long)r * Mh + N2 - k);
        if (k == 0) { a.y = (Real)0; bq.y = (Real)0; }
        const Real er = a.x + bq.x, ei = a.y - bq.y;                                   // a + conj b
        const Real dr = a.x - bq.x, di = a.y + bq.y;                                   // a - conj b
        const C t = __ldg(tw + k);                                                     // w_M^k; O = d conj(t)
        const Real orr = dr * t.x + di * t.y, oi = di * t.x - dr * t.y;
        C z;
        z.x = er - oi; z.y = ei + orr;                                                 // E + i O
        sm[r * RS + __ldg(zpos + k)] = z;
    }
    __syncthreads();
    int L = 1;
    for (int st = xs.nst - 1; st >= 0; --st) {
        L *= xs.radix[st];
        if (f < nr) zf_stage_any<Real, true, R16>(xs.radix[st], col, tw, 2, N2, L, xs.magic[st], w, BW);
        __syncthreads();
    }
    C *dst = reinterpret_cast<C *>(grid) + row0 * N2;
    for (int e = tid; e < nr * N2; e += NT) {
        const int r = (int)__umulhi((unsigned)e, mg);
        dst[e] = sm[r * RS + (e - r * N2)];
    }
}

// Complex transform over y of NF adjacent columns (consecutive kz, running on into the next x-plane), in place.
// Forward: decimation in frequency, the result stays in digit-reversed order along y; inverse: decimation in time from
// that order, the last stage writes global memory directly.
#ifndef YF_MINB
#define YF_MINB 3
#endif
#ifndef SE_YF_NF32
#define SE_YF_NF32 16      /* columns per block of k_yfft in fp32 plans */
#endif
#ifndef SE_YF_NF64
#define SE_YF_NF64 8      /* columns per block of k_yfft in fp64 plans */
#endif
template <typename Real, int NF, bool INV, bool R16>
__global__ void __launch_bounds__(192, YF_MINB)
k_yfft(int M, int Mh, long long ncols, XfStages xs, const typename XfT<Real>::C *__restrict__ tw, typename XfT<Real>::C *__restrict__ spec)
{
    typedef typename XfT<Real>::C C;
    extern __shared__ __align__(16) unsigned char xf_raw[];
    C *sm = reinterpret_cast<C *>(xf_raw);                 // [M][NF]
    const int tid = threadIdx.x, NT = blockDim.x;
    const int f = tid % NF, w = tid / NF, BW = NT / NF;
    const long long q = (long long)blockIdx.x * NF + f;
    const bool gvalid = q < ncols;
    const long long pl = q / Mh;
    C *gcol = spec + pl * (long long)M * Mh + (q - pl * Mh);
    const size_t gstride = (size_t)Mh;
    for (int iy = w; iy < M; iy += BW) {
        if (gvalid) cp_async<sizeof(C)>(&sm[iy * NF + f], gcol + (size_t)iy * gstride);
        else { sm[iy * NF + f].x = (Real)0; sm[iy * NF + f].y = (Real)0; }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
    const int nst = xs.nst;
    if (!INV) {
        int L = M;
        for (int st = 0; st < nst; ++st) {
            if (st == nst - 1) xf_stage_any<Real, false, NF, 2, R16>(xs.radix[st], sm, gcol, gstride, gvalid, tw, M, L, xs.magic[st], w, BW, f);
            else xf_stage_any<Real, false, NF, 0, R16>(xs.radix[st], sm, gcol, gstride, gvalid, tw, M, L, xs.magic[st], w, BW, f);
            L /= xs.radix[st];
            if (st < nst - 1) __syncthreads();
        }
    } else {
        int L = 1;
        for (int st = nst - 1; st >= 0; --st) {
            L *= xs.radix[st];
            if (st == 0) xf_stage_any<Real, true, NF, true, R16>(xs.radix[st], sm, gcol, gstride, gvalid, tw, M, L, xs.magic[st], w, BW, f);
            else xf_stage_any<Real, true, NF, false, R16>(xs.radix[st], sm, gcol, gstride, gvalid, tw, M, L, xs.magic[st], w, BW, f);
            if (st > 0) __syncthreads();
        }
    }
}

// radices of the x-transform; false if M has a prime factor > 7.  Large radices first (fewest passes over shared memory; the
// first stage's loads come straight from global memory), the smallest last: a last radix <= 5 is merged with K4.
bool xf_factor(int M, bool allow16, XfStages &xs, bool split_last = true)
{
    static const int pref[] = {16, 9, 8, 7, 5, 4, 3, 2};
    xs.nst = 0;
    int rem = M;
    for (int r : pref) {
        if (r == 16 && !allow16) continue;
        while (rem % r == 0 && rem > 1) {
            if (xs.nst == XF_MAXST) return false;
            xs.radix[xs.nst++] = r;
            rem /= r;
        }
    }
    if (rem != 1 || M < 2) return false;
    // a lone trailing 8 or 9 (e.g. 576 = 9 8 8, 64 = 8 8): split off a small last radix when that costs no extra pass over
    // what the unmerged K4 would, i.e. 8 -> 4 2
    if (split_last && xs.nst >= 1 && xs.radix[xs.nst - 1] == 8 && xs.nst < XF_MAXST) { xs.radix[xs.nst - 1] = 4; xs.radix[xs.nst++] = 2; }
    int L = M;
    for (int st = 0; st < xs.nst; ++st) {
        const int m = L / xs.radix[st];
        xs.magic[st] = m > 1 ? (unsigned)((0x100000000ull + (unsigned)m - 1) / (unsigned)m) : 0u;
        L = m;
    }
    return true;
}

template <typename Real, int TZ> size_t xf_smem(int M) { return (size_t)M * (3 * TZ) * sizeof(typename XfT<Real>::C); }

// threads: NF columns x BW butterfly lanes, BW chosen so that the stages' butterfly counts M / R split evenly
template <int NF> int xf_threads(int M, const XfStages &xs)
{
    int best = 1;
    double bc = 1e30;
    for (int bw = 256 / NF; bw >= 4; --bw) {
        double cost = 0;
        for (int st = 0; st < xs.nst; ++st) {
            const int nb = M / xs.radix[st];
            cost += (double)((nb + bw - 1) / bw) * xs.radix[st];           // iterations x work per butterfly
        }
        cost *= 1.0 + 2.0 / bw;                                             // fewer threads: less latency hiding
        if (cost < bc) { bc = cost; best = bw; }
    }
    return best * NF;
}

template <typename Real, int TZ, bool R16>
cudaError_t xf_launch(se_plan *p, cudaStream_t s, bool prepare)
{
    typedef typename XfT<Real>::C C;
    const SeGeom &g = p->g;
    const int M = g.M, Mh = M / 2 + 1;
    auto kern = k_xfft_scale<Real, TZ, R16>;
    const size_t smem = xf_smem<Real, TZ>(M);
    if (prepare) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    XfStages xs;
    xs.nst = p->xf_nst;
    for (int i = 0; i < XF_MAXST; ++i) { xs.radix[i] = i < p->xf_nst ? p->xf_radix[i] : 1; xs.magic[i] = i < p->xf_nst ? p->xf_magic[i] : 0u; }
    const double M3 = (double)M * M * M;
    dim3 grid((Mh + TZ - 1) / TZ, M);
    kern<<<grid, p->xf_threads, smem, s>>>(M, Mh, xs, (Real)(8.0 * SE_PI / M3), (Real)(1.0 / (4.0 * g.xi * g.xi)), (const Real *)p->ktab,
                                           (const C *)p->xf_xk, (const C *)(p->f2_ok ? p->f2_ykk : nullptr), (const C *)p->xf_tw,
                                           (C *)p->spec);
    p->launches += 1;
    return cudaGetLastError();
}

cudaError_t xf_dispatch(se_plan *p, cudaStream_t s, bool prepare)
{
    if (p->precision == SE_FP64) {
        if (p->xf_r16) return p->xf_tz == 4 ? xf_launch<double, 4, true>(p, s, prepare) : xf_launch<double, 2, true>(p, s, prepare);
        return p->xf_tz == 4 ? xf_launch<double, 4, false>(p, s, prepare) : xf_launch<double, 2, false>(p, s, prepare);
    }
    return p->xf_tz == 8 ? xf_launch<float, 8, true>(p, s, prepare) : xf_launch<float, 4, true>(p, s, prepare);
}

template <typename Real>
cudaError_t scale_impl(se_plan *p, void *spec, int y0, int ny, cudaStream_t s)
{
    const SeGeom &g = p->g;
    int Mh = g.M / 2 + 1;
    double M3 = (double)g.M * g.M * g.M;
    // (h^3 / V) * 8 pi  with h^3/V = 1/M^3
    Real pref = (Real)(8.0 * SE_PI / M3);
    Real inv4xi2 = (Real)(1.0 / (4.0 * g.xi * g.xi));
    dim3 grid((Mh + 255) / 256, ny, g.M);
    int T = Mh < 256 ? ((Mh + 31) / 32) * 32 : 256;
    grid.x = (Mh + T - 1) / T;
    k_scale<Real><<<grid, T, 0, s>>>(g.M, Mh, y0, ny, pref, inv4xi2, (const Real *)p->ktab,
                                     (typename Cplx<Real>::type *)spec);
    p->launches += 1;
    return cudaGetLastError();
}

}  // namespace

cudaError_t se_launch_scale(se_plan *p, cudaStream_t s)
{
    return p->precision == SE_FP64 ? scale_impl<double>(p, p->spec, 0, p->g.M, s) : scale_impl<float>(p, p->spec, 0, p->g.M, s);
}

// se.h: K4 on a caller-owned block of the spectrum (the ky-pencil a rank holds in a slab-decomposed transform)
extern "C" se_status se_scale_block(se_plan *p, void *spec, int ky0, int nky, void *stream)
{
    if (!p || !spec || ky0 < 0 || nky < 1 || ky0 + nky > p->g.M) return SE_EINVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) { cudaGetLastError(); return SE_EINVAL; }
    cudaError_t e = p->precision == SE_FP64 ? scale_impl<double>(p, spec, ky0, nky, (cudaStream_t)stream)
                                            : scale_impl<float>(p, spec, ky0, nky, (cudaStream_t)stream);
    return e == cudaSuccess ? SE_OK : SE_ECUDA;
}

// ================================================================================================================
// se_scale_noalloc (se.h): K4 for callers that may not allocate (CUDA graph capture, serving loops, harnesses that
// forbid cudaMalloc).  Same kernel as se_scale_block (k_scale); what a plan keeps in its cudaMalloc'ed multiplier
// table (k and e(k) per 1-D index, 2 M reals) lives here in a file-scope device array of fixed size, refilled by a
// small kernel on every call (the array keeps the previous call's table: nothing in it is reused, nothing needs to
// start at zero).  Every GPU that loads the library holds the 64 KB until the process exits.  All calls share the
// array: two calls that overlap on the GPU (different streams) race on it.
constexpr int SE_NOALLOC_MAX_M = 4096;                          // = se_plan_create's own limit on M
static __device__ __align__(256) double se_noalloc_ktab[2 * SE_NOALLOC_MAX_M];

namespace {

// table of a Gaussian-window plan (se_build_ktab builds the same in long double on the host): k_i = 2 pi n_i / L,
// e_i = exp(-(1 - eta) k_i^2 / 4 xi^2), computed in double, stored in the precision of the spectrum
template <typename Real>
__global__ void k_fill_ktab(int M, double L, double xi, double eta, Real *__restrict__ tab)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    const int n = (2 * i >= M) ? i - M : i;
    const double k = 2.0 * SE_PI * (double)n / L;
    tab[i] = (Real)k;
    tab[M + i] = (Real)exp(-(1.0 - eta) * k * k / (4.0 * xi * xi));
}

// device address of the array, looked up once per device with that device current (the array's name is only a
// host-side handle in host code, not an address a kernel can use)
constexpr int SE_NOALLOC_MAX_DEV = 64;
void *g_noalloc_ptr[SE_NOALLOC_MAX_DEV];
std::mutex g_noalloc_mutex;

cudaError_t noalloc_scratch(int dev, void **out)
{
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, se_noalloc_ktab);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_noalloc_ptr[dev] = ptr;
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

template <typename Real>
cudaError_t scale_noalloc_impl(void *spec, void *tab, int M, int P, double L, double xi, int ky0, int nky, cudaStream_t s)
{
    const int Mh = M / 2 + 1;
    const double h = L / M, m = 0.95 * std::sqrt(SE_PI * P);    // reading S4, as se_plan_create_ex
    const double eta = (P * h * xi / m) * (P * h * xi / m);
    k_fill_ktab<Real><<<(M + 255) / 256, 256, 0, s>>>(M, L, xi, eta, (Real *)tab);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const double M3 = (double)M * M * M;
    const int T = Mh < 256 ? ((Mh + 31) / 32) * 32 : 256;
    dim3 grid((Mh + T - 1) / T, nky, M);
    k_scale<Real><<<grid, T, 0, s>>>(M, Mh, ky0, nky, (Real)(8.0 * SE_PI / M3), (Real)(1.0 / (4.0 * xi * xi)), (const Real *)tab,
                                     (typename Cplx<Real>::type *)spec);
    return cudaGetLastError();
}

}  // namespace

extern "C" se_status se_scale_noalloc(void *spec, int M, int P, double L, double xi, se_precision precision, int ky0, int nky,
                                      void *stream)
{
    if (!spec || M < 2 || (M & 1) || P < 2 || (P & 1) || P > M || !(L > 0.0) || !(xi > 0.0) || ky0 < 0 || nky < 1 ||
        (precision != SE_FP64 && precision != SE_FP32))
        return SE_EINVAL;
    if (M > SE_NOALLOC_MAX_M) return SE_ELIMIT;                  // the table would not fit the fixed array
    if (ky0 + nky > M) return SE_EINVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return SE_ECUDA; }
    if (dev < 0 || dev >= SE_NOALLOC_MAX_DEV) return SE_ELIMIT;
    void *tab = nullptr;
    if (noalloc_scratch(dev, &tab) != cudaSuccess) { cudaGetLastError(); return SE_ECUDA; }
    cudaError_t e = precision == SE_FP64 ? scale_noalloc_impl<double>(spec, tab, M, P, L, xi, ky0, nky, (cudaStream_t)stream)
                                         : scale_noalloc_impl<float>(spec, tab, M, P, L, xi, ky0, nky, (cudaStream_t)stream);
    return e == cudaSuccess ? SE_OK : SE_ECUDA;
}

// Decides whether the plan's se_eval takes the fused x-transform (M 7-smooth, the columns of a block fit in shared
// memory, not switched off by SE_FFT_MODE=3d) and builds its tables: twiddles w_M^t in long double, the x-index of
// every position after the forward stages (mixed-radix digit reversal), the small-transform constants.
cudaError_t se_build_xfft(se_plan *p)
{
    p->xf_ok = 0;
    if (p->slab) return cudaSuccess;
    const char *mode = std::getenv("SE_FFT_MODE");
    if (mode && std::strcmp(mode, "3d") == 0) return cudaSuccess;
    const int M = p->g.M;
    XfStages xs;
    if (!xf_factor(M, false, xs)) return cudaSuccess;
    // passes over shared memory (32 bytes per mode each): the outermost stage half a pass each way, the inner ones a
    // whole pass each way, the innermost one pass merged with K4 or three (stage, K4, stage) unmerged
    auto passes = [](const XfStages &x) { return 1 + 2 * (x.nst >= 2 ? x.nst - 2 : 0) + (x.radix[x.nst - 1] <= 5 ? 1 : 3); };
    p->xf_r16 = p->precision == SE_FP32;
    {
        XfStages x16;
        if (xf_factor(M, true, x16) && (p->precision == SE_FP32 ? passes(x16) <= passes(xs) : passes(x16) < passes(xs))) { xs = x16; p->xf_r16 = 1; }
    }
    const size_t lim = 227 * 1024;
    if (p->precision == SE_FP64) {
        if (xf_smem<double, 4>(M) <= lim) p->xf_tz = 4;
        else if (xf_smem<double, 2>(M) <= lim) p->xf_tz = 2;
        else return cudaSuccess;
        p->xf_threads = p->xf_tz == 4 ? xf_threads<12>(M, xs) : xf_threads<6>(M, xs);
    } else {
        if (xf_smem<float, 8>(M) <= lim) p->xf_tz = 8;
        else if (xf_smem<float, 4>(M) <= lim) p->xf_tz = 4;
        else return cudaSuccess;
        p->xf_threads = p->xf_tz == 8 ? xf_threads<24>(M, xs) : xf_threads<12>(M, xs);
    }
    if (const char *e = std::getenv("SE_XF_BW")) {                  // experiments: butterfly lanes per column
        const int nf = 3 * p->xf_tz, bw = std::atoi(e);
        if (bw >= 1 && bw * nf <= 256) p->xf_threads = bw * nf;
    }
    p->xf_nst = xs.nst;
    for (int i = 0; i < xs.nst; ++i) { p->xf_radix[i] = xs.radix[i]; p->xf_magic[i] = xs.magic[i]; }
    const long double PI = 3.14159265358979323846264338327950288L;
    static double hcs[17][16][2];
    static float hcsf[17][16][2];
    for (int R = 1; R <= 16; ++R)
        for (int j = 0; j < 16; ++j) {
            const long double a = 2.0L * PI * (long double)(j % R) / (long double)R;
            hcs[R][j][0] = (double)cosl(a); hcs[R][j][1] = (double)sinl(a);
            hcsf[R][j][0] = (float)cosl(a); hcsf[R][j][1] = (float)sinl(a);
        }
    cudaError_t e = cudaMemcpyToSymbol(c_cs, hcs, sizeof(hcs));
    if (e == cudaSuccess) e = cudaMemcpyToSymbol(c_csf, hcsf, sizeof(hcsf));
    if (e != cudaSuccess) return e;
    const size_t cb = p->precision == SE_FP64 ? sizeof(double2) : sizeof(float2);
    if ((e = cudaMalloc(&p->xf_tw, (size_t)M * cb)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&p->xf_xk, (size_t)M * cb)) != cudaSuccess) return e;
    p->workspace_bytes += (size_t)M * 2 * cb;
    if (p->precision == SE_FP64) {
        std::vector<double2> tw(M);
        for (int t = 0; t < M; ++t) { const long double a = 2.0L * PI * t / M; tw[t] = make_double2((double)cosl(a), (double)-sinl(a)); }
        e = cudaMemcpy(p->xf_tw, tw.data(), (size_t)M * cb, cudaMemcpyHostToDevice);
    } else {
        std::vector<float2> tw(M);
        for (int t = 0; t < M; ++t) { const long double a = 2.0L * PI * t / M; tw[t] = make_float2((float)cosl(a), (float)-sinl(a)); }
        e = cudaMemcpy(p->xf_tw, tw.data(), (size_t)M * cb, cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess) e = xf_dispatch(p, nullptr, true);
    if (e == cudaSuccess) p->xf_ok = 1;
    return e;
}

cudaError_t se_launch_xfft_scale(se_plan *p, cudaStream_t s) { return xf_dispatch(p, s, false); }

namespace {

// frequency held at position `pos` after the decimation-in-frequency stages of a length-N transform (mixed-radix digit reversal)
int xf_rev(int pos, int N, int nst, const int *radix)
{
    int rem = pos, L = N, k = 0, mult = 1;
    for (int st = 0; st < nst; ++st) {
        const int r = radix[st], m = L / r;
        k += (rem / m) * mult;
        rem %= m; mult *= r; L = m;
    }
    return k;
}

XfStages f2_stages(const se_plan *p, bool z)
{
    XfStages xs;
    xs.nst = z ? p->f2z_nst : p->f2y_nst;
    for (int i = 0; i < XF_MAXST; ++i) {
        xs.radix[i] = i < xs.nst ? (z ? p->f2z_radix[i] : p->f2y_radix[i]) : 1;
        xs.magic[i] = i < xs.nst ? (z ? p->f2z_magic[i] : p->f2y_magic[i]) : 0u;
    }
    return xs;
}

// the own 2-D transforms of the x-planes (k_zr2c / k_zc2r over z, k_yfft over y); prepare: dynamic shared memory opt-in only
template <typename Real, int NF, bool R16>
cudaError_t fft2_impl(se_plan *p, bool forward, cudaStream_t s, bool prepare, int parts)
{
    typedef typename XfT<Real>::C C;
    const int M = p->g.M, Mh = M / 2 + 1;
    const size_t smz = (size_t)p->f2_rb * p->f2_rs * sizeof(C), smzi = (size_t)p->f2_rbi * p->f2_rs * sizeof(C), smy = (size_t)M * NF * sizeof(C);
    if (prepare) {
        const int smax = (int)((size_t)p->f2_rbmax * p->f2_rs * sizeof(C));
        cudaError_t e = cudaFuncSetAttribute(k_zr2c<Real, R16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smax);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_zc2r<Real, R16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smax);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_yfft<Real, NF, false, R16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smy);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_yfft<Real, NF, true, R16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smy);
        return e;
    }
    const long long nrows = 3LL * M * M, ncols = 3LL * M * Mh;
    const unsigned gz = (unsigned)((nrows + p->f2_rb - 1) / p->f2_rb), gzi = (unsigned)((nrows + p->f2_rbi - 1) / p->f2_rbi), gy = (unsigned)((ncols + NF - 1) / NF);
    const XfStages xz = f2_stages(p, true), xy = f2_stages(p, false);
    const C *tw = (const C *)p->xf_tw;
    // parts: 1 = the pass over z, 2 = the pass over y (the tuner times them one by one)
    if (forward) {
        if (parts & 1) k_zr2c<Real, R16><<<gz, p->f2_zthreads, smz, s>>>(M, p->f2_rs, p->f2_rb, nrows, xz, tw, p->f2_zpos, (const Real *)p->grid, (C *)p->spec);
        if (parts & 2) k_yfft<Real, NF, false, R16><<<gy, p->f2_ythreads, smy, s>>>(M, Mh, ncols, xy, tw, (C *)p->spec);
    } else {
        if (parts & 2) k_yfft<Real, NF, true, R16><<<gy, p->f2_ythreads, smy, s>>>(M, Mh, ncols, xy, tw, (C *)p->spec);
        if (parts & 1) k_zc2r<Real, R16><<<gzi, p->f2_zithreads, smzi, s>>>(M, p->f2_rs, p->f2_rbi, nrows, xz, tw, p->f2_zpos, (const C *)p->spec, (Real *)p->grid);
    }
    p->launches += 2;
    return cudaGetLastError();
}

cudaError_t fft2_dispatch(se_plan *p, bool forward, cudaStream_t s, bool prepare, int parts = 3)
{
    return p->precision == SE_FP64 ? fft2_impl<double, SE_YF_NF64, false>(p, forward, s, prepare, parts)
                                   : fft2_impl<float, SE_YF_NF32, true>(p, forward, s, prepare, parts);
}

// decides p->f2_ok and builds the tables of the own 2-D transforms (after se_build_ktab: the k_y table comes from the plan's)
template <typename Real, typename C>
cudaError_t fft2_build(se_plan *p)
{
    p->f2_ok = 0;
    const char *mode = std::getenv("SE_FFT_MODE");
    if (!p->xf_ok || (mode && std::strcmp(mode, "cufft2d") == 0)) return cudaSuccess;
    const int M = p->g.M, N2 = M / 2;
    const bool r16 = p->precision == SE_FP32;
    XfStages xz, xy;
    if (N2 < 2 || !xf_factor(N2, r16, xz, false) || !xf_factor(M, r16, xy, false)) return cudaSuccess;
    {
        // pass over z: the radix with the most factors of two first, so that consecutive k sit an odd (or less even) number of
        // positions apart and k_zc2r's stores into the digit-reversed positions spread over the banks (config 5: ifft 5.05 -> 4.87 ms)
        int best = 0;
        auto twos = [](int r) { int c = 0; while (!(r & 1)) { r >>= 1; ++c; } return c; };
        for (int i = 1; i < xz.nst; ++i) if (twos(xz.radix[i]) > twos(xz.radix[best])) best = i;
        std::swap(xz.radix[0], xz.radix[best]);
        int L = N2;
        for (int st = 0; st < xz.nst; ++st) {
            const int m = L / xz.radix[st];
            xz.magic[st] = m > 1 ? (unsigned)((0x100000000ull + (unsigned)m - 1) / (unsigned)m) : 0u;
            L = m;
        }
    }
    const int NF = p->precision == SE_FP64 ? SE_YF_NF64 : SE_YF_NF32;
    if ((size_t)M * NF * sizeof(C) > 227 * 1024) return cudaSuccess;
    // rows of the z-pass: stride = 1 mod 8 (fp32: 16) complex numbers, up to 16 rows in <= 100 KB (two blocks per SM)
    const int al = p->precision == SE_FP64 ? 8 : 16;
    int rs = N2 + 1;
    while (rs % al != 1) ++rs;
    const int rbmax = (int)std::min<size_t>(16, (size_t)113 * 1024 / ((size_t)rs * sizeof(C)));
    p->f2_rbmax = rbmax;
    int rb = std::min(8, rbmax);
    if (const char *e = std::getenv("SE_F2_RB")) rb = std::max(1, std::min(std::atoi(e), rbmax));
    if (rb < 4 && !std::getenv("SE_F2_RB")) return cudaSuccess;
    int bwz = std::max(1, std::min(192 / rb, 16)), bwy = std::max(4, 192 / NF);
    if (const char *e = std::getenv("SE_F2_BWZ")) bwz = std::max(1, std::min(std::atoi(e), 256 / rb));
    if (const char *e = std::getenv("SE_F2_BWY")) bwy = std::max(1, std::min(std::atoi(e), 192 / NF));
    int rbi = rb, bwzi = bwz;                                  // rows per block and lanes per row of the inverse pass over z
    if (const char *e = std::getenv("SE_F2_RBI")) rbi = std::max(1, std::min(std::atoi(e), rbmax));
    if (const char *e = std::getenv("SE_F2_BWZI")) bwzi = std::max(1, std::min(std::atoi(e), 256 / rbi));
    p->f2_rbi = rbi; p->f2_zithreads = rbi * bwzi;
    p->f2_rs = rs; p->f2_rb = rb; p->f2_zthreads = rb * bwz; p->f2_ythreads = NF * bwy;
    p->f2z_nst = xz.nst; p->f2y_nst = xy.nst;
    for (int i = 0; i < XF_MAXST; ++i) {
        p->f2z_radix[i] = xz.radix[i]; p->f2z_magic[i] = xz.magic[i];
        p->f2y_radix[i] = xy.radix[i]; p->f2y_magic[i] = xy.magic[i];
    }
    std::vector<int> zpos(N2);
    for (int pos = 0; pos < N2; ++pos) zpos[xf_rev(pos, N2, xz.nst, xz.radix)] = pos;
    std::vector<Real> kt(2 * (size_t)M);
    cudaError_t e = cudaMemcpy(kt.data(), p->ktab, kt.size() * sizeof(Real), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return e;
    std::vector<C> ykk(M);
    for (int pos = 0; pos < M; ++pos) {
        const int k = xf_rev(pos, M, xy.nst, xy.radix);
        ykk[pos].x = kt[k];
        ykk[pos].y = 2 * k == M ? (Real)0 : kt[M + k];
    }
    if ((e = cudaMalloc((void **)&p->f2_zpos, (size_t)N2 * sizeof(int))) != cudaSuccess) return e;
    if ((e = cudaMalloc(&p->f2_ykk, (size_t)M * sizeof(C))) != cudaSuccess) return e;
    p->workspace_bytes += (size_t)N2 * sizeof(int) + (size_t)M * sizeof(C);
    if ((e = cudaMemcpy(p->f2_zpos, zpos.data(), (size_t)N2 * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    if ((e = cudaMemcpy(p->f2_ykk, ykk.data(), (size_t)M * sizeof(C), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    if ((e = fft2_dispatch(p, true, nullptr, true)) != cudaSuccess) return e;
    p->f2_ok = 1;
    return cudaSuccess;
}

}  // namespace

// Block shape of K4x: NF columns x BW butterfly lanes.  How evenly the stages' butterfly counts M / R split over BW, how many
// blocks fit an SM and how well they hide one another's loads depends on M in a way a formula did not capture (config 3:
// 0.94 ms at BW = 12, 1.03-1.11 ms at BW = 14...21; config 5: 4.8 ms at BW = 10, 5.7-6.8 ms above), so the plan times the
// candidates once on its own (still unused) spectrum buffer.  The result of the kernel does not depend on BW.
template <typename Real, typename C>
cudaError_t xf_build_xkk(se_plan *p)
{
    // (k_x, e_x) of the mode at every position after the forward stages (mixed-radix digit reversal of the x-index), from the
    // plan's K4 table; e_x = 0 on the Nyquist plane (reading S8)
    const int M = p->g.M;
    std::vector<Real> kt(2 * (size_t)M);
    cudaError_t e = cudaMemcpy(kt.data(), p->ktab, kt.size() * sizeof(Real), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return e;
    std::vector<C> tab(M);
    for (int pos = 0; pos < M; ++pos) {
        int rem = pos, L = M, k = 0, mult = 1;
        for (int st = 0; st < p->xf_nst; ++st) {
            const int r = p->xf_radix[st], m = L / r;
            k += (rem / m) * mult;
            rem %= m; mult *= r; L = m;
        }
        tab[pos].x = kt[k];
        tab[pos].y = 2 * k == M ? (Real)0 : kt[M + k];
    }
    return cudaMemcpy(p->xf_xk, tab.data(), (size_t)M * sizeof(C), cudaMemcpyHostToDevice);
}

cudaError_t se_tune_xfft(se_plan *p)
{
    if (!p->xf_ok) return cudaSuccess;
    cudaError_t e = p->precision == SE_FP64 ? xf_build_xkk<double, double2>(p) : xf_build_xkk<float, float2>(p);
    if (e == cudaSuccess) e = p->precision == SE_FP64 ? fft2_build<double, double2>(p) : fft2_build<float, float2>(p);
    if (e != cudaSuccess || std::getenv("SE_XF_BW")) return e;
    const int nf = 3 * p->xf_tz, M = p->g.M;
    const size_t bytes = (size_t)3 * M * M * (M / 2 + 1) * 2 * p->real_bytes;
    e = cudaMemset(p->spec, 0, bytes);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    if ((e = cudaEventCreate(&e0)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return e; }
    const int saved = p->launches;
    int best = p->xf_threads;
    float bt = 1e30f;
    for (int bw = 256 / nf; bw >= 4 && e == cudaSuccess; --bw) {
        p->xf_threads = bw * nf;
        float ms = 1e30f;
        for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {              // first launch of a shape: warm-up
            cudaEventRecord(e0, nullptr);
            e = xf_dispatch(p, nullptr, false);
            cudaEventRecord(e1, nullptr);
            if (e == cudaSuccess) e = cudaEventSynchronize(e1);
            float t = 0.f;
            if (e == cudaSuccess && rep > 0 && cudaEventElapsedTime(&t, e0, e1) == cudaSuccess) ms = t < ms ? t : ms;
        }
        if (ms < bt) { bt = ms; best = bw * nf; }
    }
    p->xf_threads = best;
    // the same for the own 2-D transforms: rows per block x lanes per row of the two passes over z, lanes per column of the
    // pass over y (config 3 is fastest at 8 x 12, config 5 at 8 x 16, config 4 at 16 x 8)
    const bool f2env = std::getenv("SE_F2_RB") || std::getenv("SE_F2_BWZ") || std::getenv("SE_F2_RBI") || std::getenv("SE_F2_BWZI") ||
                       std::getenv("SE_F2_BWY");
    if (p->f2_ok && !f2env && e == cudaSuccess) e = cudaMemset(p->grid, 0, (size_t)3 * M * M * M * p->real_bytes);
    if (p->f2_ok && !f2env && e == cudaSuccess) {
        auto time_it = [&](bool forward, int parts) -> float {
            float ms = 1e30f;
            for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
                cudaEventRecord(e0, nullptr);
                e = fft2_dispatch(p, forward, nullptr, false, parts);
                cudaEventRecord(e1, nullptr);
                if (e == cudaSuccess) e = cudaEventSynchronize(e1);
                float t = 0.f;
                if (e == cudaSuccess && rep > 0 && cudaEventElapsedTime(&t, e0, e1) == cudaSuccess) ms = t < ms ? t : ms;
            }
            return ms;
        };
        static const int cand[][2] = {{8, 8}, {8, 12}, {8, 16}, {16, 8}, {16, 12}, {4, 16}};
        for (int inv = 0; inv < 2; ++inv) {
            int brb = inv ? p->f2_rbi : p->f2_rb, bth = inv ? p->f2_zithreads : p->f2_zthreads;
            float btz = 1e30f;
            for (const auto &c : cand) {
                if (c[0] > p->f2_rbmax) continue;
                (inv ? p->f2_rbi : p->f2_rb) = c[0];
                (inv ? p->f2_zithreads : p->f2_zthreads) = c[0] * c[1];
                const float ms = time_it(!inv, 1);
                if (ms < btz) { btz = ms; brb = c[0]; bth = c[0] * c[1]; }
            }
            (inv ? p->f2_rbi : p->f2_rb) = brb;
            (inv ? p->f2_zithreads : p->f2_zthreads) = bth;
        }
        const int NFy = p->precision == SE_FP64 ? SE_YF_NF64 : SE_YF_NF32;
        int bby = p->f2_ythreads;
        float bty = 1e30f;
        for (int bw = 192 / NFy; bw >= 4; bw -= (NFy <= 12 ? 2 : 1)) {
            p->f2_ythreads = bw * NFy;
            const float ms = time_it(true, 2) + time_it(false, 2);
            if (ms < bty) { bty = ms; bby = bw * NFy; }
        }
        p->f2_ythreads = bby;
    }
    p->launches = saved;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return e;
}

// the fused path's SE_STAGE_FFT / SE_STAGE_IFFT when the plan has its own 2-D transforms (p->f2_ok)
cudaError_t se_launch_fft2(se_plan *p, bool forward, cudaStream_t s) { return fft2_dispatch(p, forward, s, false); }
