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
#include "se_common.cuh"

namespace {

template <typename Real> struct Cplx;
template <> struct Cplx<double> { typedef double2 type; };
template <> struct Cplx<float> { typedef float2 type; };

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
    const Real kx = ktab[ix], ky = ktab[iy], kz = ktab[iz];
    const Real k2 = kx * kx + ky * ky + kz * kz;
    const bool nyq = (2 * ix == M) || (2 * iy == M) || (2 * iz == M);
    Real s = 0;
    if (!nyq && k2 > (Real)0) {
        const Real e = ktab[M + ix] * ktab[M + iy] * ktab[M + iz];
        s = pref * ((Real)1 + k2 * inv4xi2) * e / (k2 * k2);
    }
    C h0 = spec[idx], h1 = spec[nm + idx], h2 = spec[2 * nm + idx];
    const Real kr = kx * h0.x + ky * h1.x + kz * h2.x;
    const Real ki = kx * h0.y + ky * h1.y + kz * h2.y;
    C o0, o1, o2;
    o0.x = s * (k2 * h0.x - kx * kr); o0.y = s * (k2 * h0.y - kx * ki);
    o1.x = s * (k2 * h1.x - ky * kr); o1.y = s * (k2 * h1.y - ky * ki);
    o2.x = s * (k2 * h2.x - kz * kr); o2.y = s * (k2 * h2.y - kz * ki);
    spec[idx] = o0; spec[nm + idx] = o1; spec[2 * nm + idx] = o2;
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
