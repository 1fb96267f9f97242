// K2: near-field P2P,  u^N_i = sum_j sum_p [0 < |r| <= rc] G^N(r) f_j,  r = x_i - x_j + p
// (eq. (2.2), eq. (2.3)), over the 27 colleague cells.
//
// Design (differs from the paper's thread-per-target kernels): only ~15% of
// the candidates in the 27 cells are inside the cutoff sphere, so a thread-per-target loop
// runs the expensive erfc/exp code at ~15% lane utilisation.  Here ONE WARP owns a target:
//   phase A (cheap): lanes stride over the candidate sources, compute r and r^2, and
//            compact the in-range ones (ballot + popc) into a per-warp shared-memory queue;
//   phase B (heavy): whenever 32 pairs are queued, every lane evaluates one pair with all
//            lanes busy; G^N is evaluated in registers as
//              C1 = A - B,  C2 = (A + B)/r^2,  A = e^{-xi^2 r^2} erfcx(xi r)/r,  B = 2 xi e^{-xi^2 r^2}/sqrt(pi)
//            (erfc(x) = e^{-x^2} erfcx(x): one exponential serves both terms of (2.3));
//   per target one butterfly reduction of the three accumulators.
// The z-row of three colleague cells is contiguous in the sorted order and is scanned as one
// run.  fp64 uses absolute positions + the image shift exactly as eq. (2.2); fp32 uses
// cell-relative positions so that r keeps full float precision across periodic images.
#include "se_common.cuh"

namespace {

constexpr int P2P_WARPS = 4;
constexpr int P2P_TPW = 8;          // targets per warp
constexpr int P2P_Q = 64;           // queue slots per warp (circular)

template <typename Real> struct NearMath;

template <> struct NearMath<double> {
    static __device__ __forceinline__ void coeffs(double r2, double xi, double c2, double &C1, double &C2)
    {
        double rinv = rsqrt(r2);
        double x2 = xi * xi * r2;
        double e = exp(-x2);
        double A = e * erfcx(xi * (r2 * rinv)) * rinv;
        double B = c2 * e;
        C1 = A - B;
        C2 = (A + B) * (rinv * rinv);
    }
};

template <> struct NearMath<float> {
    static __device__ __forceinline__ void coeffs(float r2, float xi, float c2, float &C1, float &C2)
    {
        float rinv = rsqrtf(r2);
        float x2 = xi * xi * r2;
        float e = expf(-x2);
        float A = e * erfcxf(xi * (r2 * rinv)) * rinv;
        float B = c2 * e;
        C1 = A - B;
        C2 = (A + B) * (rinv * rinv);
    }
};

template <typename Real>
__global__ void __launch_bounds__(P2P_WARPS * 32)
k_p2p(SeGeom g, const Real *__restrict__ xs, const Real *__restrict__ fs,
      const int *__restrict__ cell_sorted, const int *__restrict__ cell_start, Real *__restrict__ uN)
{
    __shared__ Real qx[P2P_WARPS][P2P_Q], qy[P2P_WARPS][P2P_Q], qz[P2P_WARPS][P2P_Q];
    __shared__ int qj[P2P_WARPS][P2P_Q];

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int nc = g.ncell;
    const Real rc2 = (Real)(g.rc * g.rc);
    const Real xi = (Real)g.xi;
    const Real c2 = (Real)(2.0 * g.xi / sqrt(SE_PI));
    const Real Lr = (Real)g.L, wc = (Real)g.wcell;
    const bool rel = g.rel_coords != 0;

    const int64_t first = ((int64_t)blockIdx.x * P2P_WARPS + w) * P2P_TPW;

    for (int t = 0; t < P2P_TPW; ++t) {
        const int64_t i = first + t;
        if (i >= g.N) break;                                     // warp-uniform
        const Real xi0 = xs[3 * i + 0], xi1 = xs[3 * i + 1], xi2 = xs[3 * i + 2];
        const int ci = cell_sorted[i];
        const int cz = ci % nc, cy = (ci / nc) % nc, cx = ci / (nc * nc);
        Real a0 = 0, a1 = 0, a2 = 0;
        int head = 0, qn = 0;

        auto heavy = [&](int nvalid) {
            __syncwarp();
            if (lane < nvalid) {
                int k = (head + lane) & (P2P_Q - 1);
                Real rx = qx[w][k], ry = qy[w][k], rz = qz[w][k];
                int j = qj[w][k];
                Real f0 = fs[3 * (int64_t)j + 0], f1 = fs[3 * (int64_t)j + 1], f2 = fs[3 * (int64_t)j + 2];
                Real r2 = rx * rx + ry * ry + rz * rz;
                Real C1, C2;
                NearMath<Real>::coeffs(r2, xi, c2, C1, C2);
                Real rf = C2 * (rx * f0 + ry * f1 + rz * f2);
                a0 += C1 * f0 + rf * rx;
                a1 += C1 * f1 + rf * ry;
                a2 += C1 * f2 + rf * rz;
            }
            __syncwarp();
        };

        for (int dx = -1; dx <= 1; ++dx) {
            int nx = cx + dx;
            Real sx = 0;
            if (nx < 0) { nx += nc; sx = -Lr; } else if (nx >= nc) { nx -= nc; sx = Lr; }
            if (rel) sx = (Real)dx * wc;
            for (int dy = -1; dy <= 1; ++dy) {
                int ny = cy + dy;
                Real sy = 0;
                if (ny < 0) { ny += nc; sy = -Lr; } else if (ny >= nc) { ny -= nc; sy = Lr; }
                if (rel) sy = (Real)dy * wc;
                const int row = (nx * nc + ny) * nc;
                // z-row segments: contiguous cells [zlo, zhi], first cell has offset dzlo
                int nseg, zlo[2], zhi[2], dzlo[2];
                Real sseg[2];
                if (cz > 0 && cz < nc - 1) {
                    nseg = 1; zlo[0] = cz - 1; zhi[0] = cz + 1; dzlo[0] = -1; sseg[0] = 0;
                } else if (cz == 0) {
                    nseg = 2;
                    zlo[0] = nc - 1; zhi[0] = nc - 1; dzlo[0] = -1; sseg[0] = -Lr;
                    zlo[1] = 0; zhi[1] = 1; dzlo[1] = 0; sseg[1] = 0;
                } else {
                    nseg = 2;
                    zlo[0] = nc - 2; zhi[0] = nc - 1; dzlo[0] = -1; sseg[0] = 0;
                    zlo[1] = 0; zhi[1] = 0; dzlo[1] = 1; sseg[1] = Lr;
                }
                for (int sg = 0; sg < nseg; ++sg) {
                    const int jb = cell_start[row + zlo[sg]];
                    const int je = cell_start[row + zhi[sg] + 1];
                    // boundaries between the cells of the run (for the per-lane z offset, fp32 path)
                    const int b1 = (zhi[sg] > zlo[sg]) ? cell_start[row + zlo[sg] + 1] : 0x7fffffff;
                    const int b2 = (zhi[sg] > zlo[sg] + 1) ? cell_start[row + zlo[sg] + 2] : 0x7fffffff;
                    for (int j0 = jb; j0 < je; j0 += 32) {
                        const int j = j0 + lane;
                        bool in = false;
                        Real rx = 0, ry = 0, rz = 0;
                        if (j < je) {
                            Real sz = sseg[sg];
                            if (rel) sz = (Real)(dzlo[sg] + (j >= b1) + (j >= b2)) * wc;
                            rx = xi0 - (xs[3 * (int64_t)j + 0] + sx);
                            ry = xi1 - (xs[3 * (int64_t)j + 1] + sy);
                            rz = xi2 - (xs[3 * (int64_t)j + 2] + sz);
                            Real r2 = rx * rx + ry * ry + rz * rz;
                            in = (r2 <= rc2) && (r2 > (Real)0);
                        }
                        const unsigned m = __ballot_sync(0xffffffffu, in);
                        if (in) {
                            int k = (head + qn + __popc(m & lt_mask)) & (P2P_Q - 1);
                            qx[w][k] = rx; qy[w][k] = ry; qz[w][k] = rz; qj[w][k] = j;
                        }
                        qn += __popc(m);
                        if (qn >= 32) {
                            heavy(32);
                            head = (head + 32) & (P2P_Q - 1);
                            qn -= 32;
                        }
                    }
                }
            }
        }
        if (qn > 0) heavy(qn);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a0 += __shfl_xor_sync(0xffffffffu, a0, o);
            a1 += __shfl_xor_sync(0xffffffffu, a1, o);
            a2 += __shfl_xor_sync(0xffffffffu, a2, o);
        }
        if (lane == 0) { uN[3 * i + 0] = a0; uN[3 * i + 1] = a1; uN[3 * i + 2] = a2; }
        __syncwarp();
    }
}

template <typename Real>
cudaError_t p2p_impl(se_plan *p, cudaStream_t s)
{
    const SeGeom &g = p->g;
    int64_t per_block = (int64_t)P2P_WARPS * P2P_TPW;
    unsigned nblk = (unsigned)((g.N + per_block - 1) / per_block);
    k_p2p<Real><<<nblk, P2P_WARPS * 32, 0, s>>>(g, (const Real *)p->xs_near, (const Real *)p->fs_near,
                                               p->cell_sorted, p->cell_start, (Real *)p->uN);
    p->launches += 1;
    return cudaGetLastError();
}

}  // namespace

cudaError_t se_launch_p2p(se_plan *p, cudaStream_t s)
{
    return p->precision == SE_FP64 ? p2p_impl<double>(p, s) : p2p_impl<float>(p, s);
}
