/*
 * ORACLE O1 -- direct Ewald summation of the triply periodic Stokeslet sum.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, double precision.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may use anything under oracle/.  Shares no code with the CUDA path nor with
 * se_oracle.c.
 *
 * What it computes (the definition the spectral Ewald method approximates):
 *
 *   u(x_i) = sum_j sum_{p in L Z^3, 0<|r|<=R} G^N(r) f_j                     [real space]
 *          + (1/V) sum_{k in (2pi/L) Z^3 \ {0}, |k_d|<=K} G^F_hat(k) Re[e^{ik.x_i} S(k)]   [k space]
 *          - (4 xi / sqrt(pi)) f_i                                            [self, targets==sources only]
 *
 *   r = x_i - y_j + p,   S(k) = sum_j f_j e^{-ik.y_j}
 *
 *   G^N(r)  : PAPER.md:59  eq. (2.3), with G(r) = I/|r| + r (x) r/|r|^3:
 *             G^N(r) f = C1 f + C2 r (r.f),
 *             C1 = erfc(xi r)/r - (2 xi/sqrt(pi)) e^{-xi^2 r^2}
 *             C2 = erfc(xi r)/r^3 + (2 xi/sqrt(pi)) e^{-xi^2 r^2}/r^2
 *   G^F_hat : PAPER.md:69  eq. (2.4b):
 *             G^F_hat(k) v = 8 pi k^-4 (1 + k^2/(4 xi^2)) e^{-k^2/(4 xi^2)} (k^2 v - k (k.v))
 *   3-periodic inverse transform (1/V) sum_k  : reading S1 in DESIGN.md (the paper
 *             writes only the 1-periodic form (2.4c), and says 3P needs
 *             no kernel changes).  k = 0 dropped: reading S2.
 *   self    : reading S3, = lim_{r->0} [G^N(r) - G(r)] f from (2.3).
 *
 * R and K are passed in; the Python wrapper picks R = 6.3/xi, K = 12.6 xi so that
 * e^{-xi^2 R^2} and e^{-K^2/4xi^2} are < 1e-17: the sums are converged to rounding
 * and the result is independent of xi (the main pin).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define PI 3.14159265358979323846264338327950288

/* real-space part at one target t from all sources, all images within R */
static void de_real_one(const double *t, int64_t Ns, const double *y, const double *f,
                        double L, double xi, double R, double *u)
{
    int nimg = (int)ceil(R / L);
    double R2 = R * R, c = 2.0 * xi / sqrt(PI);
    double a0 = 0, a1 = 0, a2 = 0;
    for (int64_t j = 0; j < Ns; ++j) {
        for (int px = -nimg; px <= nimg; ++px)
        for (int py = -nimg; py <= nimg; ++py)
        for (int pz = -nimg; pz <= nimg; ++pz) {
            double rx = t[0] - y[3*j+0] + px * L;
            double ry = t[1] - y[3*j+1] + py * L;
            double rz = t[2] - y[3*j+2] + pz * L;
            double r2 = rx*rx + ry*ry + rz*rz;
            if (r2 == 0.0 || r2 > R2) continue;
            double r = sqrt(r2);
            double e = exp(-xi*xi*r2);
            double ec = erfc(xi*r);
            double C1 = ec / r - c * e;
            double C2 = ec / (r2*r) + c * e / r2;
            double rf = rx*f[3*j+0] + ry*f[3*j+1] + rz*f[3*j+2];
            a0 += C1*f[3*j+0] + C2*rx*rf;
            a1 += C1*f[3*j+1] + C2*ry*rf;
            a2 += C1*f[3*j+2] + C2*rz*rf;
        }
    }
    u[0] = a0; u[1] = a1; u[2] = a2;
}

/*
 * Nt targets xt (3*Nt), Ns sources y, forces f.  If add_self != 0 the targets are
 * the sources (Nt == Ns, xt == y) and the self term is added.  Output u (3*Nt).
 */
void de_eval(int64_t Nt, const double *xt, int64_t Ns, const double *y, const double *f,
             double L, double xi, double R, double K, int add_self, double *u)
{
    /* ---- real space ---- */
    #pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < Nt; ++i)
        de_real_one(xt + 3*i, Ns, y, f, L, xi, R, u + 3*i);

    /* ---- k space ---- */
    int nmax = (int)floor(K * L / (2.0 * PI));
    int64_t nside = 2 * (int64_t)nmax + 1;
    /* half space: enumerate all k, use k and -k separately (plain, no symmetry tricks) */
    int64_t nk = nside * nside * nside;
    double V = L * L * L;
    double *acc = (double *)calloc((size_t)(3 * Nt), sizeof(double));

    #pragma omp parallel
    {
        double *loc = (double *)calloc((size_t)(3 * Nt), sizeof(double));
        #pragma omp for schedule(dynamic, 64)
        for (int64_t q = 0; q < nk; ++q) {
            int n0 = (int)(q / (nside * nside)) - nmax;
            int n1 = (int)((q / nside) % nside) - nmax;
            int n2 = (int)(q % nside) - nmax;
            if (n0 == 0 && n1 == 0 && n2 == 0) continue;
            double kx = 2.0 * PI * n0 / L, ky = 2.0 * PI * n1 / L, kz = 2.0 * PI * n2 / L;
            double k2 = kx*kx + ky*ky + kz*kz;
            double q4 = k2 / (4.0 * xi * xi);
            double B = 8.0 * PI / (k2 * k2) * (1.0 + q4) * exp(-q4);
            if (B == 0.0) continue;
            /* structure factor S(k) = sum_j f_j e^{-i k.y_j} */
            double Sr[3] = {0, 0, 0}, Si[3] = {0, 0, 0};
            for (int64_t j = 0; j < Ns; ++j) {
                double ph = kx*y[3*j] + ky*y[3*j+1] + kz*y[3*j+2];
                double cs = cos(ph), sn = sin(ph);
                for (int c = 0; c < 3; ++c) { Sr[c] += f[3*j+c] * cs; Si[c] -= f[3*j+c] * sn; }
            }
            /* T = k^2 S - k (k.S), real and imaginary parts */
            double kSr = kx*Sr[0] + ky*Sr[1] + kz*Sr[2];
            double kSi = kx*Si[0] + ky*Si[1] + kz*Si[2];
            double kk[3] = {kx, ky, kz};
            double Tr[3], Ti[3];
            for (int c = 0; c < 3; ++c) { Tr[c] = k2*Sr[c] - kk[c]*kSr; Ti[c] = k2*Si[c] - kk[c]*kSi; }
            for (int64_t i = 0; i < Nt; ++i) {
                double ph = kx*xt[3*i] + ky*xt[3*i+1] + kz*xt[3*i+2];
                double cs = cos(ph), sn = sin(ph);
                /* Re[(cs + i sn)(Tr + i Ti)] = cs Tr - sn Ti */
                for (int c = 0; c < 3; ++c) loc[3*i+c] += B * (cs*Tr[c] - sn*Ti[c]);
            }
        }
        #pragma omp critical
        for (int64_t i = 0; i < 3 * Nt; ++i) acc[i] += loc[i];
        free(loc);
    }

    double cself = 4.0 * xi / sqrt(PI);
    for (int64_t i = 0; i < Nt; ++i)
        for (int c = 0; c < 3; ++c) {
            double v = u[3*i+c] + acc[3*i+c] / V;
            if (add_self) v -= cself * f[3*i+c];
            u[3*i+c] = v;
        }
    free(acc);
}
