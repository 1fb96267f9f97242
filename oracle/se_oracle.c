/*
 * ORACLE O2 -- spectral Ewald (SE) evaluation of the triply periodic Stokeslet sum,
 * Hasimoto split, Gaussian window.  Straight loops, double precision.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may use anything under oracle/.  Shares no
 * code with the CUDA path (paper_2606_19059_b200/csrc) nor with direct_ewald.c.
 *
 * Follows Algorithm 2.1 step by step; every stage is a separate
 * function so each intermediate (u^N, H, H~hat, H~, u^F) can be compared on its own.
 * The two FFTs are NOT here: the Python wrapper
 * (oracle/__init__.py) calls scipy.fft.fftn / ifftn (pocketfft, a library primitive) between
 * se_p2g and se_scale and between se_scale and se_g2p.
 *
 * Discretisation (readings S4, S5, S8, S11 in DESIGN.md):
 *   h = L/M;  m = 0.95 sqrt(pi P);  eta = (P h xi / m)^2;  a = 2 xi^2/eta;
 *   window w(r) = c_w e^{-a |r|^2}, c_w = (a/pi)^{3/2}, truncated to P grid points per
 *   dimension around the particle: anchor a_d = floor(x_d/h) - (P/2 - 1),
 *   offsets t_l = (a_d + l) h - x_d, l = 0..P-1, grid index (a_d + l) mod M.
 *   w_hat(k) = e^{-eta k^2/(8 xi^2)}.
 *
 * Second window (the paper's own, eq. (2.8)): truncated
 * Kaiser-Bessel  w0(r) = I0(beta sqrt(1 - r^2/a_w^2)) / I0(beta) for |r| < a_w, else 0, with
 * beta = 2.5 P, a_w = P h / 2, w(r) = w0(r1) w0(r2) w0(r3), same anchor and support points;
 * either evaluated exactly (WIN_KB, own power series of I0) or by the piecewise polynomial
 * of degree nu, one polynomial per bin of width h, Horner's rule (WIN_KBPOLY; the
 * coefficients are made by oracle/__init__.py:kb_poly_coeffs).  The deconvolution uses the
 * window's own transform w_hat0(k) (computed by quadrature in oracle/__init__.py:kb_what),
 * c_w = 1.  Readings S18-S20 in DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define PI 3.14159265358979323846264338327950288

/* ---- step 1: constants -------------------------------------------------------- */
void se_params(double L, double xi, int M, int P, double *out /* h, m, eta, a, cw */)
{
    double h = L / M;
    double m = 0.95 * sqrt(PI * P);
    double eta = (P * h * xi / m) * (P * h * xi / m);
    double a = 2.0 * xi * xi / eta;
    double cw = pow(a / PI, 1.5);
    out[0] = h; out[1] = m; out[2] = eta; out[3] = a; out[4] = cw;
}

/* ---- step 2: wrap into [0, L) -------------------------------------------------- */
void se_wrap(int64_t N, const double *x, double L, double *xw)
{
    for (int64_t i = 0; i < 3 * N; ++i) {
        double v = x[i] - L * floor(x[i] / L);
        if (v >= L) v = 0.0;
        if (v < 0.0) v = 0.0;
        xw[i] = v;
    }
}

/* near-field tensor applied to f:  G^N(r) f = C1 f + C2 r (r.f)
 * PAPER.md:59 eq. (2.3) expanded with G = I/r + r(x)r/r^3:
 *   G^N = G (erfc(xi r) + 2 xi r e^{-xi^2 r^2}/sqrt(pi)) - I 4 xi e^{-xi^2 r^2}/sqrt(pi)
 *   C1 = erfc/r + 2xi e/sqrt(pi) - 4 xi e/sqrt(pi) = erfc/r - 2 xi e/sqrt(pi)
 *   C2 = erfc/r^3 + 2 xi e/(sqrt(pi) r^2)
 */
static inline void near_pair(double rx, double ry, double rz, double r2, double xi,
                             const double *fj, double *acc)
{
    double r = sqrt(r2);
    double e = exp(-xi * xi * r2);
    double ec = erfc(xi * r);
    double c = 2.0 * xi / sqrt(PI);
    double C1 = ec / r - c * e;
    double C2 = ec / (r2 * r) + c * e / r2;
    double rf = rx * fj[0] + ry * fj[1] + rz * fj[2];
    acc[0] += C1 * fj[0] + C2 * rx * rf;
    acc[1] += C1 * fj[1] + C2 * ry * rf;
    acc[2] += C1 * fj[2] + C2 * rz * rf;
}

/* ---- step 3 (variant A): near field, plain O(Nt N 27) loop, eq. (2.2) PAPER.md:54 --
 * Targets are the particles listed in tidx (nt of them; tidx == NULL -> all N).
 * Images p in L{-1,0,1}^3 (requires rc <= L).  Keeps 0 < |r|^2 <= rc^2 (readings S6, S10).
 */
void se_near_brute(int64_t N, const double *xw, const double *f, double L, double xi, double rc,
                   int64_t nt, const int64_t *tidx, double *uN)
{
    double rc2 = rc * rc;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = tidx ? tidx[t] : t;
        double acc[3] = {0, 0, 0};
        for (int64_t j = 0; j < N; ++j)
            for (int px = -1; px <= 1; ++px)
            for (int py = -1; py <= 1; ++py)
            for (int pz = -1; pz <= 1; ++pz) {
                double rx = xw[3*i+0] - xw[3*j+0] + px * L;
                double ry = xw[3*i+1] - xw[3*j+1] + py * L;
                double rz = xw[3*i+2] - xw[3*j+2] + pz * L;
                double r2 = rx*rx + ry*ry + rz*rz;
                if (r2 > 0.0 && r2 <= rc2) near_pair(rx, ry, rz, r2, xi, f + 3*j, acc);
            }
        uN[3*t+0] = acc[0]; uN[3*t+1] = acc[1]; uN[3*t+2] = acc[2];
    }
}

/* ---- step 3 for separate targets (eq. (1.1)/(2.2)): nt target positions xt (wrapped),
 * N sources xw, plain loop over all sources and the 27 nearest images; r = 0 is skipped.
 */
void se_near_targets(int64_t N, const double *xw, const double *f, int64_t nt, const double *xt,
                     double L, double xi, double rc, double *uN)
{
    double rc2 = rc * rc;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < nt; ++t) {
        double acc[3] = {0, 0, 0};
        for (int64_t j = 0; j < N; ++j)
            for (int px = -1; px <= 1; ++px)
            for (int py = -1; py <= 1; ++py)
            for (int pz = -1; pz <= 1; ++pz) {
                double rx = xt[3*t+0] - xw[3*j+0] + px * L;
                double ry = xt[3*t+1] - xw[3*j+1] + py * L;
                double rz = xt[3*t+2] - xw[3*j+2] + pz * L;
                double r2 = rx*rx + ry*ry + rz*rz;
                if (r2 > 0.0 && r2 <= rc2) near_pair(rx, ry, rz, r2, xi, f + 3*j, acc);
            }
        uN[3*t+0] = acc[0]; uN[3*t+1] = acc[1]; uN[3*t+2] = acc[2];
    }
}

/* ---- step 3 (variant B): near field with a cell list: cells of width
 * L/ncell >= rc, ncell = floor(L/rc) (reading S7), 27 colleague cells with periodic
 * shifts.  Needs ncell >= 3.  Same pair arithmetic as variant A; cross-checked in tests.
 */
int se_near_cells(int64_t N, const double *xw, const double *f, double L, double xi, double rc,
                  double *uN)
{
    int nc = (int)floor(L / rc);
    if (nc < 3) return 1;
    double w = L / nc, rc2 = rc * rc;
    int64_t ncell = (int64_t)nc * nc * nc;
    int64_t *start = (int64_t *)calloc((size_t)(ncell + 1), sizeof(int64_t));
    int64_t *cell = (int64_t *)malloc((size_t)N * sizeof(int64_t));
    int64_t *order = (int64_t *)malloc((size_t)N * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) {
        int c[3];
        for (int d = 0; d < 3; ++d) {
            c[d] = (int)floor(xw[3*i+d] / w);
            if (c[d] >= nc) c[d] = nc - 1;
            if (c[d] < 0) c[d] = 0;
        }
        cell[i] = ((int64_t)c[0] * nc + c[1]) * nc + c[2];
        start[cell[i] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) start[c+1] += start[c];
    int64_t *fill = (int64_t *)malloc((size_t)ncell * sizeof(int64_t));
    memcpy(fill, start, (size_t)ncell * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) order[fill[cell[i]]++] = i;

    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; ++i) {
        int64_t ci = cell[i];
        int c0 = (int)(ci / ((int64_t)nc * nc)), c1 = (int)((ci / nc) % nc), c2 = (int)(ci % nc);
        double acc[3] = {0, 0, 0};
        for (int d0 = -1; d0 <= 1; ++d0)
        for (int d1 = -1; d1 <= 1; ++d1)
        for (int d2 = -1; d2 <= 1; ++d2) {
            int n0 = c0 + d0, n1 = c1 + d1, n2 = c2 + d2;
            double s0 = 0, s1 = 0, s2 = 0;        /* shift applied to the source */
            if (n0 < 0) { n0 += nc; s0 = -L; } else if (n0 >= nc) { n0 -= nc; s0 = L; }
            if (n1 < 0) { n1 += nc; s1 = -L; } else if (n1 >= nc) { n1 -= nc; s1 = L; }
            if (n2 < 0) { n2 += nc; s2 = -L; } else if (n2 >= nc) { n2 -= nc; s2 = L; }
            int64_t cj = ((int64_t)n0 * nc + n1) * nc + n2;
            for (int64_t q = start[cj]; q < start[cj+1]; ++q) {
                int64_t j = order[q];
                double rx = xw[3*i+0] - (xw[3*j+0] + s0);
                double ry = xw[3*i+1] - (xw[3*j+1] + s1);
                double rz = xw[3*i+2] - (xw[3*j+2] + s2);
                double r2 = rx*rx + ry*ry + rz*rz;
                if (r2 > 0.0 && r2 <= rc2) near_pair(rx, ry, rz, r2, xi, f + 3*j, acc);
            }
        }
        uN[3*i+0] = acc[0]; uN[3*i+1] = acc[1]; uN[3*i+2] = acc[2];
    }
    free(start); free(cell); free(order); free(fill);
    return 0;
}

/* window kinds; wpar = {a} (Gaussian), {beta, a_w} (KB), {nu, c[P][nu+1]} (KB polynomial) */
#define WIN_GAUSS 0
#define WIN_KB 1
#define WIN_KBPOLY 2

/* modified Bessel function I0(x) = sum_k (x^2/4)^k / (k!)^2  (all terms positive: no cancellation) */
double se_bessel_i0(double x)
{
    double q = 0.25 * x * x, term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

/* truncated Kaiser-Bessel window, eq. (2.8) */
double se_kb_window(double r, double beta, double aw)
{
    double z = r / aw;
    if (!(fabs(z) < 1.0)) return 0.0;
    return se_bessel_i0(beta * sqrt(1.0 - z * z)) / se_bessel_i0(beta);
}

/* one window value at the physical offset t of support point l (reading S11) */
static inline double window_value(double t, int l, double h, int P, int wkind, const double *wpar)
{
    if (wkind == WIN_GAUSS) return exp(-wpar[0] * t * t);
    if (wkind == WIN_KB) return se_kb_window(t, wpar[0], wpar[1]);
    /* WIN_KBPOLY: bin l is r in [(l - P/2) h, (l - P/2 + 1) h]; local variable s in [-1, 1] */
    int nu = (int)wpar[0];
    const double *c = wpar + 1 + (size_t)l * (nu + 1);
    double s = 2.0 * (t / h - (double)(l - P / 2)) - 1.0;
    double v = c[nu];
    for (int k = nu - 1; k >= 0; --k) v = v * s + c[k];       /* Horner: nu multiply-adds */
    return v;
}

/* 1-D window table of one particle along one dimension (step 4 of the O2 definition) */
static inline void window_1d(double xd, double h, int M, int P, int wkind, const double *wpar, double *W, int *idx)
{
    long anchor = (long)floor(xd / h) - (P / 2 - 1);
    for (int l = 0; l < P; ++l) {
        double t = (double)(anchor + l) * h - xd;
        W[l] = window_value(t, l, h, P, wkind, wpar);
        long g = (anchor + l) % M;
        if (g < 0) g += M;
        idx[l] = (int)g;
    }
}

/* the P window values of one coordinate (tests) */
void se_window_1d(double xd, double L, int M, int P, int wkind, const double *wpar, double *W, int *idx)
{
    window_1d(xd, L / M, M, P, wkind, wpar, W, idx);
}

/* ---- step 4: P2G, eq. (2.5) PAPER.md:80 ------------------------------------------
 * H_c[i1,i2,i3] += c_w W1[l1] W2[l2] W3[l3] f_c.  H is (3, M, M, M), z fastest, zeroed here.
 * Threads own disjoint slabs of x-planes and each scans all particles, so every grid
 * point is accumulated in particle order whatever the thread count.
 */
#define PMAX 64
void se_p2g(int64_t N, const double *xw, const double *f, double L, int M, int P,
            int wkind, const double *wpar, double cw, double *H)
{
    double h = L / M;
    size_t M3 = (size_t)M * M * M;
    memset(H, 0, 3 * M3 * sizeof(double));
    #pragma omp parallel for schedule(static)
    for (int i1 = 0; i1 < M; ++i1) {
        double W1[PMAX], W2[PMAX], W3[PMAX];
        int I1[PMAX], I2[PMAX], I3[PMAX];
        for (int64_t n = 0; n < N; ++n) {
            /* does this particle's support contain plane i1?  l = (i1 - anchor) mod M < P */
            long anchor = (long)floor(xw[3*n+0] / h) - (P / 2 - 1);
            long lq = ((long)i1 - anchor) % M;
            if (lq < 0) lq += M;
            if (lq >= P) continue;
            int hit = (int)lq;
            window_1d(xw[3*n+0], h, M, P, wkind, wpar, W1, I1);
            window_1d(xw[3*n+1], h, M, P, wkind, wpar, W2, I2);
            window_1d(xw[3*n+2], h, M, P, wkind, wpar, W3, I3);
            for (int l2 = 0; l2 < P; ++l2)
                for (int l3 = 0; l3 < P; ++l3) {
                    double w = cw * W1[hit] * W2[l2] * W3[l3];
                    size_t g = ((size_t)i1 * M + I2[l2]) * M + I3[l3];
                    H[0*M3 + g] += w * f[3*n+0];
                    H[1*M3 + g] += w * f[3*n+1];
                    H[2*M3 + g] += w * f[3*n+2];
                }
        }
    }
}

/* P2G evaluated one grid point at a time (gather form of the same sum): for sampled
 * grid indices gi (ns x 3) returns Hs (ns x 3 comps).  O(N) per sample. */
void se_p2g_points(int64_t N, const double *xw, const double *f, double L, int M, int P,
                   int wkind, const double *wpar, double cw, int64_t ns, const int32_t *gi, double *Hs)
{
    double h = L / M;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < ns; ++s) {
        double acc[3] = {0, 0, 0};
        for (int64_t n = 0; n < N; ++n) {
            double w = cw; int ok = 1;
            for (int d = 0; d < 3 && ok; ++d) {
                /* is grid index gi[d] inside this particle's P-point support? */
                long anchor = (long)floor(xw[3*n+d] / h) - (P / 2 - 1);
                long lq = ((long)gi[3*s+d] - anchor) % M;
                if (lq < 0) lq += M;
                if (lq >= P) { ok = 0; break; }
                double t = (double)(anchor + lq) * h - xw[3*n+d];
                w *= window_value(t, (int)lq, h, P, wkind, wpar);
            }
            if (!ok) continue;
            acc[0] += w * f[3*n+0]; acc[1] += w * f[3*n+1]; acc[2] += w * f[3*n+2];
        }
        Hs[3*s+0] = acc[0]; Hs[3*s+1] = acc[1]; Hs[3*s+2] = acc[2];
    }
}

/* ---- step 6: scaling of one mode, eq. (2.6) PAPER.md:88 with (2.4b) PAPER.md:69 ------
 *   H~hat(k) = (h^3/V) 8 pi k^-4 (1 + k^2/4xi^2) e^{-(1-eta) k^2/4xi^2} (k^2 Hhat - k (k.Hhat))
 * (G^F_hat / w_hat^2 with w_hat = e^{-eta k^2/8xi^2};  h^3 = P2G quadrature weight folded
 * in here, 1/V = Fourier-series normalisation, reading S1).  Zero for k = 0 (S2) and on
 * every Nyquist plane idx_d = M/2 when M is even (S8).
 * what == NULL: the Gaussian window as above.  what != NULL (Kaiser-Bessel): what[i] is the 1-D window
 * transform w_hat0 at the wavenumber of index i, w_hat(k) = w_hat0(k1) w_hat0(k2) w_hat0(k3), and the
 * factor is e^{-k^2/4xi^2} / w_hat(k)^2, eq. (2.6) as printed.
 * in/out: 3 complex numbers as {re,im} pairs.
 */
void se_scale_mode(int M, double L, double xi, double eta, const double *what, const int *idx,
                   const double *in, double *out)
{
    double k[3];
    int zero = 1, nyq = 0;
    for (int d = 0; d < 3; ++d) {
        int n = idx[d];
        if (2 * n == M) nyq = 1;          /* Nyquist plane (M even only) */
        if (2 * n >= M) n -= M;           /* idx >= M/2 -> idx - M */
        if (n != 0) zero = 0;
        k[d] = 2.0 * PI * n / L;
    }
    if (zero || nyq) { for (int q = 0; q < 6; ++q) out[q] = 0.0; return; }
    double k2 = k[0]*k[0] + k[1]*k[1] + k[2]*k[2];
    double q4 = k2 / (4.0 * xi * xi);
    double h = L / M;
    double dec;
    if (what) {
        double wh = what[idx[0]] * what[idx[1]] * what[idx[2]];
        dec = exp(-q4) / (wh * wh);
    } else
        dec = exp(-(1.0 - eta) * q4);
    double s = (h*h*h / (L*L*L)) * 8.0 * PI / (k2*k2) * (1.0 + q4) * dec;
    double kHr = k[0]*in[0] + k[1]*in[2] + k[2]*in[4];
    double kHi = k[0]*in[1] + k[1]*in[3] + k[2]*in[5];
    for (int c = 0; c < 3; ++c) {
        out[2*c+0] = s * (k2 * in[2*c+0] - k[c] * kHr);
        out[2*c+1] = s * (k2 * in[2*c+1] - k[c] * kHi);
    }
}

/* whole spectrum, full complex-to-complex layout (3, M, M, M) of {re,im}, in place */
void se_scale(int M, double L, double xi, double eta, const double *what, double *Hhat)
{
    size_t M3 = (size_t)M * M * M;
    #pragma omp parallel for schedule(static)
    for (int i = 0; i < M; ++i)
        for (int j = 0; j < M; ++j)
            for (int k = 0; k < M; ++k) {
                size_t g = ((size_t)i * M + j) * M + k;
                int idx[3] = {i, j, k};
                double in[6], out[6];
                for (int c = 0; c < 3; ++c) { in[2*c] = Hhat[2*(c*M3+g)]; in[2*c+1] = Hhat[2*(c*M3+g)+1]; }
                se_scale_mode(M, L, xi, eta, what, idx, in, out);
                for (int c = 0; c < 3; ++c) { Hhat[2*(c*M3+g)] = out[2*c]; Hhat[2*(c*M3+g)+1] = out[2*c+1]; }
            }
}

/* ---- step 8: G2P, eq. (2.7) PAPER.md:94 ----------------------------------------------
 * u^F_{i,c} = h^3 c_w sum_{l1 l2 l3} W1 W2 W3 H~_c[i1,i2,i3]; same W, idx as P2G.
 * Ht is (3, M, M, M); targets are the nt positions in xt (wrapped).
 */
void se_g2p(int64_t nt, const double *xt, double L, int M, int P, int wkind, const double *wpar, double cw,
            const double *Ht, double *uF)
{
    double h = L / M;
    size_t M3 = (size_t)M * M * M;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t n = 0; n < nt; ++n) {
        double W1[PMAX], W2[PMAX], W3[PMAX];
        int I1[PMAX], I2[PMAX], I3[PMAX];
        window_1d(xt[3*n+0], h, M, P, wkind, wpar, W1, I1);
        window_1d(xt[3*n+1], h, M, P, wkind, wpar, W2, I2);
        window_1d(xt[3*n+2], h, M, P, wkind, wpar, W3, I3);
        double acc[3] = {0, 0, 0};
        for (int l1 = 0; l1 < P; ++l1)
            for (int l2 = 0; l2 < P; ++l2)
                for (int l3 = 0; l3 < P; ++l3) {
                    double w = W1[l1] * W2[l2] * W3[l3];
                    size_t g = ((size_t)I1[l1] * M + I2[l2]) * M + I3[l3];
                    acc[0] += w * Ht[0*M3 + g];
                    acc[1] += w * Ht[1*M3 + g];
                    acc[2] += w * Ht[2*M3 + g];
                }
        double s = h * h * h * cw;
        uF[3*n+0] = s * acc[0]; uF[3*n+1] = s * acc[1]; uF[3*n+2] = s * acc[2];
    }
}

/* ---- step 9: SUM + self term (self term: reading S3) --------------------- */
void se_sum(int64_t N, const double *uN, const double *uF, const double *f, double xi, double *u)
{
    double cs = 4.0 * xi / sqrt(PI);
    for (int64_t i = 0; i < 3 * N; ++i) u[i] = uN[i] + uF[i] - cs * f[i];
}
