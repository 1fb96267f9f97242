// Host-side tables of the two windows and the parameter selection of PAPER.md section 2.4.
//   - se_build_ktab:   per 1-D index the wavenumber k and the factor e^{-k^2/4xi^2} / w_hat0(k)^2 of eq. (2.6)
//                      (PAPER.md:88); its 3-D value is the product of three entries, so K4 evaluates no exp.
//   - se_build_wcoef:  Kaiser-Bessel window (eq. (2.8)) as one polynomial per bin of width h
//                      (PAPER.md:421-427), interpolated at Chebyshev nodes in long double.
//   - se_select_params / se_plan_create_tol: eps -> (rc, xi, M, P) from the error estimate (2.9).
// All of it is plain host arithmetic; nothing here runs per evaluation.
#include <cmath>
#include <vector>

#include "se_common.cuh"

namespace {

// I0(x) = sum_k (x^2/4)^k / (k!)^2 in long double (all terms positive)
long double bessel_i0(long double x)
{
    const long double q = 0.25L * x * x;
    long double term = 1.0L, sum = 1.0L;
    for (int k = 1; k < 1000; ++k) {
        term *= q / ((long double)k * (long double)k);
        sum += term;
        if (term < 1e-22L * sum) break;
    }
    return sum;
}

struct KbBin { long double beta, z0, z1; };    // bin [z0, z1] of z = r / a_w

// the window on a bin, as a function of the local variable s in [-1, 1]
long double kb_on_bin(long double s, const void *ctx)
{
    const KbBin *b = (const KbBin *)ctx;
    const long double z = 0.5L * (b->z0 + b->z1) + 0.5L * (b->z1 - b->z0) * s;
    const long double a = 1.0L - z * z;
    return bessel_i0(b->beta * sqrtl(a > 0 ? a : 0.0L)) / bessel_i0(b->beta);
}

// closed-form transform of the truncated Kaiser-Bessel window: int_{-aw}^{aw} w0(r) cos(k r) dr
long double kb_what(long double k, long double beta, long double aw)
{
    const long double kap = k * aw, d = beta * beta - kap * kap;
    long double v;
    if (d > 0) { const long double q = sqrtl(d); v = sinhl(q) / q; }
    else if (d < 0) { const long double q = sqrtl(-d); v = sinl(q) / q; }
    else v = 1.0L;
    return 2.0L * aw * v / bessel_i0(beta);
}

bool smooth7(int n)
{
    for (int q : {2, 3, 5, 7})
        while (n % q == 0) n /= q;
    return n == 1;
}

}  // namespace

int se_kb_degree(int P) { return P + 3 < 13 ? P + 3 : 13; }       // reading S19

cudaError_t se_build_ktab(se_plan *p)
{
    const SeGeom &g = p->g;
    const int M = g.M;
    std::vector<long double> k(M), fac(M);
    const long double PI = 3.14159265358979323846264338327950288L;
    const long double beta = 2.5L * g.P, aw = 0.5L * g.P * (long double)g.h;
    for (int i = 0; i < M; ++i) {
        const int n = (2 * i >= M) ? i - M : i;
        k[i] = 2.0L * PI * (long double)n / (long double)g.L;
        const long double q4 = k[i] * k[i] / (4.0L * (long double)g.xi * (long double)g.xi);
        if (g.window == SE_WINDOW_KAISER_BESSEL) {
            const long double wh = kb_what(k[i], beta, aw);
            fac[i] = expl(-q4) / (wh * wh);
        } else
            fac[i] = expl(-(1.0L - (long double)g.eta) * q4);
    }
    cudaError_t e;
    if (p->precision == SE_FP64) {
        std::vector<double> h(2 * (size_t)M);
        for (int i = 0; i < M; ++i) { h[i] = (double)k[i]; h[M + i] = (double)fac[i]; }
        e = cudaMemcpy(p->ktab, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice);
    } else {
        std::vector<float> h(2 * (size_t)M);
        for (int i = 0; i < M; ++i) { h[i] = (float)k[i]; h[M + i] = (float)fac[i]; }
        e = cudaMemcpy(p->ktab, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice);
    }
    return e;
}

cudaError_t se_build_wcoef(se_plan *p)
{
    const SeGeom &g = p->g;
    if (g.window != SE_WINDOW_KAISER_BESSEL) return cudaSuccess;
    const int P = g.P, nu = g.nu;
    std::vector<double> c((size_t)P * (nu + 1));
    for (int l = 0; l < P; ++l) {
        // bin l: r in [(l - P/2) h, (l - P/2 + 1) h], i.e. z = r / a_w in [2 l / P - 1, 2 (l + 1) / P - 1]
        KbBin b{2.5L * P, 2.0L * l / P - 1.0L, 2.0L * (l + 1) / P - 1.0L};
        se_cheb_fit(kb_on_bin, &b, 0.0L, 1.0L, nu, &c[(size_t)l * (nu + 1)]);
    }
    cudaError_t e = cudaMalloc(&p->wcoef, c.size() * sizeof(double));
    if (e != cudaSuccess) return e;
    p->workspace_bytes += c.size() * sizeof(double);
    return cudaMemcpy(p->wcoef, c.data(), c.size() * sizeof(double), cudaMemcpyHostToDevice);
}

// ---- parameter selection, PAPER.md:142-167 ---------------------------------------------------------------------
namespace {

// the three terms of eq. (2.9) in unit-box variables
double err_near(double xi, double rc) { return std::sqrt(112.0 / 9.0 * xi * xi * xi * xi * rc * rc * rc) * std::exp(-xi * xi * rc * rc); }
double err_grid(double xi, double h)
{
    const double c = SE_PI / (2.0 * h * xi);
    return 4.0 / (3.0 * h) * std::sqrt(3.5) * std::exp(-c * c);
}
// E^w.  The constant C(xi) of (2.9) is not printed, and on a grid without oversampling (the 3-periodic case) the window
// error is set by aliasing at the resolved wavenumbers rather than by e^{-2.5 P}; reading S21 evaluates it directly:
//   E^w = 2 max_{0 <= theta <= 1} e^{-(theta c)^2} |w_hat0(k - 2 pi/h) / w_hat0(k)|  +  truncation,   k = theta pi/h,
// c = pi/(2 h xi): the spectrum's decay times the window's aliasing ratio, once for P2G and once for G2P.
//   Gaussian (m = 0.95 sqrt(pi P)): ratio = e^{-pi^2 P^2 (1 - theta)/(2 m^2)}, truncation = erfc(m / sqrt 2);
//   Kaiser-Bessel: ratio from the closed-form transform, truncation contained in it.
// Against the oracle's measured far-field error at config 1's split the estimate is within a factor 2 for P = 4 .. 24
// (S21).
double err_window(int window, int P, double xi, double h)
{
    const double c = SE_PI / (2.0 * h * xi);
    const double m = 0.95 * std::sqrt(SE_PI * P);
    const long double beta = 2.5L * P, aw = 0.5L * P * h;
    double worst = 0.0;
    for (int i = 0; i <= 400; ++i) {
        const double th = i / 400.0;
        double ratio;
        if (window == SE_WINDOW_GAUSSIAN)
            ratio = std::exp(-SE_PI * SE_PI * P * P * (1.0 - th) / (2.0 * m * m));
        else {
            const long double k = th * SE_PI / h;
            ratio = (double)fabsl(kb_what(k - 2.0L * SE_PI / h, beta, aw) / kb_what(k, beta, aw));
        }
        worst = std::max(worst, std::exp(-th * th * c * c) * ratio);
    }
    return 2.0 * worst + (window == SE_WINDOW_GAUSSIAN ? std::erfc(m / std::sqrt(2.0)) : 0.0);
}

// B200 stage-time model (seconds), constants from this repository's measured stage times:
// K2 72 G in-range pairs/s (fp64; x 2.5 in fp32) plus 1 ns per 32 candidates, K3 + K5 at 17 TFLOP/s on 6 P^3 flop per
// point (FP64 datapath, both precisions), FFTs at 1.0 TB/s of single-pass traffic, K4 at the HBM copy rate.
double model_time(double N, double rc, int M, int P, int prec)
{
    const double B = prec == SE_FP64 ? 8.0 : 4.0;
    const double pairs = N * (4.0 / 3.0) * SE_PI * rc * rc * rc * N;
    const double cand = N * 27.0 * rc * rc * rc * N;
    const double t_p2p = pairs / (prec == SE_FP64 ? 72e9 : 180e9) + cand / 32.0 * 0.25e-9;
    const double t_grid = 2.0 * (6.0 * P * P * P * N) / 17e12 + 2.0 * N * 1.6e3 / 3e12 + 2.0 * 3.0 * B * (double)M * M * M / 3e12;
    const double M3 = (double)M * M * M;
    const double t_fft = 2.0 * 3.0 * (B * M3 + B * M3) / 1.0e12;
    const double t_scale = 12.0 * B * (M3 / 2) / 6.5e12;
    return t_p2p + t_grid + t_fft + t_scale + N * 1.0e-9;
}

}  // namespace

extern "C" se_status se_select_params(int64_t N, double L, double eps, se_window window, se_precision prec, se_params *out)
{
    if (!out || !(N >= 1) || !(L > 0) || !std::isfinite(L) || !(eps > 1e-15) || !(eps < 1e-1)) return SE_EINVAL;
    if (window != SE_WINDOW_GAUSSIAN && window != SE_WINDOW_KAISER_BESSEL) return SE_EINVAL;
    if (prec != SE_FP64 && prec != SE_FP32) return SE_EINVAL;
    const double third = eps / 3.0;
    const int Pmax = window == SE_WINDOW_KAISER_BESSEL ? 16 : SE_PMAX;
    bool found = false;
    se_params best{};
    // scan rc (unit box) on a geometric grid from 1/3 (three cells per dimension) downwards
    for (int it = 0; it < 240; ++it) {
        const double rc = (1.0 / 3.0) * std::pow(0.98, it);
        if (rc < 1.0 / 1024) break;
        // xi(rc): smallest xi with E^N <= eps/3 (E^N falls with xi once xi rc > 1)
        double lo = 1.0 / rc, hi = 12.0 / rc;
        if (err_near(hi, rc) > third) continue;
        for (int b = 0; b < 80; ++b) { const double mid = 0.5 * (lo + hi); (err_near(mid, rc) > third ? lo : hi) = mid; }
        const double xi = hi;
        // h(rc): largest h, i.e. smallest admissible M, with E^F <= eps/3
        int M = 0;
        for (int m = 8; m <= 4096; m += 2) {
            if (!smooth7(m)) continue;
            if (err_grid(xi, 1.0 / m) <= third) { M = m; break; }
        }
        if (!M) continue;
        // P(rc): smallest even P with E^w <= eps/3 (window error falls with P), rounded up to the next support the
        // tensor-core gridding kernels are instantiated for when there is one (the generic kernel is several times slower)
        int P = 0;
        for (int q = 2; q <= Pmax && q <= M; q += 2)
            if (err_window(window, q, xi, 1.0 / M) <= third) { P = q; break; }
        if (!P) continue;
        for (int q = P; q <= Pmax && q <= M; q += 2)
            if (se_mma_supported(q, (int)prec)) { P = q; break; }
        const double t = model_time((double)N, rc, M, P, prec);
        if (!found || t < best.model_ms * 1e-3) {
            found = true;
            best.rc = rc * L; best.xi = xi / L; best.M = M; best.P = P;
            best.EN = err_near(xi, rc); best.EF = err_grid(xi, 1.0 / M); best.Ew = err_window(window, P, xi, 1.0 / M);
            best.s = (double)N * rc * rc * rc;
            best.model_ms = t * 1e3;
        }
    }
    if (!found) return SE_EINVAL;
    *out = best;
    return SE_OK;
}

extern "C" se_status se_plan_create_tol(se_plan **out, int64_t N, int64_t Nt, double L, double eps, se_window window,
                                        se_precision prec, se_params *chosen)
{
    if (!out) return SE_EINVAL;
    *out = nullptr;
    se_params q;
    se_status st = se_select_params(N, L, eps, window, prec, &q);
    if (st != SE_OK) return st;
    if (chosen) *chosen = q;
    se_plan_desc d{};
    d.N = N; d.Nt = Nt; d.L = L; d.xi = q.xi; d.rc = q.rc; d.M = q.M; d.P = q.P;
    d.precision = (int)prec; d.window = (int)window;
    return se_plan_create_ex(out, &d);
}
