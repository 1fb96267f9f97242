// C-ABI of libse_b200.so (declared in include/se.h): plan management, cuFFT plumbing,
// stage sequencing.  All arithmetic of the method lives in the kernels of se_sort.cu (K1, K6),
// se_p2p.cu (K2), se_grid.cu (K3, K5), se_scale.cu (K4); the two FFT steps of Algorithm 2.1
// are cuFFT R2C / C2R with batch 3.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "se_common.cuh"

namespace {

struct Alloc {
    se_plan *p;
    bool ok = true;
    template <typename T> void get(T **dst, size_t bytes)
    {
        *dst = nullptr;
        if (!ok) return;
        void *q = nullptr;
        if (bytes == 0) bytes = 16;
        if (cudaMalloc(&q, bytes) != cudaSuccess) { ok = false; cudaGetLastError(); return; }
        p->workspace_bytes += bytes;
        *dst = (T *)q;
    }
};

void free_all(se_plan *p)
{
    if (!p) return;
    auto free_set = [](SeSet &Q) {
        void *ptrs[] = {Q.cell_of, Q.cell_start, Q.cell_cursor, Q.perm_near, Q.inv_near, Q.cell_sorted, Q.src_near, Q.xq, Q.xp,
                        Q.bin_of, Q.bin_start, Q.bin_cursor, Q.perm_grid, Q.inv_grid, Q.anchor, Q.wtab, Q.recg, Q.fs_grid};
        for (void *q : ptrs) if (q) cudaFree(q);
    };
    free_set(p->S);
    if (p->own_targets) free_set(p->T);
    void *ptrs[] = {p->uN, p->uF, p->uFpart, p->grid, p->spec, p->ktab, p->mtab, p->wcoef, p->hx, p->hf, p->hu, p->xf_tw, p->xf_xk,
                    p->f2_zpos, p->f2_ykk};
    for (void *q : ptrs) if (q) cudaFree(q);
    if (p->fft_ok & 1) cufftDestroy(p->fft_fwd);
    if (p->fft_ok & 2) cufftDestroy(p->fft_inv);
    if (p->fft2_ok & 1) cufftDestroy(p->fft2_fwd);
    if (p->fft2_ok & 2) cufftDestroy(p->fft2_inv);
    if (p->ev_ok) for (int i = 0; i <= SE_NSTAGES; ++i) cudaEventDestroy(p->ev[i]);
    if (p->side_ok) {
        cudaEventDestroy(p->ev_fork); cudaEventDestroy(p->ev_join);
        cudaEventDestroy(p->ev_p2p[0]); cudaEventDestroy(p->ev_p2p[1]);
        cudaStreamDestroy(p->side);
    }
    delete p;
}

// planes == false: the 3-D transforms; planes == true: the 2-D transforms over (y, z) of every x-plane (fused path, K4x)
se_status run_fft(se_plan *p, bool forward, cudaStream_t s, bool planes = false)
{
    if (planes && p->f2_ok) return se_launch_fft2(p, forward, s) == cudaSuccess ? SE_OK : SE_ECUDA;
    cufftHandle h = planes ? (forward ? p->fft2_fwd : p->fft2_inv) : (forward ? p->fft_fwd : p->fft_inv);
    if (cufftSetStream(h, s) != CUFFT_SUCCESS) return SE_ECUFFT;
    cufftResult r;
    if (p->precision == SE_FP64)
        r = forward ? cufftExecD2Z(h, (cufftDoubleReal *)p->grid, (cufftDoubleComplex *)p->spec)
                    : cufftExecZ2D(h, (cufftDoubleComplex *)p->spec, (cufftDoubleReal *)p->grid);
    else
        r = forward ? cufftExecR2C(h, (cufftReal *)p->grid, (cufftComplex *)p->spec)
                    : cufftExecC2R(h, (cufftComplex *)p->spec, (cufftReal *)p->grid);
    return r == CUFFT_SUCCESS ? SE_OK : SE_ECUFFT;
}

// fused == true (se_eval and its siblings on plans with xf_ok): FFT = 2-D transforms of the x-planes, SCALE = K4x (transform
// over x, K4, inverse transform over x in one kernel), IFFT = 2-D transforms back.  The staged interface keeps the 3-D
// transforms and the stand-alone K4, so that the spectrum can be read between the stages.
se_status run_stage(se_plan *p, int stage, const void *x, const void *f, void *u, cudaStream_t s, bool fused = false)
{
    cudaError_t e = cudaSuccess;
    if (fused && !p->slab) {
        if (stage == SE_STAGE_FFT) return run_fft(p, true, s, true);
        if (stage == SE_STAGE_IFFT) return run_fft(p, false, s, true);
        if (stage == SE_STAGE_SCALE) return se_launch_xfft_scale(p, s) == cudaSuccess ? SE_OK : SE_ECUDA;
    }
    switch (stage) {
    case SE_STAGE_SORT:
        if (!x || !f || (p->own_targets && !p->xt_stage)) return SE_EINVAL;
        e = se_launch_sort(p, x, f, p->xt_stage, s);
        break;
    case SE_STAGE_P2P: e = se_launch_p2p(p, s); break;
    case SE_STAGE_P2G: e = se_launch_p2g(p, s); break;
    case SE_STAGE_FFT: if (p->slab) return SE_EINVAL; return run_fft(p, true, s);
    case SE_STAGE_SCALE: if (p->slab) return SE_EINVAL; e = se_launch_scale(p, s); break;
    case SE_STAGE_IFFT: if (p->slab) return SE_EINVAL; return run_fft(p, false, s);
    case SE_STAGE_G2P: e = se_launch_g2p(p, s); break;
    case SE_STAGE_SUM:
        if ((!f && (!p->own_targets || p->nown)) || !u) return SE_EINVAL;
        e = se_launch_sum(p, f, u, s);
        break;
    default: return SE_EINVAL;
    }
    return e == cudaSuccess ? SE_OK : SE_ECUDA;
}

size_t buffer_bytes(const se_plan *p, int which, void **ptr)
{
    const SeGeom &g = p->g;
    size_t rb = p->real_bytes;
    size_t M3 = (size_t)g.Mx * g.M * g.M, nm = p->slab ? 0 : (size_t)g.M * g.M * (g.M / 2 + 1);
    const SeSet &Q = (which & SE_BUF_TARGETS) ? p->T : p->S;       // PERM / START ids: which point set
    switch (which & ~SE_BUF_TARGETS) {
    case SE_BUF_UN: *ptr = p->uN; return (size_t)p->T.n * 3 * rb;
    case SE_BUF_UF: *ptr = p->uF; return (size_t)p->T.n * 3 * rb;
    case SE_BUF_GRID: *ptr = p->grid; return 3 * M3 * rb;
    case SE_BUF_SPEC: *ptr = p->slab ? nullptr : p->spec; return 3 * nm * 2 * rb;
    case SE_BUF_PERM_NEAR: *ptr = Q.perm_near; return (size_t)Q.n * sizeof(int);
    case SE_BUF_PERM_GRID: *ptr = Q.perm_grid; return (size_t)Q.n * sizeof(int);
    case SE_BUF_CELL_START: *ptr = Q.cell_start; return ((size_t)g.ncell * g.ncell * g.ncell + 1) * sizeof(int);
    case SE_BUF_BIN_START: *ptr = Q.bin_start; return ((size_t)g.nbins_total + 1) * sizeof(int);
    default: *ptr = nullptr; return 0;
    }
}

}  // namespace

extern "C" {

const char *se_strerror(se_status s)
{
    switch (s) {
    case SE_OK: return "ok";
    case SE_EINVAL: return "invalid argument";
    case SE_ENOMEM: return "out of memory";
    case SE_ECUDA: return "CUDA error";
    case SE_ECUFFT: return "cuFFT error";
    case SE_ELIMIT: return "size beyond the fixed capacity of an entry point that allocates nothing";
    default: return "unknown status";
    }
}

se_status se_plan_create(se_plan **out, int64_t N, double L, double xi, double rc, int M, int P,
                         se_precision prec)
{
    se_plan_desc d{};
    d.N = N; d.Nt = 0; d.L = L; d.xi = xi; d.rc = rc; d.M = M; d.P = P;
    d.precision = (int)prec; d.window = SE_WINDOW_GAUSSIAN; d.Mx = 0; d.px0 = 0; d.Nown = 0;
    return se_plan_create_ex(out, &d);
}

se_status se_plan_create_ex(se_plan **out, const se_plan_desc *d)
{
    if (!out) return SE_EINVAL;
    *out = nullptr;
    if (!d) return SE_EINVAL;
    const int64_t N = d->N, Nt = d->Nt;
    const double L = d->L, xi = d->xi, rc = d->rc;
    const int M = d->M, P = d->P, prec = d->precision, window = d->window;
    const int Mx = d->Mx > 0 ? d->Mx : M, px0 = d->Mx > 0 ? d->px0 : 0;
    const bool slab = d->Mx > 0;
    const int64_t Nown = d->Nown;
    if (Nown != 0 && (!slab || Nown != Nt || Nown > N)) return SE_EINVAL;
    if (!(N >= 1) || N >= ((int64_t)1 << 31) || Nt < 0 || Nt >= ((int64_t)1 << 31) || !(L > 0) || !(xi > 0) || !(rc > 0) ||
        !std::isfinite(L) || !std::isfinite(xi) || !std::isfinite(rc))
        return SE_EINVAL;
    if (M < 2 || (M & 1) || M > 4096 || P < 2 || (P & 1) || P > SE_PMAX || P > M) return SE_EINVAL;
    if (prec != SE_FP64 && prec != SE_FP32) return SE_EINVAL;
    if (window != SE_WINDOW_GAUSSIAN && window != SE_WINDOW_KAISER_BESSEL) return SE_EINVAL;
    if (window == SE_WINDOW_KAISER_BESSEL && P > 16) return SE_EINVAL;
    if (slab && (Mx > M || Mx < se_mma_ring(P) || Mx < P || px0 < 0 || px0 >= M || !se_mma_supported(P, prec))) return SE_EINVAL;
    double ncd = std::floor(L / rc);
    if (!(ncd >= 3)) return SE_EINVAL;
    // near cells: floor(L / rc) per dimension (reading S7), but no more than ~8 cells per point (wider cells stay
    // correct -- the 27-cell stencil only needs a width >= rc -- and keep the per-evaluation histogram and scan O(N))
    const double ncap = std::max(3.0, std::ceil(std::cbrt(8.0 * (double)std::max(N, Nt))));
    int ncell = (int)std::min(std::min(ncd, ncap), 1024.0);

    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return SE_ECUDA; }

    se_plan *p = new (std::nothrow) se_plan();
    if (!p) return SE_ENOMEM;
    std::memset(p, 0, sizeof(*p));
    p->device = dev;
    p->precision = prec;
    p->real_bytes = prec == SE_FP64 ? 8 : 4;
    p->own_targets = Nt > 0;
    p->slab = slab ? 1 : 0;
    p->nown = Nown;
    SeGeom &g = p->g;
    g.N = N; g.M = M; g.P = P; g.L = L; g.xi = xi; g.rc = rc;
    g.Mx = Mx; g.px0 = px0;
    g.window = window;
    g.nu = window == SE_WINDOW_KAISER_BESSEL ? se_kb_degree(P) : 0;
    g.ncell = ncell;
    g.nbin = (M + SE_BIN - 1) / SE_BIN;
    g.nbins_total = g.nbin * g.nbin * g.nbin;
    g.grid_mode = 0; g.nchunk = 1; g.nchunk_g2p = 1;
    {
        // Gridding kernels: FP64 tensor-core sweep where it applies, else the generic tile kernel.
        // SE_GRID_MODE = tile forces the generic kernel (tests and experiments).
        const char *force = std::getenv("SE_GRID_MODE");
        const bool want_tile = force && std::strcmp(force, "tile") == 0;
        const int zb = (M + SE_MMA_ZBIN - 1) / SE_MMA_ZBIN;
        // the sort key has M * zb * M bins: beyond ~64 bins per point the per-evaluation scan would dominate
        const double nbins_mma = (double)Mx * zb * M;
        if (se_mma_supported(P, prec) && se_mma_ring(P) <= Mx && nbins_mma < 5.0e8 &&
            (slab || (nbins_mma <= 64.0 * (double)std::max(N, Nt) + 4.0e6 && !want_tile))) {
            g.grid_mode = 2;
            g.ring = se_mma_ring(P);
            g.ring_g = se_mma_ring_g(P);
            g.nbin = zb;
            g.nbins_total = Mx * zb * M;
            const int BY = 4 * SE_MMA_NWY, BZ = 4 * SE_MMA_NWZ;
            const int tiles = ((M + BY - 1) / BY) * ((M + BZ - 1) / BZ);
            // One block per SM, so the grid should fill whole waves of one block per SM (148).  A P2G chunk re-spreads P - 1
            // warm-up planes (none when a single chunk covers the axis), a G2P chunk only re-loads them: pick the
            // chunk counts that minimise (wave quantisation) x (warm-up overhead).
            int nsm = 148;
            if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) {
                cudaGetLastError();
                nsm = 148;
            }
            auto pick = [&](int nmax, bool spread) {
                int best = 1;
                double bc = 1e30;
                for (int n = 1; n <= std::max(1, nmax); ++n) {
                    const double w = (double)tiles * n / nsm;
                    double cost = std::ceil(w) / w;
                    const double cl = (double)Mx / n;
                    if (spread) cost *= n == 1 ? 1.0 : (cl + P - 1) / cl;
                    else cost *= 1.0 + 0.15 * (P - 1) / cl;
                    if (cost < bc - 1e-9) { bc = cost; best = n; }
                }
                return best;
            };
            int nch = pick(Mx / (4 * P), true);
            int nchg = pick(2 * Mx / P, false);                  // G2P chunks may be as short as P / 2 planes
            const char *e = std::getenv("SE_NCHUNK");
            if (e && std::atoi(e) > 0) nch = std::min(std::atoi(e), Mx);
            e = std::getenv("SE_NCHUNK_G2P");
            if (e && std::atoi(e) > 0) nchg = std::min(std::atoi(e), Mx);
            g.nchunk = std::max(nch, 1);
            g.nchunk_g2p = std::max(nchg, 1);
            // P2G with whole sweeps: if the last wave is partly filled, split only its tiles along x (each piece pays
            // P - 1 warm-up planes) when that shortens the tail
            g.nfull = tiles; g.nsplit = 1;
            const int R = tiles % nsm;
            if (g.nchunk == 1 && R > 0 && tiles > nsm && !std::getenv("SE_NCHUNK")) {
                double best = 0.95;
                for (int k = 2; k <= 4 && Mx / k >= P; ++k) {
                    const double cost = std::ceil((double)R * k / nsm) * ((double)Mx / k + P - 1) / Mx;
                    if (cost < best) { best = cost; g.nsplit = k; g.nfull = tiles - R; }
                }
            }
        }
    }
    g.rel_coords = prec == SE_FP32;
    g.h = L / M;
    g.wcell = L / ncell;
    if (window == SE_WINDOW_GAUSSIAN) {
        double m = 0.95 * std::sqrt(SE_PI * P);             // reading S4
        g.eta = (P * g.h * xi / m) * (P * g.h * xi / m);
        double a = 2.0 * xi * xi / g.eta;
        g.beta = a * g.h * g.h;
        g.cw = std::pow(a / SE_PI, 1.5);
    } else {                                                // Kaiser-Bessel: w0(0) = 1, no prefactor (eq. (2.8))
        g.eta = 0.0; g.beta = 0.0; g.cw = 1.0;
    }

    size_t rb = p->real_bytes;
    size_t nc3 = (size_t)ncell * ncell * ncell, nb3 = (size_t)g.nbins_total + 1;       // + the bin of the sources that are not spread
    if (slab && g.grid_mode != 2) { delete p; return SE_EINVAL; }
    size_t M3 = (size_t)Mx * M * M, nm = slab ? 0 : (size_t)M * M * (M / 2 + 1);
    size_t scan_tiles = (std::max(nc3, nb3) + 2047) / 2048 + 1;

    Alloc A{p};
    auto alloc_set = [&](SeSet &Q, int64_t n, bool spread, bool gather) {
        Q.n = n;
        A.get(&Q.cell_of, n * sizeof(int));
        A.get(&Q.cell_start, (nc3 + 1 + scan_tiles) * sizeof(int));
        A.get(&Q.cell_cursor, (nc3 + 1) * sizeof(int));
        A.get(&Q.perm_near, n * sizeof(int));
        A.get(&Q.inv_near, n * sizeof(int));
        A.get(&Q.cell_sorted, n * sizeof(int));
        A.get(&Q.src_near, n * 6 * rb);
        A.get(&Q.xq, n * sizeof(float4));
        A.get(&Q.xp, 2 * (size_t)SE_XP_LEN(n) * 16);
        A.get(&Q.bin_of, n * sizeof(int));
        A.get(&Q.bin_start, (nb3 + 1 + scan_tiles) * sizeof(int));
        A.get(&Q.bin_cursor, (nb3 + 1) * sizeof(int));
        A.get(&Q.perm_grid, n * sizeof(int));
        A.get(&Q.inv_grid, n * sizeof(int));
        A.get(&Q.anchor, n * sizeof(short4));
        if (g.grid_mode == 2) {
            if (spread) A.get(&Q.wtab, (size_t)n * SE_MMA_RECS(g.ring) * 8);
            if (gather) A.get(&Q.recg, (size_t)n * SE_MMA_RECG(g.ring_g) * 8);
        } else
            A.get(&Q.wtab, (size_t)n * 3 * P * rb);
        A.get(&Q.fs_grid, std::max((size_t)n * 3 * rb, (size_t)n * sizeof(int)));
    };
    alloc_set(p->S, N, true, !p->own_targets);
    if (p->own_targets) alloc_set(p->T, Nt, false, true);
    else p->T = p->S;
    const int64_t NT = p->T.n;
    A.get(&p->uN, NT * 3 * rb);
    A.get(&p->uF, NT * 3 * rb);
    if (g.grid_mode == 2) A.get(&p->uFpart, (size_t)NT * se_mma_slots(P) * 3 * 8);
    A.get(&p->grid, 3 * M3 * rb);
    A.get(&p->spec, 3 * nm * 2 * rb);
    A.get(&p->ktab, 2 * (size_t)M * rb);
    if (!p->own_targets) {                                  // staging of se_eval_host
        A.get(&p->hx, N * 3 * rb); A.get(&p->hf, N * 3 * rb); A.get(&p->hu, N * 3 * rb);
    }
    if (!A.ok) { free_all(p); return SE_ENOMEM; }

    // cuFFT: batch of 3 out-of-place 3-D transforms, contiguous, z fastest, halved axis last
    int n[3] = {M, M, M};
    cufftType tf = prec == SE_FP64 ? CUFFT_D2Z : CUFFT_R2C, ti = prec == SE_FP64 ? CUFFT_Z2D : CUFFT_C2R;
    size_t wsz = 0;
    cufftResult r = slab ? CUFFT_SUCCESS : cufftPlanMany(&p->fft_fwd, 3, n, nullptr, 1, (int)0, nullptr, 1, (int)0, tf, 3);
    if (slab) {
        // a slab plan transforms nothing: the assembled grid belongs to a whole-grid plan
    } else if (r == CUFFT_SUCCESS) {
        p->fft_ok |= 1;
        if (cufftGetSize(p->fft_fwd, &wsz) == CUFFT_SUCCESS) p->fft_work_bytes += wsz;
        r = cufftPlanMany(&p->fft_inv, 3, n, nullptr, 1, (int)0, nullptr, 1, (int)0, ti, 3);
    }
    if (slab) {
    } else if (r == CUFFT_SUCCESS) {
        p->fft_ok |= 2;
        if (cufftGetSize(p->fft_inv, &wsz) == CUFFT_SUCCESS) p->fft_work_bytes += wsz;
    } else {
        se_status st = (r == CUFFT_ALLOC_FAILED) ? SE_ENOMEM : SE_ECUFFT;
        free_all(p);
        return st;
    }
    if (se_build_xfft(p) != cudaSuccess) {
        cudaGetLastError();
        free_all(p);
        return SE_ECUDA;
    }
    if (p->xf_ok) {
        // fused path: batch of 3 M out-of-place 2-D transforms over (y, z), one per x-plane and component
        int n2[2] = {M, M};
        r = cufftPlanMany(&p->fft2_fwd, 2, n2, nullptr, 1, (int)0, nullptr, 1, (int)0, tf, 3 * M);
        if (r == CUFFT_SUCCESS) {
            p->fft2_ok |= 1;
            if (cufftGetSize(p->fft2_fwd, &wsz) == CUFFT_SUCCESS) p->fft_work_bytes += wsz;
            r = cufftPlanMany(&p->fft2_inv, 2, n2, nullptr, 1, (int)0, nullptr, 1, (int)0, ti, 3 * M);
        }
        if (r == CUFFT_SUCCESS) {
            p->fft2_ok |= 2;
            if (cufftGetSize(p->fft2_inv, &wsz) == CUFFT_SUCCESS) p->fft_work_bytes += wsz;
        } else {
            se_status st = (r == CUFFT_ALLOC_FAILED) ? SE_ENOMEM : SE_ECUFFT;
            free_all(p);
            return st;
        }
    }
    p->workspace_bytes += p->fft_work_bytes;

    if (se_build_ktab(p) != cudaSuccess || se_build_wcoef(p) != cudaSuccess || se_build_mtab(p) != cudaSuccess ||
        se_prepare_grid(p) != cudaSuccess || se_tune_xfft(p) != cudaSuccess) {
        cudaGetLastError();
        free_all(p);
        return SE_ECUDA;
    }
    for (int i = 0; i <= SE_NSTAGES; ++i)
        if (cudaEventCreate(&p->ev[i]) != cudaSuccess) { free_all(p); return SE_ECUDA; }
    p->ev_ok = 1;
    {
        // side stream for K2 at the lowest priority: the grid chain on the caller's stream gets the SMs first
        int lo = 0, hi = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hi);
        const char *e = std::getenv("SE_OVERLAP");
        p->overlap = e && std::atoi(e) != 0;             // off by default: measured gain <= 0.5 %
        if (cudaStreamCreateWithPriority(&p->side, cudaStreamNonBlocking, lo) != cudaSuccess ||
            cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreate(&p->ev_p2p[0]) != cudaSuccess || cudaEventCreate(&p->ev_p2p[1]) != cudaSuccess) {
            cudaGetLastError();
            free_all(p);
            return SE_ECUDA;
        }
        p->side_ok = 1;
    }
    *out = p;
    return SE_OK;
}

// every call on a plan must be made with the plan's device current
static bool on_device(const se_plan *p)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return false; }
    return dev == p->device;
}

se_status se_plan_destroy(se_plan *p)
{
    if (!p) return SE_OK;
    if (!on_device(p)) return SE_EINVAL;
    cudaDeviceSynchronize();
    free_all(p);
    return SE_OK;
}

se_status se_plan_info(const se_plan *p, se_info *o)
{
    if (!p || !o) return SE_EINVAL;
    const SeGeom &g = p->g;
    o->N = p->S.n; o->M = g.M; o->P = g.P; o->precision = p->precision;
    o->L = g.L; o->xi = g.xi; o->rc = g.rc; o->h = g.h;
    o->m = g.window == SE_WINDOW_GAUSSIAN ? 0.95 * std::sqrt(SE_PI * g.P) : 0.0;
    o->eta = g.eta;
    o->a = g.beta / (g.h * g.h);
    o->Nt = p->own_targets ? p->T.n : 0;
    o->window = g.window; o->nu = g.nu;
    o->kb_beta = g.window == SE_WINDOW_KAISER_BESSEL ? 2.5 * g.P : 0.0;
    o->cw = g.cw;
    o->ncell = g.ncell; o->nbin = g.nbin;
    o->grid_mode = g.grid_mode; o->nbins_total = g.nbins_total; o->nchunk = g.nchunk;
    o->nmodes = (int64_t)g.M * g.M * (g.M / 2 + 1);
    o->Mx = g.Mx; o->px0 = g.px0;
    o->fft_fused = p->xf_ok;
    o->fft_threads = p->xf_ok ? p->xf_threads : 0;
    o->fft_planes_own = p->xf_ok && p->f2_ok;
    o->workspace_bytes = p->workspace_bytes;
    return SE_OK;
}

static se_status run_all(se_plan *p, const void *x, const void *f, void *u, void *stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    p->launches = 0;
    p->ev_recorded = 0;
    const bool prof = p->profiling != 0;
    const bool fork = p->overlap != 0;
    const bool fused = p->xf_ok != 0;
    if (prof && cudaEventRecord(p->ev[0], s) != cudaSuccess) return SE_ECUDA;
    for (int st = 0; st < SE_NSTAGES; ++st) {
        if (fork && st == SE_STAGE_P2P) {
            // deferred: launched on the side stream once K3 has been queued (below)
        } else if (fork && st == SE_STAGE_SUM) {
            if (cudaStreamWaitEvent(s, p->ev_join, 0) != cudaSuccess) return SE_ECUDA;
            se_status r = run_stage(p, st, x, f, u, s, fused);
            if (r != SE_OK) return r;
        } else {
            se_status r = run_stage(p, st, x, f, u, s, fused);
            if (r != SE_OK) return r;
        }
        if (fork && st == SE_STAGE_P2G) {
            if (cudaEventRecord(p->ev_fork, s) != cudaSuccess) return SE_ECUDA;
            if (cudaStreamWaitEvent(p->side, p->ev_fork, 0) != cudaSuccess) return SE_ECUDA;
            if (prof && cudaEventRecord(p->ev_p2p[0], p->side) != cudaSuccess) return SE_ECUDA;
            se_status r = run_stage(p, SE_STAGE_P2P, x, f, u, p->side);
            if (r != SE_OK) return r;
            if (prof && cudaEventRecord(p->ev_p2p[1], p->side) != cudaSuccess) return SE_ECUDA;
            if (cudaEventRecord(p->ev_join, p->side) != cudaSuccess) return SE_ECUDA;
        }
        if (prof && cudaEventRecord(p->ev[st + 1], s) != cudaSuccess) return SE_ECUDA;
    }
    if (prof) p->ev_recorded = 1;
    return SE_OK;
}

se_status se_eval(se_plan *p, const void *x, const void *f, void *u, void *stream)
{
    if (!p || !x || !f || !u || p->own_targets || p->slab || !on_device(p)) return SE_EINVAL;
    return run_all(p, x, f, u, stream);
}

se_status se_eval_targets(se_plan *p, const void *xs, const void *f, const void *xt, void *ut, void *stream)
{
    if (!p || !xs || !f || !xt || !ut || !p->own_targets || p->slab || !on_device(p)) return SE_EINVAL;
    p->xt_stage = xt;
    return run_all(p, xs, f, ut, stream);
}

se_status se_set_targets(se_plan *p, const void *xt)
{
    if (!p || !xt || !p->own_targets) return SE_EINVAL;
    p->xt_stage = xt;
    return SE_OK;
}

se_status se_eval_host(se_plan *p, const void *xh, const void *fh, void *uh, void *stream)
{
    if (!p || !xh || !fh || !uh || p->own_targets || !on_device(p)) return SE_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    size_t bytes = (size_t)p->S.n * 3 * p->real_bytes;
    if (cudaMemcpyAsync(p->hx, xh, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) return SE_ECUDA;
    if (cudaMemcpyAsync(p->hf, fh, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) return SE_ECUDA;
    se_status r = se_eval(p, p->hx, p->hf, p->hu, stream);
    if (r != SE_OK) return r;
    if (cudaMemcpyAsync(uh, p->hu, bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess) return SE_ECUDA;
    return SE_OK;
}

se_status se_eval_stage(se_plan *p, int stage, const void *x, const void *f, void *u, void *stream)
{
    if (!p || !on_device(p)) return SE_EINVAL;
    return run_stage(p, stage, x, f, u, (cudaStream_t)stream);
}

se_status se_buffer_read(se_plan *p, int which, void *dst, size_t bytes, size_t *size_out, void *stream)
{
    if (!p || !on_device(p)) return SE_EINVAL;
    void *src = nullptr;
    size_t n = buffer_bytes(p, which, &src);
    if (!src) return SE_EINVAL;
    if (size_out) *size_out = n;
    if (!dst) return SE_OK;
    if (bytes != n) return SE_EINVAL;
    return cudaMemcpyAsync(dst, src, n, cudaMemcpyDeviceToDevice, (cudaStream_t)stream) == cudaSuccess ? SE_OK
                                                                                                         : SE_ECUDA;
}

se_status se_buffer_write(se_plan *p, int which, const void *srcv, size_t bytes, void *stream)
{
    if (!p || !srcv || !on_device(p)) return SE_EINVAL;
    void *dst = nullptr;
    size_t n = buffer_bytes(p, which, &dst);
    if (!dst || bytes != n) return SE_EINVAL;
    return cudaMemcpyAsync(dst, srcv, n, cudaMemcpyDeviceToDevice, (cudaStream_t)stream) == cudaSuccess ? SE_OK
                                                                                                          : SE_ECUDA;
}

se_status se_set_profiling(se_plan *p, int on)
{
    if (!p) return SE_EINVAL;
    p->profiling = on != 0;
    return SE_OK;
}

se_status se_stage_ms(se_plan *p, float ms[SE_NSTAGES])
{
    if (!p || !ms) return SE_EINVAL;
    if (!p->ev_recorded) return SE_EINVAL;
    if (cudaEventSynchronize(p->ev[SE_NSTAGES]) != cudaSuccess) return SE_ECUDA;
    for (int st = 0; st < SE_NSTAGES; ++st)
        if (cudaEventElapsedTime(&ms[st], p->ev[st], p->ev[st + 1]) != cudaSuccess) return SE_ECUDA;
    if (p->overlap) {                                   // K2 ran on the side stream, concurrently with stages 3..6
        if (cudaEventSynchronize(p->ev_p2p[1]) != cudaSuccess) return SE_ECUDA;
        if (cudaEventElapsedTime(&ms[SE_STAGE_P2P], p->ev_p2p[0], p->ev_p2p[1]) != cudaSuccess) return SE_ECUDA;
    }
    return SE_OK;
}

se_status se_last_launch_count(const se_plan *p, int *count)
{
    if (!p || !count) return SE_EINVAL;
    *count = p->launches;
    return SE_OK;
}

}  // extern "C"
