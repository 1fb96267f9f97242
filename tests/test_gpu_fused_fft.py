"""GPU parity of the fused x-transform + K4 path (csrc/se_scale.cu K4x; se.h "FUSED"): se_eval on plans whose M is
7-smooth runs cuFFT 2-D transforms of the x-planes around ONE kernel that transforms over x, applies K4 (eq. (2.6),
PAPER.md:88) and transforms back.  The stage-by-stage parity tests go through the 3-D transforms of se_eval_stage, so
here H~ (the grid after the inverse transform) of a whole se_eval is compared with the oracle's, element
by element, for grid sizes that exercise every radix of the kernel (16, 9, 8, 7, 5, 4, 3, 2), a ragged last kz-tile,
both precisions and both windows; and with the unfused path of the same library (SE_FFT_MODE=3d)."""
import numpy as np
import pytest

import oracle
from paper_2606_19059_b200 import workloads as W
from gpu_util import gate
from test_gpu_parity import TOL

pytestmark = pytest.mark.gpu


def eval_Ht(c, x, f, window="gaussian"):
    import torch
    import paper_2606_19059_b200 as se
    dt = torch.float32 if c.precision == "fp32" else torch.float64
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, c.precision, window=window) as plan:
        fused = plan.info().fft_fused
        u = plan.eval(torch.as_tensor(x, dtype=dt, device="cuda"), torch.as_tensor(f, dtype=dt, device="cuda"))
        Ht = plan.read(se.SE_BUF_GRID).cpu().numpy()
        return fused, Ht, u.cpu().numpy()


# radices: 56 = 8 7, 60 = 5 4 3, 72 = 9 8, 80 = 16 5, 98 = 7 7 2, 100 = 5 5 4, 108 = 9 4 3, 144 = 16 9, 162 = 9 9 2
@pytest.mark.parametrize("M", [56, 60, 72, 80, 98, 100, 108, 144, 162])
def test_fused_path_fp64(M):
    from dataclasses import replace
    rng = np.random.default_rng(770 + M)
    N, P = 1500, 16
    xi = 0.8 * 0.95 * np.sqrt(np.pi * P) * M / P
    c = replace(W.CONFIGS[1], N=N, M=M, P=P, xi=xi, rc=min(0.3, 4.5 / xi), label=f"fused M={M}")
    x = rng.random((N, 3)); f = rng.standard_normal((N, 3))
    o = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P, keep=True)
    fused, Ht, u = eval_Ht(c, x, f)
    assert fused == 1
    e = gate("Ht", Ht, o["Ht"], TOL["fp64"]["Ht"])
    gate("u", u, o["u"], TOL["fp64"]["u"])
    print(f"M={M}: Ht rel-L2 {e[0]:.2e} max-abs {e[1]:.2e}")


@pytest.mark.parametrize("M,window,P", [(64, "gaussian", 12), (90, "gaussian", 12), (120, "kb", 8), (126, "gaussian", 10)])
def test_fused_path_fp32(M, window, P):
    from dataclasses import replace
    rng = np.random.default_rng(880 + M)
    N = 2000
    xi = 0.8 * 0.95 * np.sqrt(np.pi * P) * M / P
    c = replace(W.CONFIGS[4], N=N, M=M, P=P, xi=xi, rc=min(0.3, 3.2 / xi), window=window, label=f"fused fp32 M={M}")
    x = rng.random((N, 3)).astype(np.float32); f = rng.standard_normal((N, 3)).astype(np.float32)
    o = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P, keep=True, window="kb_poly" if window == "kb" else window)
    fused, Ht, u = eval_Ht(c, x, f, window)
    assert fused == 1
    gate("Ht", Ht, o["Ht"], TOL["fp32"]["Ht"])
    gate("u", u, o["u"], TOL["fp32"]["u"])


def test_kb_window_fused_fp64():
    from dataclasses import replace
    rng = np.random.default_rng(991)
    N, M, P = 3000, 96, 12
    c = replace(W.CONFIGS[1], N=N, M=M, P=P, xi=20.0, rc=0.2, window="kb", label="fused kb")
    x = rng.random((N, 3)); f = rng.standard_normal((N, 3))
    o = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P, keep=True, window="kb_poly")
    fused, Ht, u = eval_Ht(c, x, f, "kb")
    assert fused == 1
    gate("Ht", Ht, o["Ht"], TOL["fp64"]["Ht"])
    gate("u", u, o["u"], TOL["fp64"]["u"])


def test_own_and_cufft_plane_transforms_agree(monkeypatch):
    """The library's own 2-D transforms of the x-planes (real-to-complex over z, digit-reversed pass over y) against cuFFT's in
    the same fused path, fp64 and fp32, on a grid whose M / 2 needs three radices (M = 90: 45 = 9 x 5; M = 112: 56 = 8 x 7)."""
    import paper_2606_19059_b200 as se
    from dataclasses import replace
    for base, M, tol in ((3, 90, 1e-14), (3, 112, 1e-14), (4, 96, 2e-6)):
        c, x, f = W.scaled(base, 8000)
        c = replace(c, M=M, P=8 if base == 4 else 12)
        with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, c.precision) as plan:
            assert plan.info().fft_planes_own == 1
        _, Ht1, u1 = eval_Ht(c, x, f)
        monkeypatch.setenv("SE_FFT_MODE", "cufft2d")
        with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, c.precision) as plan:
            assert plan.info().fft_planes_own == 0 and plan.info().fft_fused == 1
        _, Ht0, u0 = eval_Ht(c, x, f)
        monkeypatch.delenv("SE_FFT_MODE")
        gate(f"Ht own vs cuFFT planes, M = {M}", Ht1, Ht0, tol)
        gate(f"u own vs cuFFT planes, M = {M}", u1, u0, tol)


@pytest.mark.parametrize("prec,tol", [("fp64", 2e-14), ("fp32", 3e-6)])
def test_fused_path_every_smooth_grid_size_up_to_130(prec, tol, monkeypatch):
    """Every even grid size without a prime factor above 7 from 8 to 130 (all radix orders of the transforms over x, y and the
    half-length transform over z, ragged last blocks of rows and columns): u of se_eval on the fused path with the library's own
    plane transforms against the same library on cuFFT's 3-D transforms.  (Against the oracle: the tests above.)"""
    import torch
    import paper_2606_19059_b200 as se

    def smooth7(n):
        for q in (2, 3, 5, 7):
            while n % q == 0:
                n //= q
        return n == 1

    rng = np.random.default_rng(5)
    N, P = 1500, 8
    dt = torch.float64 if prec == "fp64" else torch.float32
    xd = torch.as_tensor(rng.random((N, 3)), dtype=dt).cuda()
    fd = torch.as_tensor(rng.standard_normal((N, 3)), dtype=dt).cuda()
    sizes = [m for m in range(8, 131, 2) if smooth7(m)]
    assert len(sizes) > 30
    for M in sizes:
        xi = 0.8 * 0.95 * np.sqrt(np.pi * P) * M / P
        rc = min(0.3, 3.2 / xi)
        u = {}
        for mode in ("own", "3d"):
            if mode == "3d":
                monkeypatch.setenv("SE_FFT_MODE", "3d")
            with se.Plan(N, 1.0, xi, rc, M, P, prec) as plan:
                i = plan.info()
                assert (i.fft_fused, i.fft_planes_own) == ((1, 1) if mode == "own" else (0, 0)), (M, mode)
                u[mode] = plan.eval(xd, fd).double().cpu().numpy()
            monkeypatch.delenv("SE_FFT_MODE", raising=False)
        gate(f"u fused vs 3-D, M = {M}", u["own"], u["3d"], tol)


def test_fused_and_3d_paths_agree_and_fall_back(monkeypatch):
    """Same plan parameters through both paths: H~ agrees to rounding; a grid size with a prime factor above 7 (M = 52) and
    SE_FFT_MODE=3d take the 3-D transforms."""
    c, x, f = W.scaled(3, 20000)
    fused, Ht1, u1 = eval_Ht(c, x, f)
    assert fused == 1
    monkeypatch.setenv("SE_FFT_MODE", "3d")
    fused, Ht0, u0 = eval_Ht(c, x, f)
    assert fused == 0
    gate("Ht fused vs 3-D", Ht1, Ht0, 1e-14)
    gate("u fused vs 3-D", u1, u0, 1e-14)
    monkeypatch.delenv("SE_FFT_MODE")
    from dataclasses import replace
    c2 = replace(c, M=52, P=8)
    fused, _, u = eval_Ht(c2, x, f)
    assert fused == 0
