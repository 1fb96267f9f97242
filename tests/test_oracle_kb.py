"""Pins for the Kaiser-Bessel window variant of oracle O2 (eq. (2.8)).  CPU only.

What fixes each piece, other than itself:
  se_kb_window / se_bessel_i0   scipy.special.i0 (another implementation) and the truncation of (2.8);
  kb_what (quadrature)          the closed-form transform of the Kaiser-Bessel function
                                2 a_w sinh(sqrt(beta^2 - (k a_w)^2)) / (I0(beta) sqrt(beta^2 - (k a_w)^2));
  kb_poly_coeffs + Horner in C  the exact window to the stated nu-accuracy, evaluated through se_window_1d
                                (a wrong bin, local variable or coefficient order fails by orders of magnitude);
  P2G + deconvolution table     the DFT of one spread particle equals f e^{-ik.x} w_hat(k) on resolved modes;
  G2P                           adjointness with P2G and interpolation of a resolved mode;
  the whole chain               agreement with the direct Ewald sum O1 at the accuracy P promises, P-convergence.
"""
import numpy as np
import pytest
from scipy.special import i0

import oracle
from paper_2606_19059_b200 import workloads as W


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def test_kb_window_matches_eq_2_8():
    P, L, M = 8, 1.0, 40
    kp = oracle.kb_params(L, M, P)
    assert kp["beta"] == 2.5 * P and abs(kp["aw"] - P * (L / M) / 2) < 1e-18
    r = np.linspace(-1.2 * kp["aw"], 1.2 * kp["aw"], 1001)
    w = oracle.kb_window(r, kp["beta"], kp["aw"])
    inside = np.abs(r) < kp["aw"]
    ref = i0(kp["beta"] * np.sqrt(1 - (r[inside] / kp["aw"]) ** 2)) / i0(kp["beta"])
    np.testing.assert_allclose(w[inside], ref, rtol=1e-13)
    assert np.all(w[~inside] == 0)
    assert oracle.kb_window([0.0], kp["beta"], kp["aw"])[0] == 1.0
    assert oracle.kb_window([kp["aw"]], kp["beta"], kp["aw"])[0] == 0.0                # r < a_w is strict


@pytest.mark.parametrize("P", [4, 8, 12])
def test_kb_transform_closed_form(P):
    L, M = 1.0, 48
    kp = oracle.kb_params(L, M, P)
    wh = oracle.kb_what(L, M, P)
    n = np.fft.fftfreq(M, 1.0 / M)
    kap = 2 * np.pi * n / L * kp["aw"]
    assert np.all(np.abs(kap) < kp["beta"])                     # pi P / 2 < 2.5 P: always the sinh branch
    q = np.sqrt(kp["beta"] ** 2 - kap ** 2)
    ref = 2 * kp["aw"] * np.sinh(q) / (i0(kp["beta"]) * q)
    np.testing.assert_allclose(wh, ref, rtol=1e-12)


@pytest.mark.parametrize("P", [4, 6, 8, 10, 12, 14])
def test_kb_polynomial_accuracy(P):
    """The piecewise polynomial (degree nu = min(P + 3, 13), reading S19) through the oracle's own Horner
    loop reproduces the exact window two orders below its truncation level 1/I0(beta)."""
    L, M, xi = 1.0, 64, 10.0
    h = L / M
    kp = oracle.kb_params(L, M, P)
    nu = oracle.kb_degree(P)
    assert nu == min(P + 3, 13)
    c = oracle.kb_poly_coeffs(L, M, P)
    assert c.shape == (P, nu + 1)
    rng = np.random.default_rng(P)
    worst = 0.0
    for xd in np.concatenate([rng.random(40) * L, [0.0, 3 * h, 3 * h + 1e-12, 17.5 * h]]):
        We, ie = oracle.window_1d(xd, L, xi, M, P, "kb")
        Wp, ip = oracle.window_1d(xd, L, xi, M, P, "kb_poly")
        assert np.array_equal(ie, ip)
        # the support point at exactly r = a_w (frac = 0, l = P - 1) is where (2.8) jumps to zero
        inner = np.ones(P, bool) if We[-1] != 0 else np.arange(P) < P - 1
        worst = max(worst, np.max(np.abs(We - Wp)[inner]))
    assert worst < max(1e-2 / i0(kp["beta"]), 5e-14), worst


def test_kb_dft_of_spread_particle():
    """h^3 DFT(P2G of one particle) = f e^{-ik.x} w_hat(k) on resolved modes, w_hat from kb_what:
    pins the support/anchor of the spreading against the deconvolution table of se_scale."""
    L, xi, M, P = 1.0, 10.0, 40, 12
    x = np.array([[0.3137, 0.712, 0.05]])
    f = np.array([[1.0, 0.0, 0.0]])
    wh = oracle.kb_what(L, M, P)
    n = np.fft.fftfreq(M, 1.0 / M)
    k = 2 * np.pi * n / L
    KX, KY, KZ = np.meshgrid(k, k, k, indexing="ij")
    ref = (wh[:, None, None] * wh[None, :, None] * wh[None, None, :]
           * np.exp(-1j * (KX * x[0, 0] + KY * x[0, 1] + KZ * x[0, 2])))
    low = (np.abs(KX) < 2 * np.pi * 5) & (np.abs(KY) < 2 * np.pi * 5) & (np.abs(KZ) < 2 * np.pi * 5)
    for win in ("kb", "kb_poly"):
        H = oracle.p2g(x, f, L, xi, M, P, win)
        Hh = np.fft.fftn(H[0]) * (L / M) ** 3
        # aliasing of the truncated window: relative e^{-beta} sqrt(..) ~ 1e-11 at these low modes
        assert np.max(np.abs(Hh - ref)[low]) < 1e-9 * np.abs(ref).max()
        assert np.all(H[1:] == 0)


def test_kb_adjointness_and_interpolation():
    L, xi, M, P = 1.0, 10.0, 32, 12
    c, x, f = W.scaled(2, 400)
    xw = oracle.wrap(x, L)
    Y = W.smooth_grid(11, M)
    for win in ("kb", "kb_poly"):
        H = oracle.p2g(xw, f, L, xi, M, P, win)
        uY = oracle.g2p(xw, Y, L, xi, M, P, win)
        lhs, rhs = np.sum(uY * f), (L / M) ** 3 * np.sum(Y * H)
        assert abs(lhs - rhs) < 1e-12 * abs(rhs)
    g = np.arange(M) / M
    kv = 2 * np.pi * np.array([2, -1, 3])
    Yc = np.zeros((3, M, M, M))
    Yc[1] = np.cos(kv[0] * g[:, None, None] + kv[1] * g[None, :, None] + kv[2] * g[None, None, :])
    xt = np.array([[0.1234, 0.777, 0.4321], [0.999, 0.001, 0.5]])
    wh = oracle.kb_what(L, M, P)
    u = oracle.g2p(xt, Yc, L, xi, M, P, "kb_poly")
    ref = wh[2] * wh[M - 1] * wh[3] * np.cos(xt @ kv)
    np.testing.assert_allclose(u[:, 1], ref, atol=1e-9 * abs(wh[0]) ** 3)


def test_kb_scale_mode_closed_form():
    """One mode against (2.4b)/(2.6) typed with numpy and the closed-form Kaiser-Bessel transform."""
    L, xi, M, P = 2.0, 7.0, 32, 8
    idx = np.array([[3, M - 2, 5]])
    v = np.array([[1 + 2j, -0.5 + 0.25j, 3 - 1j]])
    out = oracle.scale_modes(idx, v, L, xi, M, P, "kb_poly")[0]
    kp = oracle.kb_params(L, M, P)
    k = 2 * np.pi * np.array([3, -2, 5]) / L
    k2 = k @ k
    GF = 8 * np.pi / k2 ** 2 * (np.eye(3) * k2 - np.outer(k, k)) * np.exp(-k2 / (2 * xi) ** 2) * (1 + k2 / (2 * xi) ** 2)
    q = np.sqrt(kp["beta"] ** 2 - (k * kp["aw"]) ** 2)
    what = np.prod(2 * kp["aw"] * np.sinh(q) / (i0(kp["beta"]) * q))
    ref = (GF @ v[0]) / what ** 2 * (L / M) ** 3 / L ** 3
    np.testing.assert_allclose(out, ref, rtol=1e-12)
    # k = 0 and the Nyquist planes stay zero (readings S2, S8)
    z = oracle.scale_modes(np.array([[0, 0, 0], [M // 2, 1, 1]]), np.array([v[0], v[0]]), L, xi, M, P, "kb_poly")
    assert np.all(z == 0)


def test_kb_se_matches_direct_ewald_and_converges_with_P():
    """Config 1's split (xi = 18, rc = 0.25, M = 56) with the paper's window: the far-field error against
    the exact sum falls with P and reaches the grid's own limit; the full sum at P = 12 is a 9-digit sum."""
    c, x, f = W.make(1)
    ud = oracle.direct_ewald(x, f, c.L, c.xi)
    xw = oracle.wrap(x, c.L)
    uN_big = oracle.near_brute(xw, f, c.L, c.xi, 0.5)
    far_exact = ud - uN_big + 4 * c.xi / np.sqrt(np.pi) * f
    errs = [rel(oracle.se_far(xw, f, c.L, c.xi, c.M, P, window="kb_poly")["uF"], far_exact) for P in (4, 8, 12)]
    assert errs[0] > 30 * errs[1] > 900 * errs[2]
    assert errs[0] < 1e-3 and errs[1] < 1e-7 and errs[2] < 2e-9
    o = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, 12, window="kb_poly")
    assert rel(o["u"], ud) < 2e-9
    # exact window and polynomial window agree far below the method error
    o2 = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, 12, window="kb")
    assert rel(o["u"], o2["u"]) < 1e-11
