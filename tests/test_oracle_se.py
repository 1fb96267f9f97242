"""Pins for oracle O2 (spectral Ewald, oracle/se_oracle.c + numpy.fft).  CPU only.

The decisive pin is agreement with O1 (a different algorithm: no grid, no window, no
FFT) to the accuracy the parameters promise; the others isolate individual stages.
"""
import numpy as np
import pytest

import oracle
from paper_2606_19059_b200 import workloads as W


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.fixture(scope="module")
def cfg1():
    c, x, f = W.make(1)
    o = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P, keep=True)
    return c, x, f, o


@pytest.fixture(scope="module")
def cfg1_direct(cfg1):
    c, x, f, _ = cfg1
    return oracle.direct_ewald(x, f, c.L, c.xi)


def test_params_closed_form():
    """Reading S4: m = 0.95 sqrt(pi P), eta = (P h xi/m)^2, a = 2 xi^2/eta, c_w = (a/pi)^1.5;
    then a (P h/2)^2 = m^2/2 independent of xi, h (window truncated at e^{-m^2/2})."""
    p = oracle.params(1.0, 18.0, 56, 24)
    assert abs(p["h"] - 1 / 56) < 1e-17
    assert abs(p["a"] * (24 * p["h"] / 2) ** 2 - p["m"] ** 2 / 2) < 1e-12
    assert abs(p["m"] - 0.95 * np.sqrt(np.pi * 24)) < 1e-14
    # eta = 0.8745 for config 1, 1.0370 for config 3
    assert abs(p["eta"] - 0.8745) < 5e-5
    assert abs(oracle.params(1.0, 126.0, 360, 24)["eta"] - 1.0370) < 1e-4


def test_se_matches_direct_ewald_cfg1(cfg1, cfg1_direct):
    """BASELINE config 1: 'target rel err 1e-9 vs direct Ewald'."""
    _, _, _, o = cfg1
    assert rel(o["u"], cfg1_direct) < 1e-9


def test_far_error_converges_with_P(cfg1, cfg1_direct):
    """Window error falls with P (S4): far-field-only error vs O1 minus exact near sum."""
    c, x, f, o = cfg1
    xw = o["xw"]
    # exact far part = direct - (untruncated near) - self; approximate the untruncated near sum by rc=0.5
    uN_big = oracle.near_brute(xw, f, c.L, c.xi, 0.5)
    far_exact = cfg1_direct - uN_big + 4 * c.xi / np.sqrt(np.pi) * f
    errs = []
    for P in (8, 12, 16, 24):
        errs.append(rel(oracle.se_far(xw, f, c.L, c.xi, c.M, P)["uF"], far_exact))
    assert errs[0] > errs[1] > errs[2] > errs[3]
    assert errs[3] < 3e-10 and errs[1] < 1e-6 and errs[0] > 1e-6


def test_near_cells_equals_brute():
    c, x, f = W.scaled(2, 3000)
    xw = oracle.wrap(x, c.L)
    a = oracle.near_cells(xw, f, c.L, c.xi, c.rc)
    b = oracle.near_brute(xw, f, c.L, c.xi, c.rc)
    assert rel(a, b) < 1e-14
    sel = np.array([0, 17, 2999])
    np.testing.assert_allclose(oracle.near_brute(xw, f, c.L, c.xi, c.rc, targets=sel), b[sel], rtol=1e-15)


def test_near_pair_closed_form():
    """Two particles: u^N_1 = C1 f + C2 r (r.f) with C1, C2 written from (2.3) via scipy's erfc."""
    from scipy.special import erfc
    xi, L = 7.0, 1.0
    r = np.array([0.03, -0.05, 0.02])
    x = np.array([[0.5, 0.5, 0.5] + r, [0.5, 0.5, 0.5]])
    f = np.array([[0.0, 0, 0], [0.3, -1.2, 0.8]])
    u = oracle.near_brute(x, f, L, xi, 0.3)
    rn = np.linalg.norm(r)
    G = np.eye(3) / rn + np.outer(r, r) / rn ** 3
    e = np.exp(-xi ** 2 * rn ** 2)
    GN = G * (erfc(xi * rn) + rn * 2 * xi * e / np.sqrt(np.pi)) - np.eye(3) * 4 * xi * e / np.sqrt(np.pi)  # (2.3)
    np.testing.assert_allclose(u[0], GN @ f[1], rtol=1e-13)
    # cutoff: beyond rc nothing
    assert np.all(oracle.near_brute(x, f, L, xi, 0.9 * rn) == 0)


def test_near_periodic_image():
    """A pair split across the periodic boundary interacts through the image (2.2)."""
    xi, L, rc = 9.0, 1.0, 0.2
    f = np.array([[0.0, 0, 0], [1.0, 2.0, 3.0]])
    xa = np.array([[0.02, 0.5, 0.5], [0.97, 0.5, 0.5]])
    xb = np.array([[0.52, 0.5, 0.5], [0.47, 0.5, 0.5]])
    np.testing.assert_allclose(oracle.near_brute(xa, f, L, xi, rc), oracle.near_brute(xb, f, L, xi, rc), rtol=1e-12)
    assert np.linalg.norm(oracle.near_brute(xa, f, L, xi, rc)[0]) > 0


def test_window_normalisation_and_mass(cfg1):
    """h^3 sum_g H_c = sum_n f_c (the Gaussian integrates to 1; S11) -- use non-zero-mean f."""
    c, x, f, o = cfg1
    g = f + np.array([1.0, -2.0, 0.5])
    H = oracle.p2g(o["xw"], g, c.L, c.xi, c.M, c.P)
    h = c.L / c.M
    np.testing.assert_allclose(h ** 3 * H.sum(axis=(1, 2, 3)), g.sum(0), rtol=1e-12)


def test_window_fourier_transform():
    """DFT of one spread particle = f e^{-ik.x} w_hat(k), w_hat = e^{-eta k^2/8 xi^2} (S4):
    pins the relation between the spreading width `a` and the deconvolution in se_scale."""
    L, xi, M, P = 1.0, 10.0, 32, 24
    p = oracle.params(L, xi, M, P)
    x = np.array([[0.3137, 0.712, 0.05]])
    f = np.array([[1.0, 0.0, 0.0]])
    H = oracle.p2g(x, f, L, xi, M, P)
    Hh = np.fft.fftn(H[0]) * (L / M) ** 3
    n = np.fft.fftfreq(M, 1.0 / M)
    k = 2 * np.pi * n / L
    KX, KY, KZ = np.meshgrid(k, k, k, indexing="ij")
    k2 = KX ** 2 + KY ** 2 + KZ ** 2
    ref = np.exp(-p["eta"] * k2 / (8 * xi ** 2)) * np.exp(-1j * (KX * x[0, 0] + KY * x[0, 1] + KZ * x[0, 2]))
    low = (np.abs(KX) < 2 * np.pi * 4) & (np.abs(KY) < 2 * np.pi * 4) & (np.abs(KZ) < 2 * np.pi * 4)   # aliasing e^{-eta (2pi 28)^2/8xi^2} ~ 1e-14
    assert np.max(np.abs(Hh - ref)[low]) < 1e-12


def test_p2g_points_equals_p2g(cfg1):
    c, x, f, o = cfg1
    rng = np.random.default_rng(3)
    gi = rng.integers(0, c.M, size=(50, 3))
    Hs = oracle.p2g_points(o["xw"], f, c.L, c.xi, c.M, c.P, gi)
    ref = o["H"][:, gi[:, 0], gi[:, 1], gi[:, 2]].T
    np.testing.assert_allclose(Hs, ref, rtol=1e-12, atol=1e-12 * np.abs(ref).max())


def test_p2g_periodic_wrap():
    """A particle near the corner spreads across the periodic boundary: shifting particle
    and grid by whole grid cells is a roll of H."""
    L, xi, M, P = 1.0, 12.0, 40, 24
    f = np.array([[1.0, -1.0, 2.0]])
    h = L / M
    x0 = np.array([[0.31 * h, 0.77 * h, 0.05 * h]])
    H0 = oracle.p2g(x0, f, L, xi, M, P)
    x1 = x0 + np.array([[17 * h, 5 * h, 33 * h]])
    H1 = oracle.p2g(x1, f, L, xi, M, P)
    np.testing.assert_allclose(np.roll(H0, (17, 5, 33), axis=(1, 2, 3)), H1, rtol=1e-9, atol=1e-13 * H0.max())


def test_g2p_is_adjoint_of_p2g(cfg1):
    """G2P is the transpose of P2G:  <G2P(Y), f> = h^3 <Y, P2G(f)>."""
    c, x, f, o = cfg1
    Y = W.smooth_grid(11, c.M)
    uY = oracle.g2p(o["xw"], Y, c.L, c.xi, c.M, c.P)
    lhs = np.sum(uY * f)
    rhs = (c.L / c.M) ** 3 * np.sum(Y * o["H"])
    assert abs(lhs - rhs) < 1e-12 * abs(rhs)


def test_g2p_interpolates_low_modes():
    """h^3 sum_g w(x-g) cos(k.g) = w_hat(k) cos(k.x) for a resolved mode (quadrature of (2.7))."""
    L, xi, M, P = 1.0, 10.0, 32, 24
    p = oracle.params(L, xi, M, P)
    g = np.arange(M) / M
    kv = 2 * np.pi * np.array([2, -1, 3])
    Y = np.zeros((3, M, M, M))
    Y[1] = np.cos(kv[0] * g[:, None, None] + kv[1] * g[None, :, None] + kv[2] * g[None, None, :])
    xt = np.array([[0.1234, 0.777, 0.4321], [0.999, 0.001, 0.5]])
    u = oracle.g2p(xt, Y, L, xi, M, P)
    ref = np.exp(-p["eta"] * (kv @ kv) / (8 * xi ** 2)) * np.cos(xt @ kv)
    np.testing.assert_allclose(u[:, 1], ref, atol=1e-13)
    assert np.all(u[:, 0] == 0)


def test_scale_structure(cfg1):
    """Discrete incompressibility k.H~hat = 0 (structure of (2.4b)); zero at k=0 and on Nyquist
    planes (S2, S8); the scaled spectrum keeps Hermitian symmetry (real inverse)."""
    c, x, f, o = cfg1
    Hs = o["Hs"]
    M = c.M
    n = np.fft.fftfreq(M, 1.0 / M)
    k = 2 * np.pi * n / c.L
    div = (k[:, None, None] * Hs[0] + k[None, :, None] * Hs[1] + k[None, None, :] * Hs[2])
    assert np.abs(div).max() < 1e-12 * np.abs(Hs).max() * np.abs(k).max()
    assert np.all(Hs[:, 0, 0, 0] == 0)
    assert np.all(Hs[:, M // 2] == 0) and np.all(Hs[:, :, M // 2] == 0) and np.all(Hs[:, :, :, M // 2] == 0)
    back = np.fft.ifftn(Hs, axes=(1, 2, 3))
    assert np.abs(back.imag).max() < 1e-14 * np.abs(back.real).max()


def test_scale_mode_closed_form():
    """One mode against (2.4b)/(2.6) typed with numpy: k=(2pi/L)(3,-2,5), M=32."""
    L, xi, M, P = 2.0, 7.0, 32, 24
    p = oracle.params(L, xi, M, P)
    idx = np.array([[3, M - 2, 5]])
    v = np.array([[1 + 2j, -0.5 + 0.25j, 3 - 1j]])
    out = oracle.scale_modes(idx, v, L, xi, M, P)[0]
    k = 2 * np.pi * np.array([3, -2, 5]) / L
    k2 = k @ k
    GF = 8 * np.pi / k2 ** 2 * (np.eye(3) * k2 - np.outer(k, k)) * np.exp(-k2 / (2 * xi) ** 2) * (1 + k2 / (2 * xi) ** 2)
    what = np.exp(-p["eta"] * k2 / (8 * xi ** 2))
    ref = (GF @ v[0]) / what ** 2 * (L / M) ** 3 / L ** 3
    np.testing.assert_allclose(out, ref, rtol=1e-13)


def test_operator_symmetry_and_linearity(cfg1):
    c, x, f, o = cfg1
    rng = np.random.default_rng(9)
    g = rng.standard_normal(f.shape)
    og = oracle.se_eval(x, g, c.L, c.xi, c.rc, c.M, c.P)
    a, b = np.sum(g * o["u"]), np.sum(f * og["u"])
    assert abs(a - b) < 1e-13 * (abs(a) + abs(b))
    ofg = oracle.se_eval(x, 2 * f - 3 * g, c.L, c.xi, c.rc, c.M, c.P)
    assert rel(ofg["u"], 2 * o["u"] - 3 * og["u"]) < 1e-13


def test_translation_invariance_to_method_error(cfg1):
    c, x, f, o = cfg1
    s = np.array([0.1234567, 0.7654321, 0.333333])
    o2 = oracle.se_eval(np.mod(x + s, c.L), f, c.L, c.xi, c.rc, c.M, c.P)
    assert rel(o2["u"], o["u"]) < 2e-9


def test_length_scaling(cfg1):
    c, x, f, o = cfg1
    Ls = 2.5
    o2 = oracle.se_eval(Ls * x, f, Ls * c.L, c.xi / Ls, Ls * c.rc, c.M, c.P)
    assert rel(Ls * o2["u"], o["u"]) < 1e-12


def test_wrap():
    x = np.array([[-0.25, 1.0, 2.75], [0.0, 0.5, -1e-18]])
    w = oracle.wrap(x, 1.0)
    assert np.all(w >= 0) and np.all(w < 1.0)
    np.testing.assert_allclose(w[0], [0.75, 0.0, 0.75])


def test_unwrapped_input_same_result(cfg1):
    c, x, f, o = cfg1
    shift = np.random.default_rng(4).integers(-2, 3, size=x.shape).astype(float)
    o2 = oracle.se_eval(x + shift * c.L, f, c.L, c.xi, c.rc, c.M, c.P)
    assert rel(o2["u"], o["u"]) < 1e-11


def test_cfg4_like_accuracy():
    """Config 4's dimensionless parameters (xi rc = 3.195, P = 12) give ~1e-5 vs the exact sum."""
    c, x, f = W.scaled(4, 1000)
    x = x.astype(np.float64); f = f.astype(np.float64)
    o = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P)
    ud = oracle.direct_ewald(x, f, c.L, min(c.xi, 12.0))
    e = rel(o["u"], ud)
    assert 1e-7 < e < 1e-4


def test_separate_targets(cfg1, cfg1_direct):
    """N_t != N_s (eq. (1.1)): at targets that ARE the sources the target form gives u + self term
    (the i = j pair is skipped by r > 0 in both); at other points it matches O1 evaluated at those targets."""
    c, x, f, o = cfg1
    sel = np.arange(0, c.N, 7)
    ot = oracle.se_eval_targets(x, f, x[sel], c.L, c.xi, c.rc, c.M, c.P)
    self_term = 4 * c.xi / np.sqrt(np.pi) * f[sel]
    assert rel(ot["u"] - self_term, o["u"][sel]) < 1e-13
    np.testing.assert_allclose(ot["uN"], o["uN"][sel], rtol=1e-12, atol=1e-12 * np.abs(o["uN"]).max())
    xt = np.random.default_rng(12).random((150, 3)) * c.L
    ot = oracle.se_eval_targets(x, f, xt, c.L, c.xi, c.rc, c.M, c.P)
    ud = oracle.direct_ewald(x, f, c.L, c.xi, targets=xt)
    assert rel(ot["u"], ud) < 1e-9
