"""Tolerance-driven parameter selection (section 2.4, eq. (2.9) at PAPER.md:153).  CPU only:
se_select_params is host arithmetic (no CUDA call), so it runs through the C-ABI here.

What fixes it, other than itself: the printed E^N and E^F of eq. (2.9) retyped with numpy; the rule of PAPER.md:159
(each term below eps/3); and the measured RMS error of the ORACLE run at the chosen parameters against the exact
direct Ewald sum O1, normalised as the paper does (unit box, sum_j |f_j|^2 = 1).
"""
import numpy as np
import pytest

import oracle
import paper_2606_19059_b200 as se
from paper_2606_19059_b200 import workloads as W


def e_near(xi, rc):
    return np.sqrt(112.0 / 9.0 * xi ** 4 * rc ** 3) * np.exp(-(xi * rc) ** 2)


def e_grid(xi, h):
    return 4.0 / (3.0 * h) * np.sqrt(7.0 / 2.0) * np.exp(-np.pi ** 2 / (2 * h * xi) ** 2)


@pytest.mark.parametrize("window", ["gaussian", "kb"])
@pytest.mark.parametrize("eps", [1e-3, 1e-6, 1e-9])
def test_terms_of_eq_2_9(window, eps):
    N, L = 200_000, 1.0
    q = se.select_params(N, L, eps, window, "fp64")
    assert q.EN == pytest.approx(e_near(q.xi, q.rc), rel=1e-12)
    assert q.EF == pytest.approx(e_grid(q.xi, L / q.M), rel=1e-12)
    assert q.EN <= eps / 3 and q.EF <= eps / 3 and q.Ew <= eps / 3
    assert q.EN > eps / 3 * 0.5                                             # xi is the smallest admissible one
    assert q.M % 2 == 0 and q.P % 2 == 0 and 2 <= q.P <= (16 if window == "kb" else 32)
    assert L / q.rc >= 3 and q.s == pytest.approx(N * q.rc ** 3, rel=1e-12)  # s = N_s rc^3
    assert q.model_ms > 0
    m = q.M
    for p in (2, 3, 5, 7):
        while m % p == 0:
            m //= p
    assert m == 1


def test_box_scaling_and_monotonicity():
    """L only rescales lengths: rc ~ L, xi ~ 1/L, same M and P; a tighter tolerance never gets a cheaper plan."""
    a = se.select_params(50_000, 1.0, 1e-6)
    b = se.select_params(50_000, 2.5, 1e-6)
    assert (a.M, a.P) == (b.M, b.P)
    assert b.rc == pytest.approx(2.5 * a.rc, rel=1e-12) and b.xi == pytest.approx(a.xi / 2.5, rel=1e-12)
    t = [se.select_params(50_000, 1.0, e).model_ms for e in (1e-3, 1e-5, 1e-7, 1e-9, 1e-11)]
    assert all(t[i] <= t[i + 1] for i in range(len(t) - 1))
    # the Kaiser-Bessel window needs a smaller support than the Gaussian for the same tolerance
    assert se.select_params(50_000, 1.0, 1e-9, "kb").P < se.select_params(50_000, 1.0, 1e-9, "gaussian").P


def test_rejects_bad_arguments():
    for kw in (dict(N=0), dict(L=0.0), dict(eps=0.5), dict(eps=1e-17), dict(eps=float("nan"))):
        a = dict(N=1000, L=1.0, eps=1e-6)
        a.update(kw)
        with pytest.raises(se.SeError) as ei:
            se.select_params(**a)
        assert ei.value.status == 1


@pytest.mark.parametrize("window,eps", [("gaussian", 1e-4), ("gaussian", 1e-8), ("kb", 1e-4), ("kb", 1e-8)])
def test_chosen_parameters_meet_the_tolerance(window, eps):
    """The oracle run at the selected (rc, xi, M, P) is within eps (RMS, paper's normalisation) of the exact sum,
    and not absurdly below it (the estimate is an upper bound, not a gross overestimate)."""
    N, L = 1200, 1.0
    x, f = W.uniform_cloud(4242, N, L)
    f /= np.sqrt((f ** 2).sum())
    q = se.select_params(N, L, eps, window, "fp64")
    o = oracle.se_eval(x, f, L, q.xi, q.rc, q.M, q.P, window="kb_poly" if window == "kb" else window)
    ud = oracle.direct_ewald(x, f, L, 8.0)
    e_rms = np.sqrt(((o["u"] - ud) ** 2).sum(axis=1).mean())
    assert e_rms <= eps, (e_rms, eps)
    assert e_rms >= 1e-3 * eps, (e_rms, eps)
