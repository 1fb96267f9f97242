"""GPU parity for the rows SURVEY.md section 8(f) marks "next": the Kaiser-Bessel polynomial window
(eq. (2.8)), separate targets N_t != N_s (eq. (1.1)), plans made from
a tolerance, and the measured-peak hook bench.py's rooflines divide by.

Kaiser-Bessel tolerances: both sides interpolate eq. (2.8) at the same nu + 1 Chebyshev points per bin, so the
polynomials are the same mathematically; each side converts to monomials on its own (numpy in double, the library in
long double), which leaves coefficient differences of ~1e-15 of the window's peak.  The gates below are those of
test_gpu_parity.py.
"""
from dataclasses import replace

import numpy as np
import pytest

import oracle
from paper_2606_19059_b200 import workloads as W
from gpu_util import gate, rel
from test_gpu_parity import TOL, check_all

pytestmark = pytest.mark.gpu


# ---- Kaiser-Bessel window --------------------------------------------------------------------------------------
@pytest.mark.parametrize("P,M", [(8, 40), (12, 50), (16, 48), (4, 26), (6, 30), (10, 44), (14, 36)])
def test_kb_window_fp64(P, M):
    """P = 8, 12, 16 run the FP64 tensor-core sweep, the others the generic tile kernel."""
    rng = np.random.default_rng(300 + P)
    c = replace(W.CONFIGS[1], N=1100, rc=0.2, xi=12.0, M=M, P=P, window="kb", label=f"KB P={P} M={M}")
    x = rng.random((1100, 3)); f = rng.standard_normal((1100, 3))
    x[0] = [0.0, 0.0, 0.0]
    x[1] = [3 * c.L / M, 7 * c.L / M, 0.5]           # on grid points: the support point at r = a_w exactly
    check_all(c, x, f)


@pytest.mark.parametrize("P,M", [(8, 40), (12, 38), (6, 30)])
def test_kb_window_fp32(P, M):
    rng = np.random.default_rng(320 + P)
    c = replace(W.CONFIGS[4], N=1500, rc=0.2, xi=12.0, M=M, P=P, window="kb", label=f"KB fp32 P={P} M={M}")
    x = rng.random((1500, 3)).astype(np.float32); f = rng.standard_normal((1500, 3)).astype(np.float32)
    check_all(c, x, f)


def test_kb_cfg1_is_a_nine_digit_sum():
    """Config 1's split with the paper's window at P = 12: the GPU result itself is within 2e-9 of the exact sum
    (the Gaussian needs P = 24 for this)."""
    import torch
    import paper_2606_19059_b200 as se
    c, x, f = W.make(1)
    xd = torch.as_tensor(x, device="cuda"); fd = torch.as_tensor(f, device="cuda")
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, 12, window="kb") as plan:
        i = plan.info()
        assert i.window == se.SE_WINDOW_KAISER_BESSEL and i.nu == 13 and i.kb_beta == 30.0 and i.grid_mode == 2
        u = plan.eval(xd, fd).cpu().numpy()
    assert rel(u, oracle.direct_ewald(x, f, c.L, c.xi)) < 2e-9


def test_kb_scaled_cfg3_like():
    """Config 3's dimensionless split with the Kaiser-Bessel window at P = 8 and P = 12, several thousand points."""
    c, x, f = W.scaled(3, 6000)
    for P in (8, 12):
        check_all(replace(c, P=P, window="kb", label=f"cfg3-scaled KB P={P}"), x, f)


def test_kb_rejects_large_support():
    import paper_2606_19059_b200 as se
    with pytest.raises(se.SeError) as ei:
        se.Plan(100, 1.0, 10.0, 0.2, 48, 18, window="kb")
    assert ei.value.status == 1


# ---- separate targets ------------------------------------------------------------------------------------------
def _targets_case(prec, window, P, M, N=4000, Nt=1777, seed=0):
    import torch
    import paper_2606_19059_b200 as se
    rng = np.random.default_rng(500 + seed)
    L, rc, xi = 1.0, 0.19, 12.5
    dt = np.float64 if prec == "fp64" else np.float32
    xs = rng.random((N, 3)).astype(dt); f = rng.standard_normal((N, 3)).astype(dt)
    xt = (rng.random((Nt, 3)) * 1.5 - 0.25).astype(dt)        # some outside the box
    k = min(40, Nt, N)
    xt[:k] = xs[:k]                                           # targets on top of sources: that pair is skipped
    xt[-1] = [0.0, 0.0, 0.0] if Nt > 1 else xt[-1]
    o = oracle.se_eval_targets(xs, f, xt, L, xi, rc, M, P, window="kb_poly" if window == "kb" else window)
    tdt = torch.float64 if prec == "fp64" else torch.float32
    xd = torch.as_tensor(xs, dtype=tdt, device="cuda"); fd = torch.as_tensor(f, dtype=tdt, device="cuda")
    td = torch.as_tensor(xt, dtype=tdt, device="cuda")
    tol = TOL[prec]
    with se.Plan(N, L, xi, rc, M, P, prec, window=window, Nt=Nt) as plan:
        info = plan.info()
        assert info.N == N and info.Nt == Nt
        ut = plan.eval_targets(xd, fd, td)
        torch.cuda.synchronize()
        gate("u", ut.cpu().numpy(), o["u"], tol["u"])
        # se_eval is for plans without own targets
        with pytest.raises(se.SeError):
            plan.eval(xd, fd)
        # stage by stage: sort both sets, near field at the targets, far field gathered at the targets
        plan.set_targets(td)
        plan.stage("sort", x=xd, f=fd)
        pn = plan.read(se.SE_BUF_PERM_NEAR | se.SE_BUF_TARGETS).cpu().numpy()
        pg = plan.read(se.SE_BUF_PERM_GRID | se.SE_BUF_TARGETS).cpu().numpy()
        ps = plan.read(se.SE_BUF_PERM_NEAR).cpu().numpy()
        assert np.array_equal(np.sort(pn), np.arange(Nt)) and np.array_equal(np.sort(pg), np.arange(Nt))
        assert np.array_equal(np.sort(ps), np.arange(N))
        plan.stage("p2p")
        uN = np.empty((Nt, 3)); uN[pn] = plan.read(se.SE_BUF_UN).cpu().numpy()
        gate("uN", uN, o["uN"], tol["uN"])
        for st in ("p2g", "fft", "scale", "ifft", "g2p"):
            plan.stage(st)
        uF = np.empty((Nt, 3)); uF[pg] = plan.read(se.SE_BUF_UF).cpu().numpy().astype(np.float64) * info.h ** 3 * info.cw
        gate("uF", uF, o["uF"], tol["uF"])
        u2 = torch.empty_like(td)
        plan.stage("sum", u=u2)
        torch.cuda.synchronize()
        if info.grid_mode == 2 and not info.fft_fused:        # the tensor-core sweep is bit-reproducible
            assert torch.equal(u2, ut)                        # (fused plans: se_eval_targets and the stages transform in different orders)
        elif info.fft_fused:                                  # two transform orders in the plan's precision
            assert rel(u2.cpu().numpy(), ut.cpu().numpy()) < 0.1 * tol["u"]
        else:                                                 # generic G2P adds with atomics: same to rounding
            assert rel(u2.cpu().numpy(), ut.cpu().numpy()) < 1e-3 * tol["u"]
    return o


@pytest.mark.parametrize("prec,window,P,M", [("fp64", "gaussian", 24, 60), ("fp64", "kb", 12, 48),
                                             ("fp64", "gaussian", 10, 40), ("fp32", "gaussian", 12, 40),
                                             ("fp32", "kb", 8, 40)])
def test_separate_targets(prec, window, P, M):
    _targets_case(prec, window, P, M)


def test_targets_more_than_sources_and_single_target():
    _targets_case("fp64", "gaussian", 16, 48, N=700, Nt=5000, seed=1)
    _targets_case("fp64", "kb", 8, 40, N=3000, Nt=1, seed=2)


def test_targets_equal_sources_differ_by_self_term():
    """Targets placed exactly on the sources: u_targets = u_eval + (4 xi / sqrt(pi)) f (the i = j pair is skipped by
    r > 0 in both; only se_eval adds the self term, reading S3)."""
    import torch
    import paper_2606_19059_b200 as se
    c, x, f = W.scaled(2, 3000)
    xd = torch.as_tensor(x, device="cuda"); fd = torch.as_tensor(f, device="cuda")
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P) as p0, se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, Nt=c.N) as p1:
        u0 = p0.eval(xd, fd).cpu().numpy()
        u1 = p1.eval_targets(xd, fd, xd).cpu().numpy()
    assert rel(u1 - 4 * c.xi / np.sqrt(np.pi) * f, u0) < 1e-13


# ---- plans from a tolerance --------------------------------------------------------------------------------------
@pytest.mark.parametrize("window,eps,prec", [("gaussian", 1e-4, "fp64"), ("gaussian", 1e-9, "fp64"), ("kb", 1e-6, "fp64"),
                                             ("kb", 1e-9, "fp64"), ("kb", 1e-4, "fp32")])
def test_plan_from_tolerance(window, eps, prec):
    """se_plan_create_tol: the GPU result is within eps (RMS, unit box, sum |f|^2 = 1) of the exact sum
    O1, and equals the oracle's SE sum at the chosen parameters to the parity gate."""
    import torch
    import paper_2606_19059_b200 as se
    N, L = 3000, 1.0
    x, f = W.uniform_cloud(777, N, L)
    f /= np.sqrt((f ** 2).sum())
    dt = np.float64 if prec == "fp64" else np.float32
    x = x.astype(dt); f = f.astype(dt)
    tdt = torch.float64 if prec == "fp64" else torch.float32
    xd = torch.as_tensor(x, dtype=tdt, device="cuda"); fd = torch.as_tensor(f, dtype=tdt, device="cuda")
    with se.Plan(N, L, eps=eps, window=window, precision=prec) as plan:
        q, i = plan.chosen, plan.info()
        assert (i.M, i.P) == (q.M, q.P) and i.rc == q.rc and i.xi == q.xi
        u = plan.eval(xd, fd).cpu().numpy().astype(np.float64)
    ud = oracle.direct_ewald(x, f, L, 8.0)
    e_rms = np.sqrt(((u - ud) ** 2).sum(axis=1).mean())
    print(f"eps {eps:g} {window} {prec}: rc {q.rc:.4f} xi {q.xi:.2f} M {q.M} P {q.P}  E_rms {e_rms:.2e}")
    assert e_rms <= eps
    o = oracle.se_eval(x, f, L, q.xi, q.rc, q.M, q.P, window="kb_poly" if window == "kb" else window)
    gate("u", u, o["u"], TOL[prec]["u"])


# ---- measured peaks ----------------------------------------------------------------------------------------------
def test_measured_peaks_are_plausible():
    """Register-only chains: FP64 FMA and FP64 tensor op in the tens of TFLOP/s, FP32 FMA above both."""
    import paper_2606_19059_b200 as se
    d, t, s = se.measure_peak("fp64"), se.measure_peak("fp64_tensor"), se.measure_peak("fp32")
    print(f"measured peaks: fp64 {d:.1f}  fp64 tensor {t:.1f}  fp32 {s:.1f} TFLOP/s")
    assert 20.0 < d < 45.0 and 20.0 < t < 45.0 and 55.0 < s < 90.0
    h = se.measure_peak("hbm")
    print(f"read + write stream: {h:.2f} TB/s")
    assert 4.0 < h < 8.5


def test_count_pairs_matches_brute_force():
    """se_count_pairs (bench.py's K2 work count) against a numpy count over all pairs and 27 images."""
    import torch
    import paper_2606_19059_b200 as se
    c, x, f = W.scaled(2, 1500)
    xd = torch.as_tensor(x, device="cuda"); fd = torch.as_tensor(f, device="cuda")
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P) as plan:
        plan.eval(xd, fd)
        cand, hits = plan.count_pairs()
        nc = plan.info().ncell
    xw = oracle.wrap(x, c.L)
    d = xw[:, None, :] - xw[None, :, :]
    d -= c.L * np.round(d / c.L)
    r2 = (d ** 2).sum(-1)
    ref = int(((r2 <= c.rc ** 2) & (r2 > 0)).sum())          # rc < L/2: the nearest image is the only one in range
    assert abs(hits - ref) <= 2                               # FP32 count: a pair at the cutoff may flip
    cid = np.minimum((xw / (c.L / nc)).astype(int), nc - 1)
    occ = np.zeros((nc, nc, nc), int)
    np.add.at(occ, (cid[:, 0], cid[:, 1], cid[:, 2]), 1)
    tot = sum(np.roll(occ, (a, b, e), (0, 1, 2)) for a in (-1, 0, 1) for b in (-1, 0, 1) for e in (-1, 0, 1))
    assert cand == int((occ * tot).sum())


def test_plan_is_bound_to_its_device():
    """Every call on a plan must be made with the plan's device current (se.h conventions); with one visible GPU the
    rule is checked on the only device, and the per-plan kernel attributes by making two plans in a row."""
    import torch
    import paper_2606_19059_b200 as se
    c, x, f = W.scaled(2, 2000)
    xd = torch.as_tensor(x, device="cuda"); fd = torch.as_tensor(f, device="cuda")
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P) as a, se.Plan(c.N, c.L, c.xi, c.rc, c.M, 16) as b:
        ua, ub = a.eval(xd, fd), b.eval(xd, fd)
        torch.cuda.synchronize()
        assert rel(ua.cpu().numpy(), ub.cpu().numpy()) < 1e-5


def test_fp32_near_field_with_thirty_thousand_neighbours():
    """fp32 K2 on a dense blob (40,000 points in a ball of radius 0.08, rc = 0.2: ~30,000 in-range sources per target):
    K2 sums the pairs of a round in float and the rounds in double, so u^N stays inside the 3e-6 gate however many
    neighbours a target has (a float accumulator drifted to 2.7e-5 here).  Not a BASELINE workload."""
    import torch
    import paper_2606_19059_b200 as se
    rng = np.random.default_rng(190590 + 77)
    N, L, rc = 40000, 1.0, 0.2
    xi = 3.195 / rc                                            # config 4's xi rc
    v = rng.standard_normal((N, 3))
    v /= np.linalg.norm(v, axis=1)[:, None]
    x = (0.5 + 0.08 * rng.random((N, 1)) ** (1.0 / 3.0) * v).astype(np.float32)
    f = rng.standard_normal((N, 3)).astype(np.float32)
    xd = torch.as_tensor(x, device="cuda"); fd = torch.as_tensor(f, device="cuda")
    with se.Plan(N, L, xi, rc, 32, 12, "fp32") as plan:
        plan.stage("sort", x=xd, f=fd)
        perm = plan.read(se.SE_BUF_PERM_NEAR).cpu().numpy()
        plan.stage("p2p")
        uN_sorted = plan.read(se.SE_BUF_UN).cpu().numpy()
        cand, hits = plan.count_pairs()
    assert hits / N > 25000
    uN = np.empty_like(uN_sorted)
    uN[perm] = uN_sorted
    # the oracle on a sample of targets (O(N) each), in double on the rounded inputs (reading S17)
    xw = oracle.wrap(x.astype(np.float64), L)
    idx = rng.choice(N, 256, replace=False)
    ref = oracle.near_brute(xw, f.astype(np.float64), L, xi, rc, targets=idx)
    e, m = gate("uN dense blob fp32", uN[idx], ref, TOL["fp32"]["uN"])
    print(f"fp32 u^N with {hits / N:.0f} neighbours per target: rel-L2 {e:.2e}, max-abs {m:.2e}")
