"""GPU parity of the slab decomposition (section 6.5; paper_2606_19059_b200/slabs.py): the ranks of a
2-, 3- or 4-slab run are executed one after the other on the one GPU of the test box, the exchanges being list shuffles
(slabs.evaluate_emulated), and the assembled result is compared with the oracle on all N.  The kernels, the slab plans
(se_plan_desc.Mx, px0, Nown), the ghost sources, the ghost-plane reduction, the slab-decomposed transform with K4 on the
pencils (se_scale_block) and the ghost planes of G2P are exactly those of a multi-GPU run; what is not exercised here is
torch.distributed itself (tests/test_slabs_host.py runs the exchanges under gloo on CPU tensors)."""
import numpy as np
import pytest

import oracle
from paper_2606_19059_b200 import workloads as W
from gpu_util import gate
from test_gpu_parity import TOL

pytestmark = pytest.mark.gpu


def run_slabs(c, x, f, world, P=None, window="gaussian"):
    import torch
    from paper_2606_19059_b200 import slabs
    P = c.P if P is None else P
    lay = slabs.SlabLayout(c.L, c.M, P, c.rc, world)
    own = lay.owner(x[:, 0].astype(np.float64))
    idx = [np.nonzero(own == r)[0] for r in range(world)]
    xs = [torch.as_tensor(x[i], device="cuda") for i in idx]
    fs = [torch.as_tensor(f[i], device="cuda") for i in idx]
    us = slabs.evaluate_emulated(lay, c.xi, xs, fs, precision=c.precision, window=window)
    u = np.empty_like(x)
    for i, ur in zip(idx, us):
        u[i] = ur.cpu().numpy()
    ref = oracle.se_eval(x.astype(np.float64), f.astype(np.float64), c.L, c.xi, c.rc, c.M, P,
                         window="kb_poly" if window == "kb" else window)["u"]
    return u, ref, [len(i) for i in idx]


@pytest.mark.parametrize("cfg,n,world", [(3, 20000, 2), (3, 20000, 4), (5, 30000, 4), (2, 20000, 2)])
def test_slabs_fp64(cfg, n, world):
    c, x, f = W.scaled(cfg, n)
    u, ref, counts = run_slabs(c, x, f, world)
    e, m = gate(f"u, {world} slabs", u, ref, TOL["fp64"]["u"])
    print(f"{c.label}: {world} slabs {counts}: rel-L2 {e:.2e}, max-abs {m:.2e}")


def test_slabs_fp32():
    c, x, f = W.scaled(4, 40000)
    u, ref, counts = run_slabs(c, x, f, 4)
    gate("u, 4 slabs fp32", u, ref, TOL["fp32"]["u"])


def test_slabs_kaiser_bessel():
    c, x, f = W.scaled(3, 20000)
    u, ref, _ = run_slabs(c, x, f, 4, P=12, window="kb")
    gate("u, 4 slabs, Kaiser-Bessel P = 12", u, ref, TOL["fp64"]["u"])


def test_slabs_config2_in_full():
    c, x, f = W.make(2)
    u, ref, _ = run_slabs(c, x, f, 3)
    gate("u, config 2, 3 slabs", u, ref, TOL["fp64"]["u"])


def test_slabs_empty_slab_and_points_on_faces():
    """All points in two of four slabs (the other two own planes but no points), some exactly on slab faces and on the box
    faces: ownership by floor(x/h), ghosts across the periodic boundary."""
    c, x, f = W.scaled(3, 6000)
    rng = np.random.default_rng(190590 + 99)
    x = x.copy()
    x[:, 0] = (0.75 + 0.5 * rng.random(c.N)) % 1.0                 # slabs 3 and 0 of four only
    x[:40, 0] = np.repeat([0.0, 0.25 - 1e-16, 0.75, 1.0 - 1e-16], 10)
    u, ref, counts = run_slabs(c, x, f, 4)
    assert counts[1] == 0 and counts[2] == 0
    gate("u, empty slabs", u, ref, TOL["fp64"]["u"])


def test_slabs_padded_ring_and_the_last_point_below_L():
    """P = 10 (ring of 16 / 12 planes, zero rows) on three slabs, M = 72: the largest double below L has x/h = M after
    rounding, so its base plane is plane 0 of rank 0 and it is a ghost source of the last rank (PAPER.md:215 anchor,
    periodic index wrap) -- at P = 10 the window's edge value (7e-7) makes a clamp to plane M - 1 visible."""
    from dataclasses import replace
    rng = np.random.default_rng(190590 + 7)
    N, M, P = 5000, 72, 10
    xi = 0.8 * 0.95 * np.sqrt(np.pi * P) * M / P
    c = replace(W.CONFIGS[3], N=N, M=M, P=P, rc=4.5 / xi, xi=xi, label="P = 10 slabs")
    x = rng.random((N, 3)); f = rng.standard_normal((N, 3))
    x[:30, 0] = np.repeat([0.0, np.nextafter(1.0, 0), np.nextafter(1.0 / 3.0, 0)], 10)
    assert np.floor(x[10, 0] / (1.0 / M)) == M
    u, ref, counts = run_slabs(c, x, f, 3)
    gate("u, 3 slabs, P = 10", u, ref, TOL["fp64"]["u"])


def test_slab_plan_rejects_bad_arguments():
    import paper_2606_19059_b200 as se
    c, x, f = W.scaled(3, 20000)
    bad = [dict(Mx=c.M + 2, px0=0), dict(Mx=8, px0=0), dict(Mx=48, px0=-1), dict(Mx=48, px0=c.M), dict(Mx=48, px0=0, Nown=5)]
    for kw in bad:
        with pytest.raises(se.SeError):
            se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, **kw)
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, Mx=48, px0=3) as p:
        i = p.info()
        assert (i.Mx, i.px0, i.grid_mode) == (48, 3, 2)
        with pytest.raises(se.SeError):
            p.stage("fft")                                          # a slab plan transforms nothing


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_scale_block_equals_the_scale_stage(prec):
    """se_scale_block on ky-pencils [3, M, nky, M/2 + 1] reproduces, block by block and bit for bit, what SE_STAGE_SCALE does
    to the whole spectrum (same kernel, ky offset), and agrees with the oracle's multiplier on sampled modes."""
    import torch
    import paper_2606_19059_b200 as se
    c, x, f = W.scaled(3 if prec == "fp64" else 4, 4000)
    M, Mh = c.M, c.M // 2 + 1
    rdt, cdt = (torch.float64, torch.complex128) if prec == "fp64" else (torch.float32, torch.complex64)
    g = torch.Generator(device="cuda").manual_seed(5)
    spec = torch.randn(3, M, M, Mh, 2, dtype=rdt, device="cuda", generator=g)
    with se.Plan(c.N, c.L, c.xi, c.rc, M, c.P, prec) as p:
        p.write(se.SE_BUF_SPEC, spec.clone())
        p.stage("scale")
        whole = torch.view_as_complex(p.read(se.SE_BUF_SPEC))
        sc = torch.view_as_complex(spec)
        for ky0, nky in ((0, 7), (7, M // 2 - 7), (M // 2, M - M // 2)):
            blk = sc[:, :, ky0:ky0 + nky].contiguous().to(cdt)
            p.scale_block(blk, ky0, nky)
            assert torch.equal(blk, whole[:, :, ky0:ky0 + nky])
    rng = np.random.default_rng(3)
    idx = np.stack([rng.integers(0, M, 300), rng.integers(0, M, 300), rng.integers(0, Mh, 300)], axis=1)
    vals = sc[:, idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy().T.astype(np.complex128)
    ref = oracle.scale_modes(idx, vals, c.L, c.xi, M, c.P)
    got = whole[:, idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy().T
    gate("scaled modes", got, ref, TOL[prec]["Hs"])


def test_slabs_config3_full_size_against_the_one_gpu_plan():
    """Config 3 at full size (N = 1,048,576, M = 360) cut into 4 slabs against se_eval on the whole problem (which
    tests/test_gpu_fullsize.py compares with the oracle on all N): same kernels, so the two agree to rounding."""
    import torch
    import paper_2606_19059_b200 as se
    from paper_2606_19059_b200 import slabs
    c, x, f = W.make(3)
    lay = slabs.SlabLayout(c.L, c.M, c.P, c.rc, 4)
    own = lay.owner(x[:, 0])
    idx = [np.nonzero(own == r)[0] for r in range(4)]
    us = slabs.evaluate_emulated(lay, c.xi, [torch.as_tensor(x[i], device="cuda") for i in idx],
                                 [torch.as_tensor(f[i], device="cuda") for i in idx])
    u = np.empty_like(x)
    for i, ur in zip(idx, us):
        u[i] = ur.cpu().numpy()
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P) as p:
        ref = p.eval(torch.as_tensor(x, device="cuda"), torch.as_tensor(f, device="cuda")).cpu().numpy()
    gate("u, config 3, 4 slabs vs one plan", u, ref, 1e-13)
