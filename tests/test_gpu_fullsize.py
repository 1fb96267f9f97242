"""GPU parity at BASELINE.json's FULL sizes (configs 3, 4, 5), in the launch configuration bench.py times.

The oracle cannot run the 4M-particle / 576^3 configs end to end in test time, so every stage is compared on
SAMPLED outputs the oracle computes one by one from the same seeded inputs:
  K1  exactly: permutations are bijections, CSR ranges complete, sampled particles lie in their cell;
  K2  u^N of sampled targets           vs  oracle.near_brute (plain loop over all N sources and 27 images);
  K3  H at sampled grid points         vs  oracle.p2g_points (gather form, loop over all N particles);
  K4  sampled modes of an index-defined synthetic spectrum  vs  oracle.scale_modes;
  K5  u^F of sampled particles on an index-defined synthetic grid  vs  oracle.g2p (P^3 sum each);
  K6  u = u^N + u^F - (4 xi / sqrt(pi)) f on the sampled particles, from the oracle's own u^N and u^F of
      that synthetic grid, against the device's sum of its own stage outputs.
The two FFT steps are cuFFT (library), covered end to end by the full config 3 run below and by the
smaller cases of test_gpu_parity.py.  Config 3 (the bench workload) is also compared in full, all N,
against oracle.se_eval.  Tolerances as in test_gpu_parity.py.
"""
import numpy as np
import pytest

import oracle
from paper_2606_19059_b200 import workloads as W
from gpu_util import MAXABS_FACTOR, gate, maxabs, rel

pytestmark = pytest.mark.gpu

TOL = {
    "fp64": dict(uN=1e-12, H=1e-13, Hs=1e-12, uF=1e-12, u=1e-11),
    "fp32": dict(uN=3e-6, H=1e-6, Hs=3e-6, uF=3e-6, u=1e-5),
}


def _sampled_stages(cfg, n_near=48, n_grid=400, n_far=400):
    import torch
    import paper_2606_19059_b200 as se

    c, x, f = W.make(cfg)
    tol = TOL[c.precision]
    N, M, P, L = c.N, c.M, c.P, c.L
    rng = np.random.default_rng(4242 + cfg)
    x64, f64 = x.astype(np.float64), f.astype(np.float64)
    xw = oracle.wrap(x64, L)
    dt = torch.float64 if c.precision == "fp64" else torch.float32
    xd = torch.as_tensor(x, dtype=dt, device="cuda").contiguous()
    fd = torch.as_tensor(f, dtype=dt, device="cuda").contiguous()
    errs = {}
    with se.Plan(N, L, c.xi, c.rc, M, P, c.precision) as plan:
        info = plan.info()
        # ---- K1 ------------------------------------------------------------------------------
        plan.stage("sort", x=xd, f=fd)
        ar = torch.arange(N, device="cuda", dtype=torch.int64)
        inv = {}
        for key, buf in (("near", se.SE_BUF_PERM_NEAR), ("grid", se.SE_BUF_PERM_GRID)):
            perm = plan.read(buf).to(torch.int64)
            assert torch.equal(torch.sort(perm).values, ar)
            iv = torch.empty_like(perm)
            iv[perm] = ar
            inv[key] = iv
        cs = plan.read(se.SE_BUF_CELL_START).cpu().numpy()
        assert cs[0] == 0 and cs[-1] == N and np.all(np.diff(cs) >= 0)
        bs = plan.read(se.SE_BUF_BIN_START)
        assert int(bs[0]) == 0 and int(bs[-1]) == N and bool((bs[1:] >= bs[:-1]).all())
        del bs
        tid = rng.choice(N, n_near, replace=False)
        nc = info.ncell
        cid = np.minimum(np.floor(xw[tid] / (L / nc)).astype(np.int64), nc - 1)
        lin = (cid[:, 0] * nc + cid[:, 1]) * nc + cid[:, 2]
        pos = inv["near"][torch.as_tensor(tid, device="cuda")].cpu().numpy()
        assert np.all((cs[lin] <= pos) & (pos < cs[lin + 1]))
        # ---- K2 ------------------------------------------------------------------------------
        plan.stage("p2p")
        uN_s = plan.read(se.SE_BUF_UN)[torch.as_tensor(pos, device="cuda")].cpu().numpy()
        uN_ref = oracle.near_brute(xw, f64, L, c.xi, c.rc, targets=tid)
        errs["uN"] = rel(uN_s, uN_ref); mx = {"uN": maxabs(uN_s, uN_ref)}
        # ---- K3 ------------------------------------------------------------------------------
        plan.stage("p2g")
        pid = rng.choice(N, n_grid, replace=False)
        g0 = np.floor(xw[pid] / (L / M)).astype(np.int64)
        gidx = np.mod(g0 + rng.integers(-(P // 2) - 1, P // 2 + 2, size=(n_grid, 3)), M)
        H = plan.read(se.SE_BUF_GRID)
        gi = torch.as_tensor(gidx, device="cuda")
        H_s = H[:, gi[:, 0], gi[:, 1], gi[:, 2]].T.cpu().numpy()
        del H
        H_ref = oracle.p2g_points(xw, f64, L, c.xi, M, P, gidx)
        errs["H"] = rel(H_s, H_ref); mx["H"] = maxabs(H_s, H_ref)
        # ---- K4 on an index-defined spectrum ---------------------------------------------------
        mh = M // 2 + 1
        for comp in range(3):                                   # written plane by plane: no 4.6 GB temporaries
            sp = torch.empty((M, M, mh, 2), dtype=dt, device="cuda")
            ii = torch.arange(M, device="cuda", dtype=torch.float64)[:, None, None]
            jj = torch.arange(M, device="cuda", dtype=torch.float64)[None, :, None]
            kk = torch.arange(mh, device="cuda", dtype=torch.float64)[None, None, :]
            step = max(1, M // 8)
            for i0 in range(0, M, step):
                re, im = W.index_spectrum(torch, comp, ii[i0:i0 + step], jj, kk)
                sp[i0:i0 + step, ..., 0] = re.to(dt)
                sp[i0:i0 + step, ..., 1] = im.to(dt)
            if comp == 0:
                spec = torch.empty((3, M, M, mh, 2), dtype=dt, device="cuda")
            spec[comp] = sp
            del sp
        plan.write(se.SE_BUF_SPEC, spec)
        midx = np.stack([rng.integers(0, M, n_far), rng.integers(0, M, n_far), rng.integers(0, mh, n_far)], axis=1)
        midx[:5] = [[0, 0, 0], [M // 2, 1, 1], [1, M // 2, 2], [3, 4, M // 2], [M - 1, M - 1, 1]]
        mi = torch.as_tensor(midx, device="cuda")
        vin = spec[:, mi[:, 0], mi[:, 1], mi[:, 2]].cpu().numpy().astype(np.float64)      # (3, ns, 2): as stored
        del spec
        plan.stage("scale")
        got = plan.read(se.SE_BUF_SPEC)[:, mi[:, 0], mi[:, 1], mi[:, 2]].cpu().numpy().astype(np.float64)
        ref = oracle.scale_modes(midx, (vin[..., 0] + 1j * vin[..., 1]).T.copy(), L, c.xi, M, P)
        gv = (got[..., 0] + 1j * got[..., 1]).T
        errs["Hs"] = rel(gv, ref); mx["Hs"] = maxabs(gv, ref)
        assert np.all(gv[:4] == 0)                              # k = 0 and the Nyquist planes (reading S8)
        # ---- K5 on an index-defined grid -------------------------------------------------------
        Y = torch.empty((3, M, M, M), dtype=dt, device="cuda")
        ii = torch.arange(M, device="cuda", dtype=torch.float64)[:, None, None]
        jj = torch.arange(M, device="cuda", dtype=torch.float64)[None, :, None]
        kk = torch.arange(M, device="cuda", dtype=torch.float64)[None, None, :]
        step = max(1, M // 8)
        for comp in range(3):
            for i0 in range(0, M, step):
                Y[comp, i0:i0 + step] = W.index_grid(torch, comp, ii[i0:i0 + step], jj, kk, M).to(dt)
        plan.write(se.SE_BUF_GRID, Y)
        del Y
        plan.stage("g2p")
        sid = rng.choice(N, n_far, replace=False)
        posg = inv["grid"][torch.as_tensor(sid, device="cuda")]
        uF_s = plan.read(se.SE_BUF_UF)[posg].cpu().numpy().astype(np.float64) * info.h ** 3 * info.cw
        # the oracle gathers from the same field, rounded to the plan's precision as the device stored it
        g = np.arange(M, dtype=np.float64)
        Yh = np.empty((3, M, M, M))
        for comp in range(3):
            v = W.index_grid(np, comp, g[:, None, None], g[None, :, None], g[None, None, :], M)
            Yh[comp] = v if c.precision == "fp64" else v.astype(np.float32)
        del v
        uF_ref = oracle.g2p(xw[sid], Yh, L, c.xi, M, P)
        del Yh
        errs["uF"] = rel(uF_s, uF_ref); mx["uF"] = maxabs(uF_s, uF_ref)
        # ---- K6 --------------------------------------------------------------------------------
        ud = torch.empty_like(xd)
        plan.stage("sum", f=fd, u=ud)
        torch.cuda.synchronize()
        u_s = ud[torch.as_tensor(sid, device="cuda")].cpu().numpy()
        uN_sid = oracle.near_brute(xw, f64, L, c.xi, c.rc, targets=sid[:n_near])
        u_ref = oracle.se_sum(uN_sid, uF_ref[:n_near], f64[sid[:n_near]], c.xi)
        errs["u"] = rel(u_s[:n_near], u_ref); mx["u"] = maxabs(u_s[:n_near], u_ref)
        launches = plan.launch_count()
    print(c.label, {k: f"{v:.2e}/{mx[k]:.2e}" for k, v in errs.items()})
    for k, v in errs.items():
        assert v <= tol[k], (k, v, tol[k])
        assert mx[k] <= MAXABS_FACTOR * tol[k], (k, "max-abs", mx[k])
    return errs


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_sampled_stages(cfg):
    _sampled_stages(cfg)


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_end_to_end(cfg):
    """BASELINE configs 3, 4 and 5 at full size, ALL N outputs of one se_eval (the real chain K1 .. K6 with both
    cuFFT batches, in the launch configuration bench.py times) against the SE oracle run in full
    (SURVEY.md 8(c) "Large configs": parity = GPU vs O2 at full size on all N)."""
    import gc
    import torch
    import paper_2606_19059_b200 as se
    c, x, f = W.make(cfg)
    dt = torch.float64 if c.precision == "fp64" else torch.float32
    xd = torch.as_tensor(x, dtype=dt, device="cuda"); fd = torch.as_tensor(f, dtype=dt, device="cuda")
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, c.precision) as plan:
        u = plan.eval(xd, fd)
        torch.cuda.synchronize()
        assert plan.launch_count() > 0
    u = u.cpu().numpy()
    del xd, fd
    torch.cuda.empty_cache()
    tm = {}
    o = oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P, timings=tm)
    ref = o["u"]
    del o
    gc.collect()
    e, m = gate("u", u, ref, TOL[c.precision]["u"])
    print(c.label, f"u rel-L2 {e:.2e} max-abs {m:.2e}; oracle seconds", {k: round(v, 1) for k, v in tm.items()})
