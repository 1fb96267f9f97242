"""Helpers for the GPU parity tests (call the CUDA path through the C-ABI binding only)."""
import numpy as np


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    dt = np.complex128 if (np.iscomplexobj(a) or np.iscomplexobj(b)) else np.float64
    a, b = a.astype(dt), b.astype(dt)
    den = float(np.linalg.norm(b))
    num = float(np.linalg.norm(a - b))
    if den == 0.0:                       # e.g. u^N of a single particle: both sides must be exactly zero
        return 0.0 if num == 0.0 else float("inf")
    return num / den


def maxabs(a, b):
    """max |a - b| over max |b|: the worst single element, next to the rel-L2 gate."""
    a, b = np.asarray(a), np.asarray(b)
    dt = np.complex128 if (np.iscomplexobj(a) or np.iscomplexobj(b)) else np.float64
    den = float(np.max(np.abs(b.astype(dt)))) if b.size else 0.0
    num = float(np.max(np.abs(a.astype(dt) - b.astype(dt)))) if b.size else 0.0
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return num / den


# gate on the worst element: MAXABS_FACTOR x the rel-L2 tolerance of the same array (a single element may sit
# above the root-mean-square error; a wrong element is orders of magnitude above either)
MAXABS_FACTOR = 10.0


def gate(name, got, ref, tol):
    """Assert rel-L2 <= tol and max-abs / max|ref| <= MAXABS_FACTOR tol; returns (rel, maxabs)."""
    e, m = rel(got, ref), maxabs(got, ref)
    assert e <= tol, (name, "rel-L2", e, tol)
    assert m <= MAXABS_FACTOR * tol, (name, "max-abs", m, MAXABS_FACTOR * tol)
    return e, m


def run_stages(c, x, f):
    """Run every stage through se_eval_stage and return the intermediates as numpy (user order)."""
    import torch
    import paper_2606_19059_b200 as se
    dt = torch.float64 if c.precision == "fp64" else torch.float32
    xd = torch.as_tensor(x, dtype=dt, device="cuda").contiguous()
    fd = torch.as_tensor(f, dtype=dt, device="cuda").contiguous()
    ud = torch.empty_like(xd)
    out = {}
    with se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, c.precision, window=c.window) as plan:
        info = plan.info()
        out["info"] = {k: getattr(info, k) for k, _ in info._fields_}
        plan.stage("sort", x=xd, f=fd)
        out["perm_near"] = plan.read(se.SE_BUF_PERM_NEAR).cpu().numpy()
        out["perm_grid"] = plan.read(se.SE_BUF_PERM_GRID).cpu().numpy()
        out["cell_start"] = plan.read(se.SE_BUF_CELL_START).cpu().numpy()
        out["bin_start"] = plan.read(se.SE_BUF_BIN_START).cpu().numpy()
        plan.stage("p2p")
        uN = plan.read(se.SE_BUF_UN).cpu().numpy()
        out["uN"] = np.empty_like(uN)
        out["uN"][out["perm_near"]] = uN
        plan.stage("p2g")
        out["H"] = plan.read(se.SE_BUF_GRID).cpu().numpy()
        plan.stage("fft")
        plan.stage("scale")
        sp = plan.read(se.SE_BUF_SPEC).cpu().numpy()
        out["Hs"] = sp[..., 0] + 1j * sp[..., 1]
        plan.stage("ifft")
        out["Ht"] = plan.read(se.SE_BUF_GRID).cpu().numpy()
        plan.stage("g2p")
        uF = plan.read(se.SE_BUF_UF).cpu().numpy().astype(np.float64)
        uF *= info.h ** 3 * info.cw
        out["uF"] = np.empty_like(uF)
        out["uF"][out["perm_grid"]] = uF
        plan.stage("sum", f=fd, u=ud)
        torch.cuda.synchronize()
        out["u"] = ud.cpu().numpy()
        # and the one-call path
        u2 = plan.eval(xd, fd)
        torch.cuda.synchronize()
        out["u_eval"] = u2.cpu().numpy()
        out["launches"] = plan.launch_count()
    return out
