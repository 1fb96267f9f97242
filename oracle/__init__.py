"""CPU oracle for the spectral Ewald Stokeslet sum -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2606_19059_b200 (the CUDA
path) and does not import it.

Two independent programs (plain C, double precision, see the headers of the .c files):
  O1  direct_ewald.c : the definition -- O(N^2) real-space sum + explicit k-space sum.
  O2  se_oracle.c    : the spectral Ewald algorithm (Alg. 2.1) stage by
                       stage; the two FFT steps are scipy.fft
                       (library primitive: pocketfft, the routine behind numpy.fft as well, here
                       with worker threads; full complex-to-complex, unnormalised forward /
                       unnormalised inverse).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): xi-independence of O1, the Hasimoto
N=1 lattice constant (tests/golden/hasimoto_sc.txt), translation invariance, linearity,
operator symmetry, length scaling, divergence-free field (finite differences), agreement
O2 <-> O1 at 1e-9 on config 1, P-convergence of O2 to O1, window normalisation and
w_hat closed form, mass conservation, discrete incompressibility, P2G/G2P adjointness,
brute-force near sum vs cell-list near sum, gather-form P2G vs scatter-form P2G.
No function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np
import scipy.fft as _fft

_HERE = Path(__file__).resolve().parent
_SRC = [_HERE / "se_oracle.c", _HERE / "direct_ewald.c"]
_lib = None


def _host_tag() -> str:
    """Short hash of this host's CPU feature flags: the library is built -march=native, and a copy
    built on another machine (the .so travels with the repo snapshot) must not be loaded here."""
    import hashlib
    flags = ""
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.startswith("flags") or ln.startswith("Features"):
                    flags = ln
                    break
    except OSError:
        pass
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


_LIB = _HERE / "_build" / f"liboracle.{_host_tag()}.so"


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc -O3 -march=native (SURVEY.md 8(d) "Oracle beside it"); floating-point
    contraction is off, so every product and sum is rounded as the source writes it."""
    newest = max(p.stat().st_mtime for p in _SRC)
    if force or not _LIB.exists() or _LIB.stat().st_mtime < newest:
        _LIB.parent.mkdir(exist_ok=True)
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        cmd = (["gcc", "-O3", "-march=native", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", str(tmp)]
               + [str(p) for p in _SRC] + ["-lm"])
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def n_threads() -> int:
    """Threads the OpenMP loops use (OMP_NUM_THREADS or all online cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


# --------------------------------------------------------------------------- O1
def direct_ewald(x, f, L, xi, targets=None, R=None, K=None):
    """Direct Ewald sum (definition).  targets=None: targets are the sources, self term added."""
    lib = _load()
    x, xp = _d(x)
    f, fp = _d(f)
    N = x.shape[0]
    if targets is None:
        t, tp, Nt, add_self = x, xp, N, 1
    else:
        t, tp = _d(targets)
        Nt, add_self = t.shape[0], 0
    R = 6.3 / xi if R is None else R
    K = 12.6 * xi if K is None else K
    u = np.zeros((Nt, 3))
    lib.de_eval(C.c_int64(Nt), tp, C.c_int64(N), xp, fp, C.c_double(L), C.c_double(xi),
                C.c_double(R), C.c_double(K), C.c_int(add_self), u.ctypes.data_as(C.POINTER(C.c_double)))
    return u


# --------------------------------------------------------------------------- O2
def params(L, xi, M, P):
    lib = _load()
    out = np.zeros(5)
    lib.se_params(C.c_double(L), C.c_double(xi), C.c_int(M), C.c_int(P), out.ctypes.data_as(C.POINTER(C.c_double)))
    return dict(h=out[0], m=out[1], eta=out[2], a=out[3], cw=out[4])


def wrap(x, L):
    lib = _load()
    x, xp = _d(x)
    xw = np.empty_like(x)
    lib.se_wrap(C.c_int64(x.shape[0]), xp, C.c_double(L), xw.ctypes.data_as(C.POINTER(C.c_double)))
    return xw


def near_brute(xw, f, L, xi, rc, targets=None):
    """u^N by the plain O(N^2 * 27) loop; `targets` = optional index array into xw."""
    lib = _load()
    xw, xp = _d(xw)
    f, fp = _d(f)
    N = xw.shape[0]
    if targets is None:
        nt, tp = N, None
    else:
        tid = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tp = tid.shape[0], tid.ctypes.data_as(C.POINTER(C.c_int64))
    u = np.zeros((nt, 3))
    lib.se_near_brute(C.c_int64(N), xp, fp, C.c_double(L), C.c_double(xi), C.c_double(rc),
                      C.c_int64(nt), tp, u.ctypes.data_as(C.POINTER(C.c_double)))
    return u


def near_targets(xw, f, xt, L, xi, rc):
    """u^N at separate (wrapped) target positions xt from the sources (xw, f): plain loop, 27 images."""
    lib = _load()
    xw, xp = _d(xw)
    f, fp = _d(f)
    xt, tp = _d(xt)
    u = np.zeros_like(xt)
    lib.se_near_targets(C.c_int64(xw.shape[0]), xp, fp, C.c_int64(xt.shape[0]), tp, C.c_double(L), C.c_double(xi),
                        C.c_double(rc), u.ctypes.data_as(C.POINTER(C.c_double)))
    return u


def near_cells(xw, f, L, xi, rc):
    lib = _load()
    xw, xp = _d(xw)
    f, fp = _d(f)
    u = np.zeros_like(xw)
    rcode = lib.se_near_cells(C.c_int64(xw.shape[0]), xp, fp, C.c_double(L), C.c_double(xi), C.c_double(rc),
                              u.ctypes.data_as(C.POINTER(C.c_double)))
    if rcode != 0:
        raise ValueError("cell list needs floor(L/rc) >= 3")
    return u


# ---- windows --------------------------------------------------------------------------------
# "gaussian": reading S4.  "kb": the truncated Kaiser-Bessel window of eq. (2.8)
# evaluated exactly; "kb_poly": its piecewise polynomial of degree nu per bin of width h
# -- the form the paper (and the CUDA path) actually evaluates.
WIN_GAUSS, WIN_KB, WIN_KBPOLY = 0, 1, 2
WINDOWS = {"gaussian": WIN_GAUSS, "kb": WIN_KB, "kb_poly": WIN_KBPOLY}


def kb_degree(P):
    """Degree nu of the piecewise polynomial (reading S19: the printed "P = 2 nu + 1", PAPER.md:103,
    contradicts the even P of every experiment and cannot reach the stated accuracies; nu = P + 3, at
    most 13, keeps the interpolation error two orders below the window's own truncation level 1/I0(beta))."""
    return min(P + 3, 13)


def kb_params(L, M, P):
    """beta = 2.5 P, a_w = P h / 2."""
    return dict(beta=2.5 * P, aw=P * (L / M) / 2.0)


def kb_window(r, beta, aw):
    """w0(r) of eq. (2.8), exact (the oracle's own I0 series)."""
    lib = _load()
    lib.se_kb_window.restype = C.c_double
    r = np.atleast_1d(np.asarray(r, dtype=np.float64))
    return np.array([lib.se_kb_window(C.c_double(v), C.c_double(beta), C.c_double(aw)) for v in r])


def kb_poly_coeffs(L, M, P, nu=None):
    """Coefficients c[l][k], l = 0..P-1, k = 0..nu: on bin l, r in [(l - P/2) h, (l - P/2 + 1) h],
    w0(r) ~ sum_k c[l][k] s^k with s = 2 (r/h - (l - P/2)) - 1 in [-1, 1]: the interpolant of degree nu
    at the nu + 1 Chebyshev points of the bin ("polynomial interpolation of degree nu",
    PAPER.md:423 "a separate polynomial in each bin of width h"), converted to monomials for Horner."""
    from numpy.polynomial import chebyshev as Ch
    nu = kb_degree(P) if nu is None else nu
    kp = kb_params(L, M, P)
    h = L / M
    out = np.empty((P, nu + 1))
    for l in range(P):
        fn = lambda s, l=l: kb_window((l - P / 2 + 0.5 * (np.asarray(s) + 1.0)) * h, kp["beta"], kp["aw"])
        out[l] = Ch.cheb2poly(Ch.chebinterpolate(fn, nu))
    return out


def kb_what(L, M, P, nquad=256):
    """w_hat0(k_i) = integral of w0(r) cos(k_i r) over (-a_w, a_w), k_i = 2 pi n_i / L, n_i = i (i < M/2) else i - M,
    by Gauss-Legendre quadrature (the integrand is entire in r inside the support)."""
    kp = kb_params(L, M, P)
    t, w = np.polynomial.legendre.leggauss(nquad)
    r = kp["aw"] * t
    w0 = kb_window(r, kp["beta"], kp["aw"])
    n = np.fft.fftfreq(M, 1.0 / M)
    k = 2.0 * np.pi * n / L
    return (np.cos(np.outer(k, r)) * (w0 * w * kp["aw"])).sum(axis=1)


def _wspec(window, L, xi, M, P):
    """(kind, parameter array, c_w, deconvolution table or None) of a window name."""
    kind = WINDOWS[window]
    if kind == WIN_GAUSS:
        pr = params(L, xi, M, P)
        return kind, np.array([pr["a"]]), pr["cw"], None
    kp = kb_params(L, M, P)
    what = kb_what(L, M, P)
    if kind == WIN_KB:
        return kind, np.array([kp["beta"], kp["aw"]]), 1.0, what
    c = kb_poly_coeffs(L, M, P)
    return kind, np.concatenate([[float(c.shape[1] - 1)], c.ravel()]), 1.0, what


def window_1d(xd, L, xi, M, P, window="gaussian"):
    """(W[P], idx[P]) of one coordinate: the window values at the P support points and their grid indices."""
    lib = _load()
    kind, wpar, _, _ = _wspec(window, L, xi, M, P)
    Wv = np.empty(P)
    idx = np.empty(P, dtype=np.int32)
    lib.se_window_1d(C.c_double(float(xd)), C.c_double(L), C.c_int(M), C.c_int(P), C.c_int(kind),
                     wpar.ctypes.data_as(C.POINTER(C.c_double)), Wv.ctypes.data_as(C.POINTER(C.c_double)),
                     idx.ctypes.data_as(C.POINTER(C.c_int)))
    return Wv, idx


def p2g(xw, f, L, xi, M, P, window="gaussian"):
    lib = _load()
    kind, wpar, cw, _ = _wspec(window, L, xi, M, P)
    xw, xp = _d(xw)
    f, fp = _d(f)
    H = np.empty((3, M, M, M))
    lib.se_p2g(C.c_int64(xw.shape[0]), xp, fp, C.c_double(L), C.c_int(M), C.c_int(P), C.c_int(kind),
               wpar.ctypes.data_as(C.POINTER(C.c_double)), C.c_double(cw), H.ctypes.data_as(C.POINTER(C.c_double)))
    return H


def p2g_points(xw, f, L, xi, M, P, gidx, window="gaussian"):
    """H at the sampled grid indices gidx (ns,3) -> (ns,3 comps), gather form, O(N) each."""
    lib = _load()
    kind, wpar, cw, _ = _wspec(window, L, xi, M, P)
    xw, xp = _d(xw)
    f, fp = _d(f)
    gi = np.ascontiguousarray(gidx, dtype=np.int32)
    out = np.zeros((gi.shape[0], 3))
    lib.se_p2g_points(C.c_int64(xw.shape[0]), xp, fp, C.c_double(L), C.c_int(M), C.c_int(P), C.c_int(kind),
                      wpar.ctypes.data_as(C.POINTER(C.c_double)), C.c_double(cw), C.c_int64(gi.shape[0]),
                      gi.ctypes.data_as(C.POINTER(C.c_int32)), out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def _what_ptr(what):
    return None if what is None else what.ctypes.data_as(C.POINTER(C.c_double))


def scale(Hhat, L, xi, M, P, window="gaussian"):
    """Scale a full c2c spectrum (3,M,M,M) complex128; returns a new array."""
    lib = _load()
    pr = params(L, xi, M, P)
    _, _, _, what = _wspec(window, L, xi, M, P)
    out = np.array(Hhat, dtype=np.complex128, order="C", copy=True)
    assert out.shape == (3, M, M, M)
    lib.se_scale(C.c_int(M), C.c_double(L), C.c_double(xi), C.c_double(pr["eta"]), _what_ptr(what),
                 out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def scale_modes(idx, vals, L, xi, M, P, window="gaussian"):
    """Scale sampled modes: idx (ns,3) int, vals (ns,3) complex -> (ns,3) complex."""
    lib = _load()
    pr = params(L, xi, M, P)
    _, _, _, what = _wspec(window, L, xi, M, P)
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    vals = np.ascontiguousarray(vals, dtype=np.complex128)
    out = np.empty_like(vals)
    for s in range(idx.shape[0]):
        lib.se_scale_mode(C.c_int(M), C.c_double(L), C.c_double(xi), C.c_double(pr["eta"]), _what_ptr(what),
                          idx[s].ctypes.data_as(C.POINTER(C.c_int)),
                          vals[s].ctypes.data_as(C.POINTER(C.c_double)),
                          out[s].ctypes.data_as(C.POINTER(C.c_double)))
    return out


def g2p(xt, Ht, L, xi, M, P, window="gaussian"):
    """u^F at (wrapped) positions xt from the real grid Ht (3,M,M,M)."""
    lib = _load()
    kind, wpar, cw, _ = _wspec(window, L, xi, M, P)
    xt, xp = _d(xt)
    Ht, hp = _d(Ht)
    assert Ht.shape == (3, M, M, M)
    u = np.zeros_like(xt)
    lib.se_g2p(C.c_int64(xt.shape[0]), xp, C.c_double(L), C.c_int(M), C.c_int(P), C.c_int(kind),
               wpar.ctypes.data_as(C.POINTER(C.c_double)), C.c_double(cw), hp, u.ctypes.data_as(C.POINTER(C.c_double)))
    return u


def se_sum(uN, uF, f, xi):
    lib = _load()
    uN, a = _d(uN)
    uF, b = _d(uF)
    f, c = _d(f)
    u = np.empty_like(uN)
    lib.se_sum(C.c_int64(uN.shape[0]), a, b, c, C.c_double(xi), u.ctypes.data_as(C.POINTER(C.c_double)))
    return u


def se_far(xw, f, L, xi, M, P, keep=False, timings=None, window="gaussian"):
    """Far field of Alg. 2.1 steps 2-6: P2G -> FFT -> CNV -> IFFT -> G2P."""
    import time
    t0 = time.perf_counter()
    H = p2g(xw, f, L, xi, M, P, window)
    t1 = time.perf_counter()
    Hhat = _fft.fftn(H, axes=(1, 2, 3), workers=n_threads())   # step 5: unnormalised forward DFT
    if not keep:
        del H
    t2 = time.perf_counter()
    Hs = scale(Hhat, L, xi, M, P, window)
    del Hhat
    t3 = time.perf_counter()
    # step 7: unnormalised inverse, real part (ifftn divides by M^3: undo it); one component at a time
    # so that the complex temporaries of a 576^3 grid are freed as they go
    Ht = np.empty((3, M, M, M))
    for c in range(3):
        Ht[c] = _fft.ifftn(Hs[c], workers=n_threads()).real
        Ht[c] *= float(M) ** 3
    if not keep:
        del Hs
    t4 = time.perf_counter()
    uF = g2p(xw, Ht, L, xi, M, P, window)
    t5 = time.perf_counter()
    if timings is not None:
        timings.update(p2g=t1 - t0, fft=t2 - t1, scale=t3 - t2, ifft=t4 - t3, g2p=t5 - t4)
    out = dict(uF=uF)
    if keep:
        out.update(H=H, Hs=Hs, Ht=Ht)
    return out


def se_eval(x, f, L, xi, rc, M, P, keep=False, near="auto", timings=None, window="gaussian"):
    """Full SE oracle.  Returns dict with u, uN, uF (+ H, Hs, Ht if keep)."""
    import time
    x = np.asarray(x, dtype=np.float64)
    f = np.asarray(f, dtype=np.float64)
    xw = wrap(x, L)
    t0 = time.perf_counter()
    if near == "brute" or (near == "auto" and int(np.floor(L / rc)) < 3):
        uN = near_brute(xw, f, L, xi, rc)
    else:
        uN = near_cells(xw, f, L, xi, rc)
    t1 = time.perf_counter()
    if timings is not None:
        timings["near"] = t1 - t0
    out = se_far(xw, f, L, xi, M, P, keep=keep, timings=timings, window=window)
    out["uN"] = uN
    out["xw"] = xw
    out["u"] = se_sum(uN, out["uF"], f, xi)
    return out


def se_eval_targets(xs, f, xt, L, xi, rc, M, P, keep=False, window="gaussian"):
    """SE oracle with separate targets (eq. (1.1)): u(x_i) = sum_j sum_p G(x_i - y_j + p) f_j at the
    targets xt; no self term.  Near: plain loop; far: the sources' grid (steps 4-7) gathered at the targets (step 8)."""
    xs = np.asarray(xs, dtype=np.float64)
    f = np.asarray(f, dtype=np.float64)
    xt = np.asarray(xt, dtype=np.float64)
    xw, tw = wrap(xs, L), wrap(xt, L)
    uN = near_targets(xw, f, tw, L, xi, rc)
    H = p2g(xw, f, L, xi, M, P, window)
    Hs = scale(_fft.fftn(H, axes=(1, 2, 3), workers=n_threads()), L, xi, M, P, window)
    Ht = np.ascontiguousarray(_fft.ifftn(Hs, axes=(1, 2, 3), workers=n_threads()).real) * float(M) ** 3
    uF = g2p(tw, Ht, L, xi, M, P, window)
    out = dict(u=uN + uF, uN=uN, uF=uF, xw=xw, tw=tw)
    if keep:
        out.update(H=H, Hs=Hs, Ht=Ht)
    return out
