"""CPU oracle for the spectral Ewald Stokeslet sum -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2606_19059_b200 (the CUDA
path) and does not import it.

Two independent programs (plain C, double precision, see the headers of the .c files):
  O1  direct_ewald.c : the definition -- O(N^2) real-space sum + explicit k-space sum.
  O2  se_oracle.c    : the spectral Ewald algorithm (Alg. 2.1) stage by
                       stage; the two FFT steps are numpy.fft
                       (library primitive, full complex-to-complex, unnormalised forward /
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

_HERE = Path(__file__).resolve().parent
_SRC = [_HERE / "se_oracle.c", _HERE / "direct_ewald.c"]
_LIB = _HERE / "_build" / "liboracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (no -march=native: the .so travels to other hosts)."""
    newest = max(p.stat().st_mtime for p in _SRC)
    if force or not _LIB.exists() or _LIB.stat().st_mtime < newest:
        _LIB.parent.mkdir(exist_ok=True)
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", str(tmp)] + [str(p) for p in _SRC] + ["-lm"]
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


def p2g(xw, f, L, xi, M, P):
    lib = _load()
    pr = params(L, xi, M, P)
    xw, xp = _d(xw)
    f, fp = _d(f)
    H = np.empty((3, M, M, M))
    lib.se_p2g(C.c_int64(xw.shape[0]), xp, fp, C.c_double(L), C.c_int(M), C.c_int(P),
               C.c_double(pr["a"]), C.c_double(pr["cw"]), H.ctypes.data_as(C.POINTER(C.c_double)))
    return H


def p2g_points(xw, f, L, xi, M, P, gidx):
    """H at the sampled grid indices gidx (ns,3) -> (ns,3 comps), gather form, O(N) each."""
    lib = _load()
    pr = params(L, xi, M, P)
    xw, xp = _d(xw)
    f, fp = _d(f)
    gi = np.ascontiguousarray(gidx, dtype=np.int32)
    out = np.zeros((gi.shape[0], 3))
    lib.se_p2g_points(C.c_int64(xw.shape[0]), xp, fp, C.c_double(L), C.c_int(M), C.c_int(P),
                      C.c_double(pr["a"]), C.c_double(pr["cw"]), C.c_int64(gi.shape[0]),
                      gi.ctypes.data_as(C.POINTER(C.c_int32)), out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def scale(Hhat, L, xi, M, P):
    """Scale a full c2c spectrum (3,M,M,M) complex128; returns a new array."""
    lib = _load()
    pr = params(L, xi, M, P)
    out = np.array(Hhat, dtype=np.complex128, order="C", copy=True)
    assert out.shape == (3, M, M, M)
    lib.se_scale(C.c_int(M), C.c_double(L), C.c_double(xi), C.c_double(pr["eta"]),
                 out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def scale_modes(idx, vals, L, xi, M, P):
    """Scale sampled modes: idx (ns,3) int, vals (ns,3) complex -> (ns,3) complex."""
    lib = _load()
    pr = params(L, xi, M, P)
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    vals = np.ascontiguousarray(vals, dtype=np.complex128)
    out = np.empty_like(vals)
    for s in range(idx.shape[0]):
        lib.se_scale_mode(C.c_int(M), C.c_double(L), C.c_double(xi), C.c_double(pr["eta"]),
                          idx[s].ctypes.data_as(C.POINTER(C.c_int)),
                          vals[s].ctypes.data_as(C.POINTER(C.c_double)),
                          out[s].ctypes.data_as(C.POINTER(C.c_double)))
    return out


def g2p(xt, Ht, L, xi, M, P):
    """u^F at (wrapped) positions xt from the real grid Ht (3,M,M,M)."""
    lib = _load()
    pr = params(L, xi, M, P)
    xt, xp = _d(xt)
    Ht, hp = _d(Ht)
    assert Ht.shape == (3, M, M, M)
    u = np.zeros_like(xt)
    lib.se_g2p(C.c_int64(xt.shape[0]), xp, C.c_double(L), C.c_int(M), C.c_int(P),
               C.c_double(pr["a"]), C.c_double(pr["cw"]), hp, u.ctypes.data_as(C.POINTER(C.c_double)))
    return u


def se_sum(uN, uF, f, xi):
    lib = _load()
    uN, a = _d(uN)
    uF, b = _d(uF)
    f, c = _d(f)
    u = np.empty_like(uN)
    lib.se_sum(C.c_int64(uN.shape[0]), a, b, c, C.c_double(xi), u.ctypes.data_as(C.POINTER(C.c_double)))
    return u


def se_far(xw, f, L, xi, M, P, keep=False, timings=None):
    """Far field of Alg. 2.1 steps 2-6: P2G -> FFT -> CNV -> IFFT -> G2P."""
    import time
    t0 = time.perf_counter()
    H = p2g(xw, f, L, xi, M, P)
    t1 = time.perf_counter()
    Hhat = np.fft.fftn(H, axes=(1, 2, 3))                 # step 5: unnormalised forward DFT
    t2 = time.perf_counter()
    Hs = scale(Hhat, L, xi, M, P)
    del Hhat
    t3 = time.perf_counter()
    # step 7: unnormalised inverse, real part (numpy's ifftn divides by M^3: undo it)
    Ht = np.ascontiguousarray(np.fft.ifftn(Hs, axes=(1, 2, 3)).real) * float(M) ** 3
    t4 = time.perf_counter()
    uF = g2p(xw, Ht, L, xi, M, P)
    t5 = time.perf_counter()
    if timings is not None:
        timings.update(p2g=t1 - t0, fft=t2 - t1, scale=t3 - t2, ifft=t4 - t3, g2p=t5 - t4)
    out = dict(uF=uF)
    if keep:
        out.update(H=H, Hs=Hs, Ht=Ht)
    return out


def se_eval(x, f, L, xi, rc, M, P, keep=False, near="auto", timings=None):
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
    out = se_far(xw, f, L, xi, M, P, keep=keep, timings=timings)
    out["uN"] = uN
    out["xw"] = xw
    out["u"] = se_sum(uN, out["uF"], f, xi)
    return out
