#!/usr/bin/env python3
"""Generator of csrc/se_erf_rational.h: the rational approximations p/q of erf(x)/x used by the near field (K2).

PAPER.md:429-431 (section 4): erfc(x)/x = 1/x - erf(x)/x, and erf(x)/x "is a smooth and slowly decaying function that
is suitable for rational function approximation": the AAA algorithm gives a barycentric approximant, which is converted
to p(x)/q(x) "allowing us to use 2(m-1) DFMAs and a single division".  The paper's coefficients are not printed
(reading S16), so they are regenerated here, for single precision (m = 7) and -- because K2 on B200 is bound
by shared-memory wavefronts, not by FP64 issue, so that dropping the table look-ups of erfcx pays -- for double precision
(m = 13) as well.  Choices that differ from the paper's figure 4, all stated in DESIGN.md:
  * erf(x)/x is even, so the fit is made in s = x^2 on [0, 36] (x in [0, 6], the paper's interval; beyond it
    erf(x)/x = 1/x to 2e-17), which halves the degree for the same accuracy;
  * the polynomials are written in t = s/36 in [0, 1]: the zeros and poles of these fits lie off the interval in the
    left half plane and all coefficients come out positive, so Horner evaluation has no cancellation;
  * AAA (Nakatsukasa, Sete, Trefethen 2018: greedy support points, weights = smallest right singular vector of the
    Loewner matrix) is run here in 60-digit arithmetic on 500 Chebyshev-distributed samples, and p, q are formed
    directly from the barycentric weights, p(t) = sum_j w_j f_j prod_{k != j} (t - t_k), q likewise without f_j:
    double-precision AAA stalls at 3e-15 and grows spurious pole-zero pairs beyond m = 12.

Run:  python paper_2606_19059_b200/csrc/gen_erf_rational.py   (mpmath and numpy; no GPU; about half a minute).  It
rewrites se_erf_rational.h beside itself and prints the max-error table the header carries as a comment.
"""
import os
import sys

import mpmath as mp
import numpy as np

mp.mp.dps = 60
SMAX = mp.mpf(36)
NSAMP = 500
HERE = os.path.dirname(os.path.abspath(__file__))


def f_exact(s):
    """erf(sqrt s)/sqrt s"""
    s = mp.mpf(s)
    if s == 0:
        return 2 / mp.sqrt(mp.pi)
    x = mp.sqrt(s)
    return mp.erf(x) / x


def aaa(Z, F, m):
    """m steps of AAA on the samples (Z, F): support points zs, values fs, barycentric weights w."""
    N = len(Z)
    free = [True] * N
    R = [sum(F) / N] * N
    zs, fs, w = [], [], None
    for _ in range(m):
        j = max((i for i in range(N) if free[i]), key=lambda i: abs(F[i] - R[i]))
        zs.append(Z[j]); fs.append(F[j]); free[j] = False
        idx = [i for i in range(N) if free[i]]
        A = mp.matrix(len(idx), len(zs))                       # Loewner matrix
        for a, i in enumerate(idx):
            for b in range(len(zs)):
                A[a, b] = (F[i] - fs[b]) / (Z[i] - zs[b])
        E, Q = mp.eigsy(A.T * A)                               # smallest right singular vector of A
        k = min(range(len(zs)), key=lambda q: E[q])
        w = [Q[b, k] for b in range(len(zs))]
        for i in idx:
            num = sum(w[b] * fs[b] / (Z[i] - zs[b]) for b in range(len(zs)))
            den = sum(w[b] / (Z[i] - zs[b]) for b in range(len(zs)))
            R[i] = num / den
    return zs, fs, w


def to_poly(zs, fs, w):
    """barycentric form -> monomial coefficients of p, q in t = s / SMAX, normalised to q(0) = 1"""
    m = len(zs)
    p = [mp.mpf(0)] * m
    q = [mp.mpf(0)] * m
    for j in range(m):
        c = [mp.mpf(1)]
        for k in range(m):
            if k == j:
                continue
            rt = zs[k] / SMAX
            c = [mp.mpf(0)] + c
            for i in range(len(c) - 1):
                c[i] -= rt * c[i + 1]
        for i in range(m):
            p[i] += w[j] * fs[j] * c[i]
            q[i] += w[j] * c[i]
    q0 = q[0]
    return [v / q0 for v in p], [v / q0 for v in q]


def horner(c, t, dtype):
    acc = dtype(c[-1])
    for v in c[-2::-1]:
        acc = dtype(acc * t + dtype(v))
    return acc


def max_errors(pc, qc, n=4001):
    """max |p/q - erf(x)/x| over a grid of t: in exact arithmetic, float32 Horner + division, float64 Horner + division"""
    pcf, qcf = [float(v) for v in pc], [float(v) for v in qc]
    e_exact = e32 = e64 = 0.0
    for i in range(n):
        t = mp.mpf(i) / (n - 1)
        ref = f_exact(t * SMAX)
        pe = sum(c * t ** k for k, c in enumerate(pc))
        qe = sum(c * t ** k for k, c in enumerate(qc))
        e_exact = max(e_exact, abs(float(pe / qe - ref)))
        t32, t64 = np.float32(float(t)), np.float64(float(t))
        v32 = np.float32(horner(pcf, t32, np.float32)) / np.float32(horner(qcf, t32, np.float32))
        v64 = horner(pcf, t64, np.float64) / horner(qcf, t64, np.float64)
        e32 = max(e32, abs(float(v32) - float(ref)))
        e64 = max(e64, float(abs(mp.mpf(float(v64)) - ref)))
    return e_exact, e32, e64


def main():
    Z = [SMAX * (1 - mp.cos(mp.pi * i / (NSAMP - 1))) / 2 for i in range(NSAMP)]
    F = [f_exact(z) for z in Z]
    rows, keep = [], {}
    for m in (5, 6, 7, 8, 10, 11, 12, 13, 14):
        zs, fs, w = aaa(Z, F, m)
        pc, qc = to_poly(zs, fs, w)
        ee, e32, e64 = max_errors(pc, qc)
        positive = min(pc) > 0 and min(qc) > 0
        rows.append((m, ee, e32, e64, positive))
        keep[m] = (pc, qc)
    table = ["   m  degree  exact arithmetic  float32 Horner  float64 Horner  all coefficients > 0"]
    for m, ee, e32, e64, pos in rows:
        table.append(f"  {m:2d}  {m - 1:2d}      {ee:.2e}          {e32:.2e}        {e64:.2e}        {'yes' if pos else 'NO'}")
    print("\n".join(table))
    (p32, q32), (p64, q64) = keep[7], keep[13]
    assert min(p32) > 0 and min(q32) > 0 and min(p64) > 0 and min(q64) > 0
    fmt = lambda c: ", ".join(mp.nstr(v, 25) for v in c)
    lines = [
        "// GENERATED by gen_erf_rational.py (beside this file) -- do not edit.",
        "// erf(x)/x ~ p(t)/q(t), t = x^2/36, for x^2 in [0, 36] (PAPER.md:429-431; DESIGN.md reading S16): AAA on",
        "// erf(sqrt s)/sqrt s, s in [0, 36], converted to polynomial form with q(0) = 1; m = 7 support points (degree 6",
        "// over 6) for single precision, m = 13 (degree 12 over 12) for double.  Max |p/q - erf(x)/x| (the function is",
        "// <= 1.13) of the generator run that wrote this file:",
    ] + ["//" + r for r in table] + [
        "#pragma once",
        "#define SE_ERFR_DEG_F32 6",
        "#define SE_ERFR_DEG_F64 12",
        "static const double se_erfr_p32[SE_ERFR_DEG_F32 + 1] = {" + fmt(p32) + "};",
        "static const double se_erfr_q32[SE_ERFR_DEG_F32 + 1] = {" + fmt(q32) + "};",
        "static const double se_erfr_p64[SE_ERFR_DEG_F64 + 1] = {" + fmt(p64) + "};",
        "static const double se_erfr_q64[SE_ERFR_DEG_F64 + 1] = {" + fmt(q64) + "};",
        "",
    ]
    with open(os.path.join(HERE, "se_erf_rational.h"), "w") as fh:
        fh.write("\n".join(lines))


if __name__ == "__main__":
    sys.exit(main())
