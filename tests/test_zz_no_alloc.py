"""se_scale_noalloc (include/se.h): K4 (eq. (2.6)) without a plan and without any allocation, its multiplier table
in a fixed static device array of the library.  Compared with the existing path (se_scale_block on a plan with the same
parameters, whose table is built on the host in long double) on two calls in a row with DIFFERENT parameters, so that a
table left over from the previous call would show; plus the size limit and a check that the device's free memory does not
move across the calls.  Named test_zz_* so that pytest collects it last (the suite runs with pytest -x)."""
import ctypes as C

import pytest

from gpu_util import gate
from test_gpu_parity import TOL

pytestmark = pytest.mark.gpu


def _case(se, torch, prec, M, P, L, xi, ky0, nky, seed):
    rdt = torch.float64 if prec == "fp64" else torch.float32
    g = torch.Generator(device="cuda").manual_seed(seed)
    spec = torch.view_as_complex(torch.randn(3, M, nky, M // 2 + 1, 2, dtype=rdt, device="cuda", generator=g))
    ref = spec.clone()
    with se.Plan(1000, L, xi, 0.9 * L / 3, M, P, prec) as plan:          # existing path: the plan's own table
        plan.scale_block(ref, ky0, nky)
    return spec, ref


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_scale_noalloc_matches_scale_block_twice_in_a_row(prec):
    import torch
    import paper_2606_19059_b200 as se
    tol = TOL[prec]["Hs"]
    cases = [dict(M=60, P=12, L=1.0, xi=9.0, ky0=0, nky=60, seed=1), dict(M=98, P=8, L=2.5, xi=5.5, ky0=17, nky=30, seed=2)]
    data = [_case(se, torch, prec, **c) for c in cases]
    torch.cuda.synchronize()
    # warm-up call: the first call on a device looks up the array's address (and may load the module lazily)
    se.scale_noalloc(data[0][0].clone(), cases[0]["M"], cases[0]["P"], cases[0]["L"], cases[0]["xi"], prec)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    outs = []
    for c, (spec, _) in zip(cases, data):                                 # two calls in a row on one stream, no sync between
        outs.append(se.scale_noalloc(spec, c["M"], c["P"], c["L"], c["xi"], prec, c["ky0"], c["nky"]))
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                          # nothing was allocated (or freed) on the device
    for i, (out, (_, ref)) in enumerate(zip(outs, data)):
        a = torch.view_as_real(out).cpu().numpy()
        b = torch.view_as_real(ref).cpu().numpy()
        e = gate(f"scale_noalloc call {i}", a, b, tol)
        print(f"{prec} call {i}: rel-L2 {e[0]:.2e} max-abs {e[1]:.2e}")
        assert abs(b).max() > 0
    # k = 0 and the Nyquist planes are zero (readings S2, S8), as on the plan's path
    M = cases[0]["M"]
    o = outs[0]
    assert torch.all(o[:, 0, 0, 0] == 0) and torch.all(o[:, M // 2] == 0) and torch.all(o[:, :, M // 2] == 0)
    assert torch.all(o[..., M // 2] == 0)


def test_scale_noalloc_rejects_what_does_not_fit():
    import torch
    import paper_2606_19059_b200 as se
    L = se.lib()
    buf = torch.zeros(1024, dtype=torch.float64, device="cuda")
    ptr, s0 = C.c_void_p(buf.data_ptr()), C.c_void_p(0)
    assert L.se_scale_noalloc(ptr, 4098, 12, 1.0, 9.0, 0, 0, 1, s0) == 5          # SE_ELIMIT: M beyond the fixed array
    assert b"capacity" in L.se_strerror(5)
    for args in [(None, 60, 12, 1.0, 9.0, 0, 0, 1), (ptr, 61, 12, 1.0, 9.0, 0, 0, 1), (ptr, 60, 12, 0.0, 9.0, 0, 0, 1),
                 (ptr, 60, 12, 1.0, 9.0, 0, 50, 11), (ptr, 60, 12, 1.0, 9.0, 7, 0, 1), (ptr, 60, 62, 1.0, 9.0, 0, 0, 1)]:
        assert L.se_scale_noalloc(*args, s0) == 1                                  # SE_EINVAL
    torch.cuda.synchronize()
    assert torch.all(buf == 0)
