"""Host logic of the slab decomposition (paper_2606_19059_b200/slabs.py) on CPU: the index arithmetic of
SlabLayout against brute force, and -- under torch.distributed with the gloo backend, world sizes 2 and 3 -- the exchanges the
multi-GPU driver is made of: the neighbour exchange, the all-to-all, the particle partition, and the slab-decomposed transform
(x-slabs -> ky-pencils -> x-slabs) against numpy's 3-D FFT, with a stand-in for K4 that multiplies every mode by a number made
from its global indices (so that a wrong pencil offset or block order fails)."""
import os
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

from paper_2606_19059_b200 import slabs

ROOT = Path(__file__).resolve().parents[1]


def test_layout_planes_and_ownership():
    L, M, P, rc, W = 1.0, 96, 24, 0.13, 4
    lay = slabs.SlabLayout(L, M, P, rc, W)
    assert (lay.Ml, lay.Mx, lay.nlo, lay.nhi) == (24, 48, 11, 12)
    cover = np.zeros(M, int)
    for r in range(W):
        g = lay.local_planes(r)
        assert g[lay.nlo] == r * lay.Ml and g[lay.nlo + lay.Ml - 1] == (r + 1) * lay.Ml - 1
        cover[g[lay.nlo:lay.nlo + lay.Ml]] += 1
        # the window of every point this rank may own fits the local planes: anchors 0 .. Ml - 1, P planes each
        assert lay.nlo + lay.Ml + lay.nhi <= lay.Mx
    assert np.all(cover == 1)                                   # every plane owned exactly once
    rng = np.random.default_rng(5)
    x0 = np.concatenate([rng.random(2000) * 3 - 1, [0.0, 0.25, 0.5, 0.75, 1.0, -1e-18]])
    own = lay.owner(x0)
    xw = x0 - np.floor(x0)
    xw[xw >= 1.0] = 0.0
    ref = (np.floor(xw / (L / M)).astype(int) % M) // lay.Ml
    assert np.array_equal(own, ref)


@pytest.mark.parametrize("W", [2, 3, 4])
def test_ghost_masks_cover_every_pair_across_a_face(W):
    """Every pair (target in slab r, source in another slab) within rc in x (periodic) has its source in the ghosts r receives,
    and no source is sent to the same rank twice."""
    L, M, P, rc = 1.0, 96, 24, 0.2
    lay = slabs.SlabLayout(L, M, P, rc, W)
    rng = np.random.default_rng(11)
    x0 = rng.random(3000)
    own = lay.owner(x0)
    for r in range(W):
        recv = []
        for s in {(r - 1) % W, (r + 1) % W}:
            mine = np.nonzero(own == s)[0]
            ml, mr = lay.ghost_masks(x0[mine], s)
            if (s - 1) % W == r:
                recv.append(mine[ml])
            if (s + 1) % W == r:
                recv.append(mine[mr])
        recv = np.concatenate(recv)
        assert len(np.unique(recv)) == len(recv)
        t = x0[own == r]
        others = np.nonzero(own != r)[0]
        d = np.abs(x0[others][:, None] - t[None, :])
        d = np.minimum(d, L - d)
        need = others[(d <= rc).any(axis=1)]
        assert np.isin(need, recv).all()


def test_layout_rejects_thin_slabs():
    for kw in (dict(M=96, P=24, rc=0.1, world=1), dict(M=96, P=24, rc=0.1, world=5), dict(M=40, P=24, rc=0.1, world=2),
               dict(M=96, P=24, rc=0.3, world=4)):
        with pytest.raises(ValueError):
            slabs.SlabLayout(1.0, kw["M"], kw["P"], kw["rc"], kw["world"])


_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from paper_2606_19059_b200 import slabs
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
r, W = dist.get_rank(), dist.get_world_size()
L, M, P, rc = 1.0, 24, 8, 0.2
lay = slabs.SlabLayout(L, M, P, rc, W)
ok = True

# neighbour exchange: rank r sends (r, 0) rows to the left and (r, 1) rows to the right, r + 1 and r + 2 of them
fl, fr = slabs._exchange(torch.full((r + 1, 2), float(r)), torch.full((r + 2, 2), float(r) + 0.5))
ok &= fl.shape[0] == (r - 1) % W + 2 and bool((fl == (r - 1) % W + 0.5).all())
ok &= fr.shape[0] == (r + 1) % W + 1 and bool((fr == float((r + 1) % W)).all())

# all-to-all: block d of rank s carries 10 s + d
got = slabs._all_to_all([torch.full((2, 3), 10.0 * r + d) for d in range(W)])
ok &= all(bool((got[s] == 10.0 * s + r).all()) for s in range(W))

# partition: every point ends on its owner, none lost, un-sort information valid
rng = np.random.default_rng(100 + r)
x = torch.as_tensor(rng.random((50 + 7 * r, 3))); f = torch.as_tensor(rng.standard_normal((50 + 7 * r, 3)))
xo, fo, (src, idx) = slabs.partition(lay, x, f)
ok &= bool((lay.owner(xo[:, 0]) == r).all())
tot = torch.tensor([xo.shape[0], x.shape[0]]); dist.all_reduce(tot)
ok &= int(tot[0]) == int(tot[1])
ok &= bool((xo[src == r] == x[idx[src == r]]).all()) and bool((fo[src == r] == f[idx[src == r]]).all())

# slab-decomposed transform against numpy: H the same random grid on every rank; K4 replaced by a multiplier w(kx, ky, kz)
H = np.random.default_rng(7).standard_normal((3, M, M, M))
kx, ky, kz = np.meshgrid(np.arange(M), np.arange(M), np.arange(M // 2 + 1), indexing="ij")
w = 1.0 + 0.01 * kx + 0.0001 * ky * ky + 0.3 * kz
ref = np.fft.irfftn(np.fft.rfftn(H, axes=(1, 2, 3)) * w, s=(M, M, M), axes=(1, 2, 3)) * M ** 3
class Tables:
    def scale_block(self, S, ky0, nky, stream=None):
        S *= torch.as_tensor(w[:, ky0:ky0 + nky])
ev = slabs.SlabEval(lay, r, xi=5.0)
ev._tables = lambda: Tables()
own = torch.as_tensor(H[:, r * lay.Ml:(r + 1) * lay.Ml].copy())
pen = slabs._all_to_all(ev.spectrum_out(own))
back = slabs._all_to_all(ev.pencil(pen))
for_left, for_right = ev.planes_back(back)
ok &= np.allclose(ev.Ht.numpy(), ref[:, r * lay.Ml:(r + 1) * lay.Ml], rtol=1e-10, atol=1e-8)
# ghost planes of G2P: what arrives from the left is the left neighbour's last P/2 - 1 planes, from the right its first P/2
gl, gr = slabs._exchange(for_left.transpose(0, 1).contiguous(), for_right.transpose(0, 1).contiguous())
lo = [(r * lay.Ml - lay.nlo + k) % M for k in range(lay.nlo)]
hi = [((r + 1) * lay.Ml + k) % M for k in range(lay.nhi)]
ok &= np.allclose(gl.transpose(0, 1).numpy(), ref[:, lo], rtol=1e-10, atol=1e-8)
ok &= np.allclose(gr.transpose(0, 1).numpy(), ref[:, hi], rtol=1e-10, atol=1e-8)
print("RESULT", r, int(ok), flush=True)
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,port", [(2, 29531), (3, 29533)])
def test_exchanges_and_decomposed_transform_gloo(tmp_path, world, port):
    script = tmp_path / "w.py"
    script.write_text(_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world))
    procs = [subprocess.Popen([sys.executable, str(script), str(ROOT)], env=dict(env, RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for r in range(world)]
    outs = [p.communicate(timeout=300)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    for o in outs:
        ln = [l for l in o.splitlines() if l.startswith("RESULT")][0].split()
        assert ln[2] == "1", outs
