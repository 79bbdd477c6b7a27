"""Host logic of the slab-decomposed step (include/wdm_dist.h), on CPU: exported symbols, the pack / unpack index maps of
the four exchanges against a global field in numpy, and the same maps between two real processes over gloo."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def wd():
    from paper_2606_25026_b200 import build
    build.build()
    import paper_2606_25026_b200.dist as wd
    wd._lib()
    return wd


def test_exports_every_symbol_of_wdm_dist_h(wd):
    header = open(os.path.join(ROOT, "include", "wdm_dist.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(wdm_dist_[a-z_0-9]+)\s*\(", header))
    assert declared == set(wd.EXPORTS)
    for name in declared:
        assert hasattr(wd._lib(), name)
    # argument validation without a GPU
    with pytest.raises(Exception):
        wd.wdm_dist_copy_plan(64, 3, 0)          # world must divide N


def apply_plan(plan, src_lines, dst_lines):
    """the copy kernel in numpy: lines are rows of a 2-D array"""
    n0, n1, n2, s0, s1, s2, d0, d1, d2, kmul, ksel, klim = plan
    for i0 in range(n0):
        for i1 in range(n1):
            for i2 in range(n2):
                if kmul > 0 and i0 * kmul + (i1 if ksel == 1 else i2) >= klim:
                    continue
                dst_lines[i0 * d0 + i1 * d1 + i2 * d2] = src_lines[i0 * s0 + i1 * s1 + i2 * s2]


def exchange(sends, nlines_per_peer):
    """all-to-all of equal blocks between the emulated ranks"""
    P = len(sends)
    recvs = [np.zeros_like(s) for s in sends]
    for d in range(P):
        for s in range(P):
            recvs[d][s * nlines_per_peer:(s + 1) * nlines_per_peer] = sends[s][d * nlines_per_peer:(d + 1) * nlines_per_peer]
    return recvs


@pytest.mark.parametrize("N,P", [(8, 1), (8, 2), (16, 4), (16, 8), (32, 4)])
def test_copy_plans_transpose_a_global_field(wd, N, P):
    xl, NH = N // P, N // 2 + 1
    kxb = -(-NH // P)
    rng = np.random.default_rng(N * 10 + P)
    psi = rng.normal(size=(N, N, N))                      # [x][y][z]
    H = rng.normal(size=(NH, N, N))                       # [kx][y][z]
    blk_psi, blk_h = xl * xl, xl * kxb

    def roundtrip(op_pack, op_unpack, src_of_rank, nlines_block, dst_shape):
        sends = []
        for r in range(P):
            s = np.full((P * nlines_block, N), np.nan)
            apply_plan(wd.wdm_dist_copy_plan(N, P, op_pack), src_of_rank(r).reshape(-1, N), s)
            sends.append(s)
        recvs = exchange(sends, nlines_block)
        out = []
        for r in range(P):
            dflat = np.full((int(np.prod(dst_shape[:-1])), N), np.nan)
            apply_plan(wd.wdm_dist_copy_plan(N, P, op_unpack), recvs[r], dflat)
            out.append(dflat.reshape(dst_shape))
        return out

    psiT = lambda r: np.ascontiguousarray(psi[:, r * xl:(r + 1) * xl, :].transpose(1, 0, 2))     # [y_l][x][z]
    psiX = lambda r: np.ascontiguousarray(psi[r * xl:(r + 1) * xl])                               # [x_l][y][z]
    got = roundtrip(0, 1, psiT, blk_psi, (xl, N, N))
    for r in range(P):
        assert np.array_equal(got[r], psiX(r))
    got = roundtrip(2, 3, psiX, blk_psi, (xl, N, N))
    for r in range(P):
        assert np.array_equal(got[r], psiT(r))
    HT = lambda r: np.ascontiguousarray(H[:, r * xl:(r + 1) * xl, :].transpose(1, 0, 2))         # [y_l][kx][z]
    got = roundtrip(4, 5, HT, blk_h, (kxb, N, N))
    for r in range(P):
        nkx = max(0, min(kxb, NH - r * kxb))
        assert np.array_equal(got[r][:nkx], H[r * kxb:r * kxb + nkx])
    HK = lambda r: np.concatenate([H[r * kxb:min(NH, (r + 1) * kxb)], np.zeros((kxb - max(0, min(kxb, NH - r * kxb)), N, N))])
    got = roundtrip(6, 7, HK, blk_h, (xl, NH, N))
    for r in range(P):
        assert np.array_equal(got[r], HT(r))


_WORKER = r'''
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
sys.path.insert(0, os.path.join(sys.argv[1], "tests"))
import paper_2606_25026_b200.dist as wd
from test_dist_maps import apply_plan
dist.init_process_group("gloo")
r, P = dist.get_rank(), dist.get_world_size()
N = 16
xl, NH = N // P, N // 2 + 1
rng = np.random.default_rng(5)
psi = rng.normal(size=(N, N, N))                          # every rank builds the same global field
mine_T = np.ascontiguousarray(psi[:, r * xl:(r + 1) * xl, :].transpose(1, 0, 2))
send = np.zeros((P * xl * xl, N))
apply_plan(wd.wdm_dist_copy_plan(N, P, 0), mine_T.reshape(-1, N), send)
st = torch.from_numpy(send)
rt = torch.zeros_like(st)
blk = xl * xl
reqs = []
for peer in range(P):                                      # all-to-all of equal blocks by point-to-point calls
    if peer == r:
        rt[r * blk:(r + 1) * blk] = st[r * blk:(r + 1) * blk]
    else:
        reqs.append(dist.isend(st[peer * blk:(peer + 1) * blk].contiguous(), peer))
        reqs.append(dist.irecv(rt[peer * blk:(peer + 1) * blk], peer))
for q in reqs:
    q.wait()
out = np.zeros((xl * N, N))
apply_plan(wd.wdm_dist_copy_plan(N, P, 1), rt.numpy(), out)
assert np.array_equal(out.reshape(xl, N, N), psi[r * xl:(r + 1) * xl]), "rank %d: wrong x-slab" % r
dist.barrier()
dist.destroy_process_group()
print("rank", r, "ok")
'''


def test_exchange_between_two_processes_over_gloo(wd, tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29631", str(script), ROOT]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rank 0 ok" in r.stdout and "rank 1 ok" in r.stdout
