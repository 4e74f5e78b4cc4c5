"""NEXT-4: one QR-CTMRG iteration sharded over the column index m of Q.

* CPU (gloo, world_size 2): the exchange step -- all-gather of the T' row blocks (or sum for a ragged split) and
  all-reduce of the partial C' -- assembles on every rank exactly what a single process holds.
* GPU (one device): the sharded kernels.  The shards of nranks = 1..5 "virtual ranks" are computed one after the
  other on the same device, assembled on the host the way the exchange does, and compared with the unsharded step
  and with the oracle.  (Ranks do not wait on one another, so this is not a stand-in for a multi-GPU run.)"""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _slices(chi, nranks):
    q, r = divmod(chi, nranks)
    out, m0 = [], 0
    for k in range(nranks):
        m1 = m0 + q + (1 if k < r else 0)
        out.append((m0, m1)); m0 = m1
    return out


def _exchange_worker(rank, world, port, chi, b, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2505_00494_b200.binding import shard_exchange
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    g = np.random.default_rng(99)                       # same stream on every rank
    T_full = g.standard_normal((chi, b * chi))
    C_parts = g.standard_normal((world, chi, chi))
    m0, m1 = _slices(chi, world)[rank]
    Tn = np.zeros_like(T_full); Tn[m0:m1] = T_full[m0:m1]
    Tn = torch.from_numpy(Tn); Cn = torch.from_numpy(C_parts[rank].copy())
    shard_exchange(Cn, Tn, rank, world)
    ok = np.array_equal(Tn.numpy(), T_full) and np.allclose(Cn.numpy(), C_parts.sum(0), rtol=0, atol=1e-14)
    open(f"{out}.{rank}", "w").write("ok" if ok else "bad")
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("chi,port", [(8, 29641), (7, 29643)])      # equal slices: all-gather; ragged: sum
def test_shard_exchange_gloo_world2(tmp_path, chi, port):
    out = str(tmp_path / "ex")
    mp.spawn(_exchange_worker, args=(2, port, chi, 4, out), nprocs=2, join=True)
    assert [open(f"{out}.{r}").read() for r in (0, 1)] == ["ok", "ok"]


def test_shard_range_partitions_every_m():
    import paper_2505_00494_b200 as pkg
    for chi in (1, 7, 8, 196):
        for nranks in (1, 2, 3, 5, 8, 9):
            got = [pkg.shard_range(chi, r, nranks) for r in range(nranks)]
            assert got == _slices(chi, nranks)
            assert got[0][0] == 0 and got[-1][1] == chi
    with pytest.raises(pkg.QrctmError):
        pkg.shard_range(8, 2, 2)


# ------------------------------------------------------------------ GPU
def rel(x, y):
    return np.linalg.norm(np.asarray(x) - np.asarray(y)) / np.linalg.norm(np.asarray(y))


@pytest.mark.gpu
@pytest.mark.parametrize("d,D,chi,seed", [(2, 2, 8, 0), (2, 3, 36, 1), (2, 3, 7, 8), (2, 4, 64, 2), (2, 5, 100, 3)])
@pytest.mark.parametrize("nranks", [1, 2, 3, 5])
def test_sharded_step_equals_unsharded_and_oracle(d, D, chi, seed, nranks):
    import paper_2505_00494_b200 as pkg
    from paper_2505_00494_b200 import build as bld
    from oracle import ctmrg as o
    from qrctm_inputs import gen_config
    bld.build()
    A, C0, T0 = gen_config(d, D, chi, seed)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A); h.set_env(C0, T0)
    Csum, Tsum = None, None
    for r in range(nranks):
        h.shard_front(r, nranks)
        Cn, Tn = h.shard_buffers()
        h.synchronize()
        Cn, Tn = Cn.cpu().numpy().copy(), Tn.cpu().numpy().copy()
        m0, m1 = pkg.shard_range(chi, r, nranks)
        assert not Tn[:m0].any() and not Tn[m1:].any()          # zeros outside this rank's rows
        Csum = Cn if Csum is None else Csum + Cn
        Tsum = Tn if Tsum is None else Tsum + Tn
    # what the exchange leaves in every rank's buffers
    import torch
    Cd, Td = h.shard_buffers()
    with torch.cuda.stream(h.stream):
        Cd.copy_(torch.from_numpy(Csum)); Td.copy_(torch.from_numpy(Tsum))
    h.shard_finish()
    C, T = h.get_env()
    h.close()
    h2 = pkg.QRCTM(d, D, chi)
    h2.set_A(A); h2.set_env(C0, T0)
    h2.step()
    Cu, Tu = h2.get_env()
    Cnu, Tnu = h2.get_raw()
    h2.close()
    assert rel(Tsum.reshape(Tnu.shape), Tnu) < 1e-13 and rel(Csum, Cnu) < 1e-12
    assert rel(C, Cu) < 1e-12 and rel(T, Tu) < 1e-13
    a = o.build_a(A)
    s = o.qr_step(*o.normalize(C0, T0), a)
    Co, To = o.normalize(s["Cn"], s["Tn"])
    assert rel(C, Co) < 1e-11 and rel(T, To) < 1e-11


@pytest.mark.gpu
def test_shard_step_single_rank_is_an_ordinary_step():
    import paper_2505_00494_b200 as pkg
    from qrctm_inputs import gen_config
    A, C0, T0 = gen_config(2, 3, 36, 1)
    h = pkg.QRCTM(2, 3, 36)
    h.set_A(A); h.set_env(C0, T0)
    for _ in range(3):
        h.shard_step(0, 1)
    C, T = h.get_env()
    h.set_env(C0, T0)
    for _ in range(3):
        h.step()
    Cu, Tu = h.get_env()
    h.close()
    assert rel(C, Cu) < 1e-12 and rel(T, Tu) < 1e-12
