"""The re-balancing step of PAPER.md:297-335 across PROCESSES, on CPU with gloo, world_size 2: every
rank measures the loads of the patches it owns, the loads are gathered, every rank runs the same
Appendix A on them (psc_balance, host code of the library), the owners before and after are
compared (psc_balance_owners), and the patches that change rank are sent to their new owner.  No
GPU and no NCCL are involved: this is the host-side logic a multi-GPU run would use, with the
patch payload standing in for a patch's particles and fields."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _patch_load(py, pz, npy):
    """synthetic load of a patch: a density ridge along the diagonal + its cells"""
    d = abs(py - pz) / npy
    return 64 + int(round(6400 * (0.1 + 0.9 * (1.0 - min(1.0, d / 0.2)) ** 2)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import paper_1310_7866_b200 as psc
    from oracle import balance as ob

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    np3 = (1, 8, 8)
    order = psc.hilbert_order(np3)                       # row-major index of the i-th patch on the curve
    npatch = len(order)
    # before: the curve cut into equal halves; a patch's payload = `load` copies of its curve index
    owner_old = psc.balance_owners([npatch // world] * world)
    mine = {}
    for i, o in enumerate(owner_old):
        if o == rank:
            p = order[i]
            mine[i] = torch.full((_patch_load(p % 8, p // 8, 8),), i, dtype=torch.int32)
    # every rank contributes the loads of ITS patches; all ranks end up with the whole array
    loads = torch.zeros(npatch, dtype=torch.float64)
    for i, t in mine.items():
        loads[i] = float(t.numel())
    dist.all_reduce(loads)
    L = loads.tolist()
    count = psc.balance(L, [1.0] * world)
    assert count == ob.balance(L, [1.0] * world)
    owner_new = psc.balance_owners(count)
    assert owner_new == ob.owners(count)
    # the patches that change rank, in curve order on both sides: sends are posted first
    reqs = []
    for i in range(npatch):
        if owner_old[i] == rank and owner_new[i] != rank:
            reqs.append(dist.isend(mine[i], dst=owner_new[i], tag=i))
    for i in range(npatch):
        if owner_new[i] == rank and owner_old[i] != rank:
            buf = torch.empty(int(L[i]), dtype=torch.int32)
            dist.recv(buf, src=owner_old[i], tag=i)
            mine[i] = buf
    for r in reqs:
        r.wait()
    for i in range(npatch):
        if owner_old[i] == rank and owner_new[i] != rank:
            del mine[i]
    ok = sorted(mine) == [i for i in range(npatch) if owner_new[i] == rank]
    ok = ok and all(int(t[0]) == i and t.numel() == int(L[i]) and bool((t == i).all()) for i, t in mine.items())
    out[rank] = (ok, sum(t.numel() for t in mine.values()), sum(L), len(mine), sum(1 for a, b in zip(owner_old, owner_new) if a != b))
    dist.barrier()
    dist.destroy_process_group()


def test_rebalance_moves_patches_between_two_ranks():
    world = 2
    port = 31000 + os.getpid() % 2000
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    total = res[0][2]
    assert all(res[r][0] for r in range(world))              # every rank holds exactly its new patches, intact
    assert res[0][1] + res[1][1] == total                    # no load lost or duplicated
    assert res[0][3] + res[1][3] == 64
    assert abs(res[0][1] - total / 2) / (total / 2) < 0.10   # balanced to within 10 % of the mean
    assert res[0][4] == res[1][4]                            # both ranks derived the same plan
