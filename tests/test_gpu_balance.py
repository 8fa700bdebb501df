"""GPU parity of the patch loads (particles + cells per patch), counted by
psc_patch_loads from the cell store, against the oracle's count of the same particles; and the
whole balancing chain (loads -> Hilbert-Peano order -> Appendix A) on the Harris sheet, the
"strongly nonuniform load" of BASELINE.json's config 3."""
import numpy as np
import pytest
import torch

import paper_1310_7866_b200 as psc
import psc_inputs
from oracle import balance as ob
from tests.util import gpu_state, key_to_cell, library_block

pytestmark = pytest.mark.gpu


def _sim(pl, **kw):
    from paper_1310_7866_b200.harness import Simulation

    return Simulation(pl, **kw)


def _cases(kind):
    if kind == "2d":
        return psc_inputs.make_config(1), (1, 2, 2)
    if kind == "harris":
        return psc_inputs.make_config(3, scale=(1, 64, 128)), (1, 1, 2)
    if kind == "3d":
        return psc_inputs.thermal((16, 8, 24), 6, seed=12, name="3d"), (2, 1, 3)
    return psc_inputs.make_config(5, scale=(8, 8, 32)), (1, 2, 2)


def _loads(sim, pb):
    nb = [n // b for n, b in zip(sim.n, library_block(sim.n, (0, 0, 0)))]
    npatch = int(np.prod([a // b for a, b in zip(nb, pb)]))
    L = torch.full((npatch,), -1, dtype=torch.int64, device="cuda")
    np3 = sim.psc.patch_loads(pb, L)
    torch.cuda.synchronize()
    return np3, L.cpu().numpy()


@pytest.mark.parametrize("kind", ["2d", "harris", "3d", "beam"])
def test_patch_loads_match_oracle(kind):
    """after a few steps (residents in their cells, leavers waiting in the exchange rows of their
    source cells): every particle counts for the patch of the cell it is filed under -- exact"""
    pl, pb = _cases(kind)
    sim = _sim(pl)
    sim.step(3)
    np3, got = _loads(sim, pb)
    st = gpu_state(sim)
    block = library_block(pl.n, (0, 0, 0))
    cx, cy, cz = key_to_cell(st["key"].astype(np.int64), pl.n, block)
    pc = tuple(int(b * p) for b, p in zip(block, pb))
    assert np3 == tuple(n // c for n, c in zip(pl.n, pc))
    want = ob.patch_loads(np3, pc, cx.tolist(), cy.tolist(), cz.tolist())
    assert got.tolist() == want
    assert int(got.sum()) == pl.n_particles + int(np.prod(pl.n))
    assert sim.psc.status() == 0


def test_balance_chain_on_the_harris_sheet():
    """loads from the device, order and cut on the host: a slab decomposition of the double Harris
    sheet into equal strips is badly unbalanced, the patch-based one is not"""
    pl, _ = _cases("harris")
    sim = _sim(pl)
    sim.step(2)
    np3, L = _loads(sim, (1, 1, 1))                     # one patch per sort block: 8 x 16 patches
    order = psc.hilbert_order(np3)
    assert sorted(order) == list(range(len(L)))
    Lc = [float(L[i]) for i in order]
    ranks = 8
    N = psc.balance(Lc, [1.0] * ranks)
    assert N == ob.balance(Lc, [1.0] * ranks)
    assert sum(N) == len(L) and min(N) >= 1
    per, i = [], 0
    for n in N:
        per.append(sum(Lc[i:i + n]))
        i += n
    mean = sum(Lc) / ranks
    assert max(abs(v - mean) for v in per) / mean < 0.15
    # equal strips along z (the direction of the density gradient)
    Lz = L.reshape(np3[2], np3[1]).sum(axis=1)
    strips = Lz.reshape(ranks, -1).sum(axis=1)
    assert strips.max() / strips.min() > 1.5
    # a rank with twice the capability gets about twice the load
    cap = [1.0] * (ranks - 1) + [2.0]
    N2 = psc.balance(Lc, cap)
    assert N2 == ob.balance(Lc, cap)
    last = sum(Lc[sum(N2[:-1]):])
    assert abs(last / (sum(Lc) * 2.0 / (ranks + 1)) - 1.0) < 0.2


def test_patch_loads_argument_errors():
    pl, _ = _cases("2d")
    sim = _sim(pl)
    L = torch.zeros(64, dtype=torch.int64, device="cuda")
    with pytest.raises(psc.PscError):
        sim.psc.patch_loads((1, 1, 1), L)               # not in the internal form yet
    sim.psc.particles_sort()
    with pytest.raises(psc.PscError):
        sim.psc.patch_loads((1, 3, 1), L)               # 3 does not divide the 8 blocks
    sim.psc.patch_loads((1, 1, 1), L)
    torch.cuda.synchronize()
    assert int(L.sum().item()) == pl.n_particles + 64 * 64
