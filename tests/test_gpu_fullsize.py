"""Parity at BASELINE.json's FULL sizes in the launch configuration bench.py times (no id column;
no x column in 2-d): the oracle cannot push 210 M particles in seconds, so it pushes a SAMPLE it
can compute one by one -- all particles of a 3 x 3 (x 3) block of tiles -- with the full-size E
and B, and the current it deposits must equal the GPU's J on the inner tile's nodes (J there
receives contributions from exactly those particles: a particle reaches nodes c-1 .. c+2 of its
cell c); plus properties that hold at any size."""
import numpy as np
import pytest
import torch

import psc_inputs
from tests.util import key_to_cell, library_block, oracle_for

pytestmark = pytest.mark.gpu
TOL = 1e-5


def _tile_slots(offs, tiles, cpb):
    idx = [torch.arange(int(offs[t * cpb]), int(offs[(t + 1) * cpb]), device=offs.device) for t in tiles]
    return torch.cat(idx)


@pytest.mark.parametrize("cfg", [2, 4, 5])
def test_full_size_push_matches_oracle_on_a_tile_neighbourhood(cfg):
    from paper_1310_7866_b200 import PSC_B
    from paper_1310_7866_b200.harness import Simulation

    pl = psc_inputs.make_config(cfg, device="cuda:0")
    d3 = pl.n[0] > 1
    sim = Simulation(pl, with_id=False, with_x=d3)      # bench.py's configuration
    n_p = sim.np
    del pl.y, pl.z, pl.ux, pl.uy, pl.uz, pl.qw           # the simulation owns its copies
    torch.cuda.empty_cache()
    sim.step(3)                                          # self-consistent fields, mixed cells
    assert sim.psc.status() == 0
    sim.psc.particles_sort()                             # stable physical sort: contiguous cells
    sim.psc.push_fields(PSC_B, 0.5)                      # the push sees B^{n+1/2} (Fig. 8)
    lb = library_block(pl.n)
    nb = [pl.n[d] // lb[d] for d in range(3)]
    cpb = lb[0] * lb[1] * lb[2]
    offs = sim.sort_result()[2]
    assert int(offs[-1]) == n_p
    # 3 x 3 (x 3) tiles around an inner tile away from the periodic boundary
    ctr = [min(2, nb[0] // 2) if d3 else 0, nb[1] // 2, nb[2] // 2]
    rng = lambda d: range(ctr[d] - 1, ctr[d] + 2) if pl.n[d] > 1 else range(0, 1)
    tiles = [(bz * nb[1] + by) * nb[0] + bx for bz in rng(2) for by in rng(1) for bx in rng(0)]
    slots = _tile_slots(offs, tiles, cpb)
    cur = sim.current()
    keys = sim.keys()[slots].cpu().numpy().astype(np.int64)
    cells = key_to_cell(keys, pl.n, lb)
    col = lambda c: cur[c][slots].cpu().numpy().astype(np.float64)
    pos = [np.ascontiguousarray((cells[d] + col(c)) * pl.dx[d]) if pl.n[d] > 1 else np.zeros(len(keys))
           for d, c in enumerate(("x", "y", "z"))]
    u = [np.ascontiguousarray(col(c)) for c in ("ux", "uy", "uz")]
    qw = np.ascontiguousarray(col("qw"))
    sp = np.ascontiguousarray(cur["species"][slots].cpu().numpy().astype(np.int32))
    E = np.ascontiguousarray(sim.interior(sim.E).cpu().numpy().astype(np.float64))
    B = np.ascontiguousarray(sim.interior(sim.B).cpu().numpy().astype(np.float64))
    orc = oracle_for(pl)
    J = orc.zeros_field()
    orc.push_particles(E, B, J, pos[0], pos[1], pos[2], u[0], u[1], u[2], qw, sp)

    sim.psc.push_particles()
    assert sim.psc.status() == 0
    Jg = sim.interior(sim.J)
    lo = [ctr[d] * lb[d] for d in range(3)]
    sl = tuple(slice(lo[d], lo[d] + lb[d]) for d in (2, 1, 0))
    got = Jg[(slice(None),) + sl].cpu().numpy().astype(np.float64)
    want = J[(slice(None),) + sl]
    for c in range(3):
        den = np.abs(J[c]).max()
        assert den > 0
        assert np.abs(got[c] - want[c]).max() <= TOL * den, (cfg, c)
    # properties at any size: every particle is filed under a valid cell, none lost, offsets in [0,1)
    k2 = sim.keys()
    assert int(k2.min()) >= 0 and int(k2.max()) < pl.n[0] * pl.n[1] * pl.n[2]
    cur = sim.current()
    for c in ("y", "z") + (("x",) if d3 else ()):
        assert float(cur[c].min()) >= 0.0 and float(cur[c].max()) < 1.0
    # the sampled particles themselves: momenta as per-species sums over the inner tile's cells
    inner = tiles[len(tiles) // 2]
    seg = torch.arange(int(offs[inner * cpb]), int(offs[(inner + 1) * cpb]), device=offs.device)
    m_in = np.isin(keys // cpb, [inner])
    for s_ in range(len(pl.q)):
        mg = cur["species"][seg] == s_
        mo = m_in & (sp == s_)
        if not mo.any():
            continue
        for c, uo in zip(("ux", "uy", "uz"), u):
            a = float(cur[c][seg][mg].double().sum())
            b = float(uo[mo].sum())
            scale = float(np.abs(uo[mo]).sum())
            assert abs(a - b) <= TOL * scale, (cfg, s_, c)
