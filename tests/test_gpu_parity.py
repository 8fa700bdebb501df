"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element on
the same seeded inputs.  Tolerances are BASELINE.json's north_star: sort results bit-exact;
positions, momenta within 1e-5 relative; J and fields within 1e-5 of the component max-norm;
continuity residual at fp32 rounding level (<= 1e-5 relative)."""
import numpy as np
import pytest
import torch

import psc_inputs
from tests.util import (gpu_cols, gpu_positions_f64, gpu_state, key_to_cell, library_block, oracle_for, oracle_sorted_state,
                        oracle_state, order_by_id, periodic_dist, positions_f64, rel_fieldnorm, rel_maxnorm, smooth_fields)

pytestmark = pytest.mark.gpu

TOL = 1e-5


def _sim(pl, block=(0, 0, 0), **kw):
    from paper_1310_7866_b200.harness import Simulation

    return Simulation(pl, block=block, **kw)


def _small(kind):
    if kind == "2d":
        return psc_inputs.make_config(1)                        # 1x64x64, 32/cell: config 1 itself
    if kind == "2d-ragged":
        return psc_inputs.thermal((1, 24, 40), 7, seed=11, name="ragged2d")
    if kind == "3d":
        return psc_inputs.make_config(4, scale=(16, 16, 16))    # 50+50 per cell
    if kind == "3d-ragged":
        return psc_inputs.thermal((12, 20, 8), 5, seed=12, name="ragged3d")
    if kind == "harris":
        return psc_inputs.make_config(3, scale=(1, 32, 128))
    if kind == "beam":                                          # config 5 recipe, order 2, 80/cell
        return psc_inputs.make_config(5, scale=(8, 8, 32))
    if kind == "3d-ragged-o2":
        return psc_inputs.thermal((12, 20, 8), 5, seed=13, order=2, name="ragged3d-o2")
    if kind == "2d-o2":                                         # order 2 in the yz plane (NEXT #2)
        return psc_inputs.thermal((1, 24, 40), 9, seed=14, order=2, name="ragged2d-o2")
    if kind in ("2d-aniso", "2d-aniso-o2", "3d-aniso", "3d-aniso-o2"):
        # anisotropic cells (dx != dy != dz != 1), four species, per-particle random weights
        d3 = kind.startswith("3d")
        pl = psc_inputs.thermal((12, 20, 8) if d3 else (1, 24, 40), 5 if d3 else 7,
                                dx=(0.8, 1.25, 0.5) if d3 else (1.0, 0.5, 2.0), seed=31 + d3,
                                order=2 if kind.endswith("o2") else 1, name=kind)
        g = torch.Generator().manual_seed(77)
        n = pl.qw.numel()
        pl.qw = (pl.qw * (0.5 + torch.rand(n, generator=g))).float()
        pl.q = list(pl.q) + [-2.0, 3.0]
        pl.m = list(pl.m) + [4.0, 50.0]
        flip = torch.rand(n, generator=g) < 0.3        # a third of the particles become species 2 / 3
        pl.species = torch.where(flip, pl.species + 2, pl.species).to(torch.int32)
        return pl
    raise ValueError(kind)


# ------------------------------------------------------------------------------------------------
# fields

@pytest.mark.parametrize("n", [(1, 24, 40), (12, 20, 8), (1, 64, 64)])
def test_fdtd_matches_oracle(n):
    pl = psc_inputs.thermal(n, 1, seed=3)
    smooth_fields(pl, 0.3, seed=5)
    sim = _sim(pl)
    orc = oracle_for(pl)
    _, E, B = oracle_state(pl)
    rng = np.random.default_rng(9)
    Jn = rng.normal(size=E.shape)
    sim.interior(sim.J).copy_(torch.from_numpy(Jn.astype(np.float32)).cuda())
    Jn = Jn.astype(np.float32).astype(np.float64)
    sim.psc.fill_ghosts(2)
    for _ in range(5):
        sim.psc.push_fields(1, 0.5)
        sim.psc.push_fields(1, 0.5)
        sim.psc.push_fields(0, 1.0)
        orc.push_b(E, B, 0.5)
        orc.push_b(E, B, 0.5)
        orc.push_e(E, B, Jn, 1.0)
    assert rel_maxnorm(sim.interior(sim.E).cpu().numpy(), E) < TOL
    # B: the Harris sheet has |B_y| ~ 0.06 next to self-generated B_x, B_z ~ 1e-4 whose fp32
    # round-off (ulp of the E and B_y they are differenced from) is ~1e-9 absolute; the bar is the
    # north_star's "relative to the field's max-norm", the per-component figure is 10x looser
    assert rel_fieldnorm(sim.interior(sim.B).cpu().numpy(), B) < TOL
    assert rel_maxnorm(sim.interior(sim.B).cpu().numpy(), B) < 10 * TOL
    # ghost points are bit-identical periodic images of the interior
    for F in (sim.E, sim.B):
        G = F.clone()
        sim.psc.bind_fields(G, sim.B, sim.J)
        sim.psc.fill_ghosts(0)
        sim.psc.bind_fields(sim.E, sim.B, sim.J)
        assert torch.equal(G, F)


@pytest.mark.parametrize("n", [(1, 8, 12), (4, 8, 12), (1, 4, 4)])
def test_exchange_j_folds_ghosts(n):
    """add_and_fill_ghosts_j: interior += all periodic ghost images, ghosts := images"""
    pl = psc_inputs.thermal(n, 1, seed=3)
    sim = _sim(pl)
    rng = np.random.default_rng(1)
    full = rng.integers(-8, 9, size=sim.psc.field_shape).astype(np.float32)  # exact in fp32
    sim.J.copy_(torch.from_numpy(full).cuda())
    sim.psc.exchange_j()
    got = sim.J.cpu().numpy()
    g = sim.g
    want = np.zeros((3, n[2], n[1], n[0]))
    ez, ey, ex = full.shape[1:]
    for k in range(ez):
        for j in range(ey):
            for i in range(ex):
                want[:, (k - g[2]) % n[2], (j - g[1]) % n[1], (i - g[0]) % n[0]] += full[:, k, j, i]
    assert np.array_equal(sim.interior(sim.J).cpu().numpy().astype(np.float64), want)
    for k in range(ez):
        for j in range(ey):
            for i in range(ex):
                assert np.array_equal(got[:, k, j, i],
                                      want[:, (k - g[2]) % n[2], (j - g[1]) % n[1], (i - g[0]) % n[0]])


# ------------------------------------------------------------------------------------------------
# sort

@pytest.mark.parametrize("kind,block", [("2d", (0, 0, 0)), ("2d-ragged", (1, 4, 8)),
                                        ("3d", (0, 0, 0)), ("3d-ragged", (2, 4, 2)),
                                        ("harris", (1, 8, 8))])
def test_sort_bit_exact(kind, block):
    pl = _small(kind).shuffled()
    sim = _sim(pl, block=block)
    orc = oracle_for(pl, block=library_block(pl.n, block))
    before = {k: getattr(pl, k).numpy().copy() for k in ("x", "y", "z", "ux", "uy", "uz", "qw", "species", "id")}
    cell_idx, key, perm, offs = orc.sort(before["x"], before["y"], before["z"])
    sim.psc.particles_sort()
    assert sim.psc.status() == 0
    g_ci, g_pm, g_co = (t.cpu().numpy() for t in sim.sort_result())
    assert np.array_equal(g_ci, cell_idx)
    assert np.array_equal(g_co, offs)
    assert np.array_equal(g_pm, perm)
    after = gpu_cols(sim)
    for k, v in before.items():
        assert np.array_equal(after[k], v[perm]), k


@pytest.mark.parametrize("kind,block", [("2d", (0, 0, 0)), ("2d-ragged", (1, 4, 8)), ("2d-ragged", (1, 24, 40)),
                                        ("3d", (0, 0, 0)), ("3d-ragged", (2, 4, 2)), ("3d-ragged", (1, 1, 1)),
                                        ("harris", (1, 8, 8)), ("beam", (0, 0, 0))])
def test_sort_of_a_pushed_store_bit_exact(kind, block):
    """psc_particles_sort on a store that pushes have advanced (residents in their cells, leavers
    waiting in the exchange rows).  The cell a particle is filed under is the
    GPU's own decision (its fp32 move); GIVEN those cells, the stable permutation, the offsets and
    the sorted columns must equal the oracle's counting sort bit for bit.  (The assertion
    `key == keys of the gathered list` only checks the test's own key <-> cell conversion; the
    offsets, permutation and column comparisons carry the weight.)"""
    pl = _small(kind)
    smooth_fields(pl, 0.05, seed=21)
    sim = _sim(pl, block=block)
    lb = library_block(pl.n, block)
    orc = oracle_for(pl, block=lb)
    sim.psc.particles_sort()
    for it in range(3):
        if it < 2:
            sim.psc.push_particles()
        else:
            sim.psc.step()
            sim.psc.step()                       # arrivals filed into holes, new leavers waiting
        before = gpu_state(sim)
        cells = [np.ascontiguousarray(v.astype(np.int32)) for v in
                 key_to_cell(before["key"].astype(np.int64), pl.n, lb)]
        cell_idx, key, perm, offs = orc.sort_cells(*cells)
        assert np.array_equal(key, before["key"])
        moved = int((np.diff(key) < 0).sum())
        assert moved > 0                         # the push really un-sorted the list
        sim.psc.particles_sort()
        assert sim.psc.status() == 0
        g_ci, g_pm, g_co = (t.cpu().numpy() for t in sim.sort_result())
        assert np.array_equal(g_co, offs)
        assert np.array_equal(g_pm, perm)
        assert np.array_equal(g_ci, cell_idx)
        after = gpu_state(sim)
        for k, v in before.items():
            assert np.array_equal(after[k], v[perm]), k


def test_step_equals_explicit_calls():
    """psc_step (index sort + reorder on load) gives the same state as the explicit sequence
    psc_particles_sort, psc_push_fields, psc_push_particles, ... of Fig. 8: particle columns
    bit for bit after the first step (same arithmetic on the same values), within rounding of
    the atomically summed J afterwards"""
    pl = _small("2d")
    a, b = _sim(pl), _sim(pl)
    for it in range(4):
        a.psc.step()
        b.psc.particles_sort()
        b.psc.push_fields(1, 0.5)
        b.psc.push_particles()
        b.psc.push_fields(1, 0.5)
        b.psc.exchange_j()
        b.psc.push_fields(0, 1.0)
        ca, cb = gpu_state(a), gpu_state(b)
        ia, ib = np.argsort(ca["id"], kind="stable"), np.argsort(cb["id"], kind="stable")
        if it == 0:
            for k in ca:
                assert np.array_equal(ca[k][ia], cb[k][ib]), k
        else:
            for k in ("ux", "uy", "uz"):
                assert np.abs(ca[k][ia] - cb[k][ib]).max() < 1e-6
        assert (a.J - b.J).abs().max() <= 1e-5 * b.J.abs().max()
    assert a.psc.status() == 0 and b.psc.status() == 0


@pytest.mark.parametrize("kind", ["2d", "3d-ragged-o2"])
def test_fig7_composition_lands_on_psc_step(kind):
    """Fig. 7's ordering composed from the half-step calls -- psc_push_fields(E,
    0.5), psc_push_fields(B, 0.5), psc_push_particles, psc_push_fields(B, 0.5), psc_exchange_j,
    psc_push_fields(E, 0.5) -- entered with E^{1/2} and left with one more E half step, against N
    psc_step (Fig. 8) from the same state, and both against the oracle's Fig. 8."""
    pl = _small(kind)
    smooth_fields(pl, 0.05, seed=77)
    a, b = _sim(pl), _sim(pl)
    N = 5
    a.step(N)
    b.psc.particles_sort()
    for k in range(N):
        if k > 0:
            b.psc.push_fields(0, 0.5)
        b.psc.push_fields(1, 0.5)
        b.psc.push_particles()
        b.psc.push_fields(1, 0.5)
        b.psc.exchange_j()
        b.psc.push_fields(0, 0.5)
    b.psc.push_fields(0, 0.5)
    assert a.psc.status() == 0 and b.psc.status() == 0
    f64 = lambda t: t.cpu().numpy().astype(np.float64)
    for F in ("E", "B", "J"):
        assert rel_maxnorm(f64(b.interior(getattr(b, F))), f64(a.interior(getattr(a, F)))) < TOL, F
    ca, cb = gpu_state(a), gpu_state(b)
    ia, ib = np.argsort(ca["id"], kind="stable"), np.argsort(cb["id"], kind="stable")
    assert np.array_equal(ca["key"][ia], cb["key"][ib]) or \
        np.mean(ca["key"][ia] != cb["key"][ib]) < 1e-4            # (a particle within rounding of a face)
    for k in ("ux", "uy", "uz"):
        assert np.abs(ca[k][ia] - cb[k][ib]).max() < TOL * max(1.0, np.abs(ca[k]).max())
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], N)
    assert rel_maxnorm(f64(b.interior(b.E)), E) < TOL and rel_maxnorm(f64(b.interior(b.B)), B) < 10 * TOL
    assert rel_maxnorm(f64(b.interior(b.J)), J) < TOL


def test_invariant_coordinate_is_optional():
    """2-d run with x == NULL (not carried): same y, z, u as with x bound"""
    from paper_1310_7866_b200.harness import Simulation
    pl = _small("2d-ragged")
    a = Simulation(pl)
    b = Simulation(pl, with_x=False)
    a.step(3)
    b.step(3)
    ca, cb = gpu_cols(a, export=False), gpu_cols(b, export=False)
    assert "x" not in cb
    ia, ib = np.argsort(ca["id"], kind="stable"), np.argsort(cb["id"], kind="stable")
    for k in ("y", "z", "ux", "uy", "uz", "qw", "species"):
        assert np.allclose(ca[k][ia], cb[k][ib], rtol=0, atol=1e-6), k
    assert b.psc.status() == 0


def test_sort_degenerate_cases():
    # empty list
    pl = psc_inputs.thermal((1, 8, 8), 1, seed=3)
    for k in ("x", "y", "z", "ux", "uy", "uz", "qw", "species", "id"):
        setattr(pl, k, getattr(pl, k)[:0])
    sim = _sim(pl)
    sim.psc.particles_sort()
    assert int(sim.sort_result()[2].abs().max()) == 0
    sim.psc.push_particles()
    sim.psc.particles_sort()                     # sort of an empty pushed store
    assert int(sim.sort_result()[2].abs().max()) == 0
    sim.step(2)
    assert sim.psc.status() == 0
    # everything in very few cells: segments of ~3000 (shared-memory block sort) and ~70000
    # (in-place global sort) particles
    for count in (3000, 70000):
        pl = psc_inputs.thermal((1, 8, 8), 1, seed=3)
        g = torch.Generator().manual_seed(5)
        n = count
        pl.y = (torch.rand(n, generator=g) * 0.999 + 3.0).float()
        pl.z = (torch.rand(n, generator=g) * 0.999 + (torch.rand(n, generator=g) < 0.9).float() * 2.0).float()
        pl.x = torch.full((n,), 0.5)
        pl.ux = torch.zeros(n); pl.uy = torch.zeros(n); pl.uz = torch.zeros(n)
        pl.qw = torch.ones(n); pl.species = torch.zeros(n, dtype=torch.int32)
        pl.id = torch.arange(n, dtype=torch.int32)
        sim = _sim(pl, block=(1, 4, 4))
        orc = oracle_for(pl, block=(1, 4, 4))
        ci, key, perm, offs = orc.sort(pl.x.numpy(), pl.y.numpy(), pl.z.numpy())
        sim.psc.particles_sort()
        g_ci, g_pm, g_co = (t.cpu().numpy() for t in sim.sort_result())
        assert np.array_equal(g_co, offs) and np.array_equal(g_pm, perm) and np.array_equal(g_ci, ci)


def test_sort_flags_out_of_domain():
    pl = psc_inputs.thermal((1, 8, 8), 2, seed=3)
    pl.y[5] = 8.0
    sim = _sim(pl)
    sim.psc.particles_sort()
    assert sim.psc.status() & 1


def test_sort_flags_bad_species_and_files_x_just_below_L():
    """a species index outside [0, n_species) raises PSC_F_SPECIES at the sort (the particle is then
    pushed as species 0 instead of reading past the species table); a position whose fp32 product
    with 1/dx rounds up to n although x < L is filed in the last cell without a flag, key and
    offset referring to the same cell"""
    from paper_1310_7866_b200 import PSC_F_SPECIES
    pl = psc_inputs.thermal((1, 8, 8), 2, seed=3)
    pl.species[3] = 7
    pl.species[4] = -1
    sim = _sim(pl)
    sim.psc.particles_sort()
    assert sim.psc.status() == PSC_F_SPECIES
    sim.step(2)
    g = gpu_state(sim)
    assert g["species"].min() >= 0 and g["species"].max() <= 1
    # dx = 0.48: L = 3.84f; the largest float below L times fl(1/0.48) rounds to 8.0
    pl = psc_inputs.thermal((1, 8, 8), 2, dx=(1.0, 0.48, 0.48), seed=3)
    Lf = np.float32(8) * np.float32(0.48)
    below = np.nextafter(Lf, np.float32(0))
    assert np.float32(below * (np.float32(1) / np.float32(0.48))) >= 8.0   # the case this test is about
    pl.y[0] = float(below)
    pl.z[1] = float(below)
    sim = _sim(pl)
    sim.psc.particles_sort()
    assert sim.psc.status() == 0
    g = gpu_state(sim)
    o = np.argsort(g["id"])
    cells = key_to_cell(g["key"][o].astype(np.int64), pl.n, library_block(pl.n))
    assert cells[1][0] == 7 and cells[2][1] == 7
    assert 0.999 < g["y"][o][0] < 1.0 and 0.999 < g["z"][o][1] < 1.0


@pytest.mark.parametrize("order", [1, 2])
def test_store_spill_relayout_and_big_cells(order):
    """the exceptional paths of the cell store, all at once: 300 particles per cell (more than the
    256-slot shared-memory image: the BIG launch streams those cells from global memory), a drift
    that makes a third of them change cell every step (more leavers than the 32 records of an
    exchange row: the rest spills and the next step re-lays the store out on the device), cells
    that fill beyond their capacity.  Six steps against the oracle, particle by particle."""
    pl = psc_inputs.thermal((1, 16, 16), 150, seed=23, order=order, name="dense")
    n = pl.y.numel()
    vy = 0.33 * pl.dx[1] / pl.dt
    gam = 1.0 / np.sqrt(1.0 - vy * vy)
    pl.uy = pl.uy + float(gam * vy)
    pl.qw = pl.qw * 1e-2
    # a clump: one cell holds 900 more particles than the rest
    g = torch.Generator().manual_seed(4)
    extra = 900
    for k in ("x", "ux", "uz"):
        setattr(pl, k, torch.cat([getattr(pl, k), torch.zeros(extra)]))
    pl.y = torch.cat([pl.y, 5.0 + torch.rand(extra, generator=g)])
    pl.z = torch.cat([pl.z, 9.0 + torch.rand(extra, generator=g)])
    pl.uy = torch.cat([pl.uy, torch.full((extra,), float(gam * vy))])
    pl.qw = torch.cat([pl.qw, torch.full((extra,), float(pl.qw[0]))])
    pl.species = torch.cat([pl.species, torch.zeros(extra, dtype=torch.int32)])
    pl.id = torch.arange(n + extra, dtype=torch.int32)
    sim = _sim(pl)
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    L = [pl.n[d] * pl.dx[d] for d in range(3)]
    for it in range(6):
        orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], 1)
        sim.step(1)
        assert sim.psc.status() == 0
        g1 = gpu_state(sim)
        assert np.array_equal(np.sort(g1["id"]), np.arange(n + extra))      # nobody lost, nobody duplicated
        o = order_by_id(g1["id"], st["id"])
        _, py, pz = positions_f64(g1, pl)
        assert periodic_dist(py[o], st["y"], L[1]).max() < 1e-4
        assert periodic_dist(pz[o], st["z"], L[2]).max() < 1e-4
        for c in ("ux", "uy", "uz"):
            assert np.abs(g1[c][o] - st[c]).max() < TOL
        assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL
    info = sim.psc.store_info()
    assert info["relayouts"] >= 1 and info["max_count"] > 256


def test_spilled_leavers_are_filed_without_a_relayout():
    """more than 32 particles leave one cell in a step (the exchange row holds 32 records): the rest
    goes to the spill list, and because their destination cell has room the next step files them
    straight into it -- no re-layout.  Five steps against the oracle, particle by particle."""
    pl = psc_inputs.thermal((1, 16, 16), 12, seed=37, name="row-overflow")
    n = pl.y.numel()
    vy = 0.33 * pl.dx[1] / pl.dt
    gam = 1.0 / np.sqrt(1.0 - vy * vy)
    pl.qw = pl.qw * 1e-2
    g = torch.Generator().manual_seed(6)
    extra = 38
    for k in ("x", "ux", "uz"):
        setattr(pl, k, torch.cat([getattr(pl, k), torch.zeros(extra)]))
    pl.y = torch.cat([pl.y, 5.9 + 0.0999 * torch.rand(extra, generator=g)])
    pl.z = torch.cat([pl.z, 9.2 + 0.6 * torch.rand(extra, generator=g)])
    pl.uy = torch.cat([pl.uy, torch.full((extra,), float(gam * vy))])
    pl.qw = torch.cat([pl.qw, torch.full((extra,), float(pl.qw[0]))])
    pl.species = torch.cat([pl.species, torch.zeros(extra, dtype=torch.int32)])
    pl.id = torch.arange(n + extra, dtype=torch.int32)
    sim = _sim(pl)
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    L = [pl.n[d] * pl.dx[d] for d in range(3)]
    for it in range(5):
        orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], 1)
        sim.step(1)
        assert sim.psc.status() == 0
        g1 = gpu_state(sim)
        assert np.array_equal(np.sort(g1["id"]), np.arange(n + extra))
        o = order_by_id(g1["id"], st["id"])
        _, py, pz = positions_f64(g1, pl)
        assert periodic_dist(py[o], st["y"], L[1]).max() < 1e-4
        assert periodic_dist(pz[o], st["z"], L[2]).max() < 1e-4
        for c in ("ux", "uy", "uz"):
            assert np.abs(g1[c][o] - st[c]).max() < TOL
        assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL
    info = sim.psc.store_info()
    assert info["inserted"] >= 2 and info["relayouts"] == 0


def test_big_cell_whole_chunks_leave():
    """a cell of the BIG launch (more particles than the image holds) whose particles ALL cross
    the same face in one step: batches of 32 leavers against a 24-entry crosser queue (2-d) -- the
    trajectories beyond the queue's room are walked at once; the exchange row overflows (32
    records) into the spill list and the store is re-laid out.  Three steps against the oracle."""
    pl = psc_inputs.thermal((1, 16, 16), 12, seed=29, name="clump")
    n = pl.y.numel()
    vy = 0.33 * pl.dx[1] / pl.dt
    gam = 1.0 / np.sqrt(1.0 - vy * vy)
    pl.qw = pl.qw * 1e-2
    g = torch.Generator().manual_seed(5)
    extra = 600
    for k in ("x", "ux", "uz"):
        setattr(pl, k, torch.cat([getattr(pl, k), torch.zeros(extra)]))
    pl.y = torch.cat([pl.y, 5.9 + 0.0999 * torch.rand(extra, generator=g)])       # just below the face y = 6
    pl.z = torch.cat([pl.z, 9.2 + 0.6 * torch.rand(extra, generator=g)])
    pl.uy = torch.cat([pl.uy, torch.full((extra,), float(gam * vy))])
    pl.qw = torch.cat([pl.qw, torch.full((extra,), float(pl.qw[0]))])
    pl.species = torch.cat([pl.species, torch.zeros(extra, dtype=torch.int32)])
    pl.id = torch.arange(n + extra, dtype=torch.int32)
    sim = _sim(pl)
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    L = [pl.n[d] * pl.dx[d] for d in range(3)]
    sim.psc.particles_sort()
    assert sim.psc.store_info()["max_count"] > 256
    for it in range(3):
        orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], 1)
        sim.step(1)
        assert sim.psc.status() == 0
        g1 = gpu_state(sim)
        assert np.array_equal(np.sort(g1["id"]), np.arange(n + extra))
        o = order_by_id(g1["id"], st["id"])
        _, py, pz = positions_f64(g1, pl)
        assert periodic_dist(py[o], st["y"], L[1]).max() < 1e-4
        assert periodic_dist(pz[o], st["z"], L[2]).max() < 1e-4
        for c in ("ux", "uy", "uz"):
            assert np.abs(g1[c][o] - st[c]).max() < TOL
        assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL


def test_3d_tma_tile_path_matches_oracle():
    """the 3-d order-1 kernel with its tiles staged by TMA tensor copies (no optional columns, the
    default 4x4x4 block, a cell image of 128 / 160 slots): J, E, B after five steps against the
    oracle, and the same run with the id column bound (plain 4-byte staging) for comparison"""
    pl = psc_inputs.thermal((16, 16, 16), 35, seed=31, name="3d-tma")
    smooth_fields(pl, 0.05, seed=8)
    sim = _sim(pl, with_id=False)
    sim.step(5)
    assert sim.psc.status() == 0
    info = sim.psc.store_info()
    assert info["tma_tiles"] == 1 and info["image_slots"] in (128, 160)
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], 5)
    for got, want in ((sim.J, J), (sim.E, E), (sim.B, B)):
        g = sim.interior(got).cpu().numpy()
        for c in range(3):
            assert np.abs(g[c] - want[c]).max() <= TOL * np.abs(want[c]).max()
    sim2 = _sim(pl, with_id=True)
    sim2.step(5)
    assert sim2.psc.store_info()["tma_tiles"] == 0
    for a, b in ((sim.J, sim2.J), (sim.E, sim2.E)):
        ga, gb = sim.interior(a).cpu().numpy(), sim2.interior(b).cpu().numpy()
        assert np.abs(ga - gb).max() <= TOL * np.abs(gb).max()


# ------------------------------------------------------------------------------------------------
# particle loop, open loop: same sorted state in, one psc_push_particles, compare

def _push_once(kind, block, amp=0.05):
    pl = _small(kind)
    smooth_fields(pl, amp, seed=21)
    sim = _sim(pl, block=block)
    sim.psc.particles_sort()
    cols0 = oracle_sorted_state(pl, block)        # the sorted fp32 input both paths see
    mine = gpu_cols(sim, export=False)            # internal form: offsets; the rest verbatim
    for k, v in cols0.items():
        if k in ("x", "y", "z") and pl.n["xyz".index(k)] > 1:
            continue
        assert np.array_equal(mine[k], v), k
    px, py, pz = gpu_positions_f64(sim, block)
    for d, (k, got) in enumerate(zip("xyz", (px, py, pz))):
        assert np.abs(got - cols0[k].astype(np.float64)).max() <= 1.2e-7 * pl.n[d] * pl.dx[d], k
    orc = oracle_for(pl)
    _, E, B = oracle_state(pl)
    st = {k: np.ascontiguousarray(cols0[k].astype(np.float64)) for k in ("x", "y", "z", "ux", "uy", "uz", "qw")}
    sp = np.ascontiguousarray(cols0["species"])
    J = orc.zeros_field()
    orc.push_particles(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], sp)
    sim.psc.push_particles()
    sim.psc.exchange_j()
    assert sim.psc.status() == 0
    return pl, sim, orc, cols0, st, sp, J


@pytest.mark.parametrize("kind,block", [("2d", (0, 0, 0)), ("2d-ragged", (1, 4, 8)),
                                        ("2d-ragged", (1, 24, 40)), ("3d", (0, 0, 0)),
                                        ("3d-ragged", (2, 4, 2)), ("3d-ragged", (1, 1, 1)),
                                        ("harris", (1, 8, 8)), ("beam", (0, 0, 0)),
                                        ("3d-ragged-o2", (2, 4, 2)), ("3d-ragged-o2", (1, 1, 1)),
                                        ("2d-o2", (0, 0, 0)), ("2d-o2", (1, 3, 5)),
                                        ("2d-aniso", (0, 0, 0)), ("2d-aniso-o2", (1, 4, 8)),
                                        ("3d-aniso", (0, 0, 0)), ("3d-aniso-o2", (2, 4, 2))])
def test_push_particles_matches_oracle(kind, block):
    pl, sim, orc, cols0, st, sp, J = _push_once(kind, block)
    got = gpu_cols(sim)
    o = order_by_id(got["id"], cols0["id"])       # the push regroups inside each cell's segment
    got = {k: v[o] for k, v in got.items()}
    L = [pl.n[d] * pl.dx[d] for d in range(3)]
    for d, c in enumerate(("x", "y", "z")):
        if pl.n[d] == 1:
            assert np.array_equal(got[c], cols0[c])        # invariant coordinate is carried
            continue
        assert (periodic_dist(got[c], st[c], L[d]) / L[d]).max() < TOL
        assert periodic_dist(got[c], st[c], L[d]).max() < 1e-4 * pl.dx[d]
        assert got[c].min() >= 0.0 and got[c].max() < L[d]
    for s in range(len(pl.q)):
        m = sp == s
        rms = np.sqrt(np.mean(st["ux"][m] ** 2 + st["uy"][m] ** 2 + st["uz"][m] ** 2))
        for c in ("ux", "uy", "uz"):
            assert np.abs(got[c][m] - st[c][m]).max() / rms < TOL
    assert np.array_equal(got["qw"], cols0["qw"]) and np.array_equal(got["species"], cols0["species"])
    assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL


@pytest.mark.parametrize("kind", ["2d", "3d", "beam", "2d-o2", "2d-aniso", "3d-aniso-o2"])
def test_gpu_continuity_residual(kind):
    """(rho^{n+3/2} - rho^{n+1/2})/dt + div- j^{n+1} = 0 (Eq. 25) with the GPU's J and the GPU's
    stored fp32 positions, evaluated by the oracle's rho / div-; normalised by max|rho_s|/dt of one
    species."""
    pl, sim, orc, cols0, st, sp, J = _push_once(kind, (0, 0, 0), amp=0.05)
    f64 = lambda a: np.ascontiguousarray(a.astype(np.float64))
    g1 = gpu_state(sim)
    x1, y1, z1 = positions_f64(g1, pl)             # internal form: no export rounding
    o = order_by_id(g1["id"], cols0["id"])
    x1, y1, z1 = (np.ascontiguousarray(v[o]) for v in (x1, y1, z1))
    rho0 = orc.rho(f64(cols0["x"]), f64(cols0["y"]), f64(cols0["z"]), f64(cols0["qw"]))
    rho1 = orc.rho(x1, y1, z1, f64(cols0["qw"]))
    Jg = np.ascontiguousarray(sim.interior(sim.J).cpu().numpy().astype(np.float64))
    res = (rho1 - rho0) / pl.dt + orc.div_minus(Jg)
    m = sp == 0
    rho_s = orc.rho(f64(cols0["x"][m]), f64(cols0["y"][m]), f64(cols0["z"][m]), f64(cols0["qw"][m]))
    assert np.abs(res).max() / (np.abs(rho_s).max() / pl.dt) < TOL


# ------------------------------------------------------------------------------------------------
# closed loop: 10 psc_step, particles matched by id

@pytest.mark.parametrize("kind", ["2d", "3d", "harris", "beam", "2d-o2", "2d-aniso-o2", "3d-aniso"])
def test_ten_steps_match_oracle(kind):
    pl = _small(kind)
    sim = _sim(pl)
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    nsteps = 10
    orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], nsteps)
    sim.step(nsteps)
    assert sim.psc.status() == 0
    got = gpu_cols(sim)
    order = np.argsort(got["id"], kind="stable")
    assert np.array_equal(got["id"][order], st["id"])
    L = [pl.n[d] * pl.dx[d] for d in range(3)]
    g1 = gpu_state(sim)
    o1 = np.argsort(g1["id"], kind="stable")
    p64 = positions_f64(g1, pl)
    for d, c in enumerate(("x", "y", "z")):
        if pl.n[d] > 1:
            # north_star's reading (relative to the domain) and, stricter, in units of a cell from
            # the internal form without export rounding: ten steps of fp32 round-off in the
            # gathered fields (~1e-6 of the thermal velocity per step) stay below 1e-4 cell
            assert (periodic_dist(got[c][order], st[c], L[d]) / L[d]).max() < TOL
            assert periodic_dist(p64[d][o1], st[c], L[d]).max() < 1e-4 * pl.dx[d]
    for s in range(len(pl.q)):
        m = st["species"] == s
        rms = np.sqrt(np.mean(st["ux"][m] ** 2 + st["uy"][m] ** 2 + st["uz"][m] ** 2))
        for c in ("ux", "uy", "uz"):
            assert np.abs(got[c][order][m] - st[c][m]).max() / rms < TOL
    assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL
    assert rel_maxnorm(sim.interior(sim.E).cpu().numpy(), E) < TOL
    # B: the Harris sheet has |B_y| ~ 0.06 next to self-generated B_x, B_z ~ 1e-4 whose fp32
    # round-off (ulp of the E and B_y they are differenced from) is ~1e-9 absolute; the bar is the
    # north_star's "relative to the field's max-norm", the per-component figure is 10x looser
    assert rel_fieldnorm(sim.interior(sim.B).cpu().numpy(), B) < TOL
    assert rel_maxnorm(sim.interior(sim.B).cpu().numpy(), B) < 10 * TOL


@pytest.mark.parametrize("order", [1, 2])
def test_store_under_mass_migration(order):
    """the cell store (in-place stayers, exchange rows, hole filling, spill + re-layout) under stress: a cold drifting slab in which whole
    cells empty out and refill (v dt/dx = 0.3 along y, 0.15 along z, |v| = 0.95 c: two fifths of
    the particles change cell every step, cells receive > 32 arrivals, cells start with zero
    stayers), most of the grid empty.  Eight psc_step against the oracle, matched by id; keys agree with positions."""
    pl = psc_inputs.thermal((1, 16, 24), 40, seed=17, order=order, name="slab")
    keep = (pl.y >= 3.0) & (pl.y < 6.0) & (pl.species == 0)     # a slab three cells thick, one species
    for k in ("x", "y", "z", "ux", "uy", "uz", "qw", "species"):
        setattr(pl, k, getattr(pl, k)[keep].contiguous())
    n = pl.y.numel()
    pl.id = torch.arange(n, dtype=torch.int32)
    vy, vz = 0.3 * pl.dx[1] / pl.dt, 0.15 * pl.dx[2] / pl.dt   # cells per step -> velocity
    gam = 1.0 / np.sqrt(1.0 - vy * vy - vz * vz)
    pl.ux = torch.zeros(n); pl.uy = torch.full((n,), float(gam * vy)); pl.uz = torch.full((n,), float(gam * vz))
    pl.qw = pl.qw * 1e-3                                        # nearly a test-particle beam
    sim = _sim(pl)
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    lb = library_block(pl.n)
    for it in range(8):
        orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], 1)
        sim.step(1)
        assert sim.psc.status() == 0
        # the cell each particle is filed under is the cell its position is in
        g1 = gpu_state(sim)
        _, py, pz = positions_f64(g1, pl)
        cells = key_to_cell(g1["key"].astype(np.int64), pl.n, lb)
        assert np.array_equal(np.floor(py / pl.dx[1]).astype(np.int64), cells[1])
        assert np.array_equal(np.floor(pz / pl.dx[2]).astype(np.int64), cells[2])
        ids = g1["id"]
        assert np.array_equal(np.sort(ids), np.arange(n))      # nobody lost, nobody duplicated
        o = order_by_id(ids, st["id"])
        L = [pl.n[d] * pl.dx[d] for d in range(3)]
        assert (periodic_dist(py[o], st["y"], L[1]) / L[1]).max() < TOL
        assert (periodic_dist(pz[o], st["z"], L[2]) / L[2]).max() < TOL
        assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL


def test_step_host_end_to_end():
    """psc_step_host (host buffers in, host buffers out) equals the device-resident path"""
    pl = _small("2d")
    sim = _sim(pl)
    sim.step(3)
    ref = gpu_cols(sim)
    refE = sim.E.cpu()
    sim2 = _sim(pl)
    host = {k: getattr(pl, k).clone().pin_memory() for k in ("x", "y", "z", "ux", "uy", "uz", "qw", "species", "id")}
    hE = sim2.E.cpu().pin_memory()
    hB = sim2.B.cpu().pin_memory()
    hJ = torch.zeros_like(hE).pin_memory()
    sim2.psc.step_host(pl.n_particles, host, hE, hB, hJ, nsteps=3)
    # (J is accumulated with floating-point atomics, so two runs agree to rounding, not bitwise)
    for k in ("id", "species", "qw"):
        assert np.array_equal(host[k].numpy(), ref[k]), k
    for k in ("y", "z", "ux", "uy", "uz"):
        assert np.abs(host[k].numpy() - ref[k]).max() < 1e-5, k
    assert (hE - refE).abs().max() <= 1e-5 * refE.abs().max()


# ------------------------------------------------------------------------------------------------
# alternating-order interpolation (A29)

@pytest.mark.parametrize("kind", ["2d", "3d", "2d-o2", "beam", "3d-aniso", "2d-aniso-o2"])
def test_alternating_order_ten_steps_match_oracle(kind):
    """PSC_SCHEME_ALTERNATING against the oracle's scheme 1: ten psc_step, particles by id"""
    from paper_1310_7866_b200.harness import Simulation
    pl = _small(kind)
    smooth_fields(pl, 0.05, seed=29)
    sim = Simulation(pl, scheme=1)
    orc = oracle_for(pl, scheme=1)
    std = oracle_for(pl, scheme=0)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    s0 = {k: v.copy() for k, v in st.items()}
    orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], 10)
    sim.step(10)
    assert sim.psc.status() == 0
    got = gpu_cols(sim)
    order = np.argsort(got["id"], kind="stable")
    L = [pl.n[d] * pl.dx[d] for d in range(3)]
    for d, c in enumerate(("x", "y", "z")):
        if pl.n[d] > 1:
            assert (periodic_dist(got[c][order], st[c], L[d]) / L[d]).max() < TOL
    for s_ in range(len(pl.q)):
        m = st["species"] == s_
        rms = np.sqrt(np.mean(st["ux"][m] ** 2 + st["uy"][m] ** 2 + st["uz"][m] ** 2))
        for c in ("ux", "uy", "uz"):
            assert np.abs(got[c][order][m] - st[c][m]).max() / rms < TOL
    assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL
    assert rel_maxnorm(sim.interior(sim.E).cpu().numpy(), E) < TOL
    assert rel_fieldnorm(sim.interior(sim.B).cpu().numpy(), B) < TOL
    # and it is not the standard scheme in disguise
    E0 = oracle_state(pl)[1]
    B0 = oracle_state(pl)[2]
    J0 = std.zeros_field()
    std.step(E0, B0, J0, s0["x"], s0["y"], s0["z"], s0["ux"], s0["uy"], s0["uz"], s0["qw"], s0["species"], 10)
    assert np.abs(s0["ux"] - st["ux"]).max() > 1e-4 * np.abs(st["ux"]).max()
