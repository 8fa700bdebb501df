"""Error behaviour of the C ABI on a device and degenerate inputs of the particle loop."""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_1310_7866_b200 as psc
import psc_inputs
from tests.util import gpu_cols, oracle_for, oracle_state, order_by_id, periodic_dist, rel_maxnorm

pytestmark = pytest.mark.gpu
TOL = 1e-5


def _sim(pl, **kw):
    from paper_1310_7866_b200.harness import Simulation

    return Simulation(pl, **kw)


def test_call_order_and_binding_errors():
    pl = psc_inputs.thermal((1, 8, 8), 2, seed=5)
    sim = _sim(pl)
    L, h = psc.lib(), sim.psc._h
    assert L.psc_push_particles(h, None) == -3                  # PSC_ERR_NOT_SORTED: no sort yet
    sim.psc.particles_sort()
    sim.psc.push_particles()
    assert L.psc_push_particles(h, None) == 0                   # the store stays ordered by cell: no sort needed
    sim.psc.particles_sort()
    assert L.psc_push_fields(h, 7, C.c_float(0.5), None) == -1  # which must be PSC_E or PSC_B
    assert L.psc_push_fields(h, 1, C.c_float(0.0), None) == -1  # frac > 0
    assert L.psc_fill_ghosts(h, 9, None) == -1
    # a workspace that is too small / misaligned is refused
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    assert L.psc_bind_workspace(h, C.c_void_p(small.data_ptr() + 8), C.c_size_t(1016)) == -5   # PSC_ERR_ALIGN
    sim.psc.particles_export()                                  # (keys live in the workspace)
    assert L.psc_bind_workspace(h, C.c_void_p(small.data_ptr()), C.c_size_t(1024)) == -8       # PSC_ERR_WORKSPACE
    assert sim.psc.status() == 0


def test_unbound_context_reports_not_bound():
    pl = psc_inputs.thermal((1, 8, 8), 1, seed=5)
    p = psc.Psc(pl.n, pl.dx, pl.dt, 1, pl.q, pl.m, (0, 0, 0))
    L = psc.lib()
    assert L.psc_step(p._h, None) == -2                         # PSC_ERR_NOT_BOUND
    assert L.psc_particles_sort(p._h, None) == -2
    assert L.psc_push_fields(p._h, 1, C.c_float(0.5), None) == -2


@pytest.mark.parametrize("order", [1, 2])
def test_eight_species_and_particles_on_faces(order):
    """PSC_MAX_SPECIES species (one neutral, one heavy), particles placed exactly on cell faces,
    on the domain origin and one ulp below the upper edge; five steps against the oracle."""
    pl = psc_inputs.thermal((1, 16, 12), 6, seed=41, order=order, name="faces")
    n = pl.y.numel()
    g = torch.Generator().manual_seed(3)
    pl.q = [-1.0, 1.0, 0.0, 2.0, -3.0, 1.0, -1.0, 0.5]
    pl.m = [1.0, 100.0, 1.0, 4.0, 9.0, 1836.0, 2.0, 0.7]
    pl.species = torch.randint(0, 8, (n,), generator=g, dtype=torch.int32)
    k = n // 4
    pl.y[:k] = torch.floor(pl.y[:k])                            # exactly on faces
    pl.z[k:2 * k] = torch.floor(pl.z[k:2 * k])
    pl.y[0], pl.z[0] = 0.0, 0.0
    pl.y[1] = float(np.nextafter(np.float32(16.0), np.float32(0.0)))
    pl.z[2] = float(np.nextafter(np.float32(12.0), np.float32(0.0)))
    sim = _sim(pl)
    orc = oracle_for(pl)
    st, E, B = oracle_state(pl)
    J = orc.zeros_field()
    orc.step(E, B, J, st["x"], st["y"], st["z"], st["ux"], st["uy"], st["uz"], st["qw"], st["species"], 5)
    sim.step(5)
    assert sim.psc.status() == 0
    got = gpu_cols(sim)
    o = order_by_id(got["id"], st["id"])
    L = [pl.n[d] * pl.dx[d] for d in range(3)]
    for d, c in ((1, "y"), (2, "z")):
        assert (periodic_dist(got[c][o], st[c], L[d]) / L[d]).max() < TOL
    assert np.array_equal(got["species"][o], st["species"])
    for c in ("ux", "uy", "uz"):
        assert np.abs(got[c][o] - st[c]).max() < TOL * 0.1
    assert rel_maxnorm(sim.interior(sim.J).cpu().numpy(), J) < TOL
    assert rel_maxnorm(sim.interior(sim.E).cpu().numpy(), E) < TOL


def test_step_host_without_optional_columns():
    """psc_step_host in bench.py's configuration (no x, no id) equals the device-resident run"""
    pl = psc_inputs.thermal((1, 16, 16), 4, seed=9)
    a = _sim(pl, with_id=False, with_x=False)
    a.step(2)
    ref = gpu_cols(a)
    b = _sim(pl, with_id=False, with_x=False)
    host = {k: (None if k in ("x", "id") else getattr(pl, k).clone().pin_memory())
            for k in ("x", "y", "z", "ux", "uy", "uz", "qw", "species", "id")}
    hE, hB = b.E.cpu().pin_memory(), b.B.cpu().pin_memory()
    hJ = torch.zeros_like(hE).pin_memory()
    b.psc.step_host(pl.n_particles, host, hE, hB, hJ, nsteps=2)
    # no id to match by: compare per-cell-independent aggregates and the fields
    for k in ("ux", "uy", "uz", "qw"):
        assert abs(float(host[k].double().sum()) - float(ref[k].astype(np.float64).sum())) <= 1e-6 * np.abs(ref[k]).sum()
    assert np.array_equal(np.sort(host["species"].numpy()), np.sort(ref["species"]))
    assert (hE - a.E.cpu()).abs().max() <= 1e-5 * a.E.abs().max().cpu()


@pytest.mark.parametrize("cfg,scale,steps", [(1, None, 100), (3, (1, 32, 128), 200), (5, (8, 8, 32), 100)])
def test_full_step_counts_keep_gauss_law(cfg, scale, steps):
    """BASELINE.json's step counts (config 1: its own size; configs 3, 5: the recipe on a smaller
    grid): the Gauss residual div- E - rho of the GPU state stays at its initial value up to fp32
    round-off accumulation, nothing is flagged, no particle is lost."""
    pl = psc_inputs.make_config(cfg, scale=scale)
    sim = _sim(pl)
    orc = oracle_for(pl)
    f64 = lambda a: np.ascontiguousarray(a.astype(np.float64))

    def residual():
        cur = gpu_cols(sim)                       # export: absolute positions
        x = f64(cur["x"]) if pl.n[0] > 1 else np.zeros(len(cur["y"]))
        rho = orc.rho(x, f64(cur["y"]), f64(cur["z"]), f64(cur["qw"]))
        E = f64(sim.interior(sim.E).cpu().numpy())
        m = cur["species"] == 0
        rho_e = orc.rho(x[m], f64(cur["y"][m]), f64(cur["z"][m]), f64(cur["qw"][m]))
        return orc.div_minus(E) - rho, np.abs(rho_e).max(), np.sort(cur["id"])

    r0, scale_rho, ids0 = residual()
    sim.step(steps)
    assert sim.psc.status() == 0
    r1, _, ids1 = residual()
    assert np.array_equal(ids0, ids1)
    # one fp32 rounding of J per step and node, accumulated: well below 1e-4 of the species density
    assert np.abs(r1 - r0).max() < 1e-4 * scale_rho, np.abs(r1 - r0).max() / scale_rho


def test_column_sets_have_fixed_roles():
    """include/psc.h (psc_bind_particles): the primary set is the dense one -- n entries, never
    written beyond -- and the secondary set holds the store, whatever the sequence of calls: sort,
    steps with re-layouts, export, a second sort, psc_step_host entered in the store form."""
    pl = psc_inputs.thermal((1, 16, 16), 150, seed=23, name="dense")
    vy = 0.33 * pl.dx[1] / pl.dt
    pl.uy = pl.uy + float(vy / np.sqrt(1.0 - vy * vy))       # a third of the particles leave per step
    pl.qw = pl.qw * 1e-2
    extra, g = 900, torch.Generator().manual_seed(4)         # a clump that outgrows its cell's room
    for k in ("x", "ux", "uz"):
        setattr(pl, k, torch.cat([getattr(pl, k), torch.zeros(extra)]))
    pl.y = torch.cat([pl.y, 5.0 + torch.rand(extra, generator=g)])
    pl.z = torch.cat([pl.z, 9.0 + torch.rand(extra, generator=g)])
    pl.uy = torch.cat([pl.uy, torch.full((extra,), float(pl.uy[0]))])
    pl.qw = torch.cat([pl.qw, torch.full((extra,), float(pl.qw[0]))])
    pl.species = torch.cat([pl.species, torch.zeros(extra, dtype=torch.int32)])
    pl.id = torch.arange(pl.y.numel(), dtype=torch.int32)
    sim = _sim(pl)
    dense, store = sim.sets[0]["y"].data_ptr(), sim.sets[1]["y"].data_ptr()
    assert sim.sets[0]["y"].numel() == sim.np + sim.GUARD < sim.capacity
    cur = lambda: sim.psc.particles_current()["y"]
    assert cur() == dense and sim.psc.particles_form() == 0
    sim.psc.particles_sort()
    assert cur() == store and sim.psc.particles_form() == 1
    sim.step(4)
    info = sim.psc.store_info()
    assert info["relayouts"] >= 1 and cur() == store, info
    sim.psc.particles_sort()                                 # a store sorted again stays where it is
    assert cur() == store
    sim.psc.particles_export()
    assert cur() == dense and sim.psc.particles_form() == 0
    sim.step(2)
    assert cur() == store
    # psc_step_host while the particles are in the store: the host's list goes to the dense set
    host = {c: (None if t is None else t.cpu().pin_memory()) for c, t in sim.gather(absolute=True).items()
            if c != "key"}
    hE, hB = sim.E.cpu().pin_memory(), sim.B.cpu().pin_memory()
    sim.psc.step_host(sim.np, host, hE, hB, None, 2)
    assert cur() == dense and sim.psc.particles_form() == 0
    assert np.array_equal(np.sort(host["id"].numpy()), np.arange(sim.np))
    sim.step(1)
    assert cur() == store
    assert sim.psc.status() == 0
    assert sim.guards_intact()
    m = sim.memory()
    assert m["multiplier"] == pytest.approx(1 + sim.capacity / sim.np)


@pytest.mark.parametrize("kind", ["2d", "3d", "2d-o2", "beam"])
def test_a_non_finite_momentum_is_flagged_and_the_particle_is_kept(kind):
    """one particle with u = NaN, one with u = +inf: PSC_F_NAN is raised, and both stay in the
    population (in their cells, old offsets) instead of leaving under the code of "no move" that no
    cell collects; every other particle still moves"""
    if kind == "2d":
        pl = psc_inputs.make_config(1)
    elif kind == "3d":
        pl = psc_inputs.thermal((12, 20, 8), 5, seed=12, dx=(0.8, 1.25, 0.5), name="3d")
    elif kind == "2d-o2":
        pl = psc_inputs.thermal((1, 24, 40), 9, seed=14, order=2, dx=(1.0, 0.5, 2.0), name="o2")
    else:
        pl = psc_inputs.make_config(5, scale=(8, 8, 32))
    n = pl.n_particles
    bad = [n // 3, 2 * n // 3]
    pl.ux[bad[0]] = float("nan")
    pl.uz[bad[1]] = float("inf")
    sim = _sim(pl)
    sim.psc.particles_sort()
    before = sim.gather()
    # the NaN current spreads by a stencil width per step; the steps taken here keep the number of
    # affected particles below the spill list's n/4 entries (8^2 x 32 cells at order 2: one step)
    for it in range(1 if kind == "beam" else 2):
        sim.step(1)
        flags = sim.psc.status()
        assert flags & psc.PSC_F_NAN and not flags & psc.PSC_F_OVERFLOW
        g = sim.gather()
        ids = g["id"].cpu().numpy()
        assert np.array_equal(np.sort(ids), np.arange(n)), (kind, it)      # nobody lost or duplicated
    pos = {int(i): k for k, i in enumerate(before["id"].cpu().numpy())}
    now = {int(i): k for k, i in enumerate(ids)}
    for b in bad:                                                          # same cell, same offsets
        assert int(g["key"][now[b]]) == int(before["key"][pos[b]])
        for c in ("y", "z"):
            assert float(g[c][now[b]]) == float(before[c][pos[b]])
    info = sim.psc.store_info()
    assert info["spilled"] >= 2 or info["inserted"] + info["relayouts"] > 0    # they travel through the spill list


def test_image_size_follows_cells_that_grow_between_layouts():
    """a column of cells whose particles all walk through the next column: the cell counts there
    nearly double without any re-layout (the spare room suffices); the status block's largest count and, from the
    host's next look at it, the per-warp image of the kernels follow"""
    pl = psc_inputs.thermal((1, 16, 16), 20, vth_e=1e-4, vth_i=1e-4, seed=3, name="walk")
    pl.qw = pl.qw * 1e-6                                    # (no fields to speak of)
    v = 0.9
    walkers = (pl.y >= 4.0) & (pl.y < 5.0)
    pl.uy = torch.where(walkers, torch.full_like(pl.uy, v / np.sqrt(1.0 - v * v)), pl.uy)
    sim = _sim(pl)
    sim.psc.particles_sort()
    i0 = sim.psc.store_info()
    assert i0["max_count"] == 40 and i0["image_slots"] == 96
    sim.step(3)                     # 0.45 cell per step: most walkers are in the next column, none beyond
    assert sim.psc.status() == 0
    i1 = sim.psc.store_info()
    assert i1["relayouts"] == 0 and 65 <= i1["max_count"] <= 80, i1
    assert i1["image_slots"] == 128                         # e.g. 74 + 74/8 + 24 -> 128
    sim.step(3)
    g = sim.gather()
    assert np.array_equal(np.sort(g["id"].cpu().numpy()), np.arange(sim.np))
    assert sim.psc.status() == 0
