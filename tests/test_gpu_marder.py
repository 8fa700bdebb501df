"""GPU parity of the node charge density and of Marder's Gauss-law correction
 against the fp64 oracle, and what the correction is for: a long fp32 run whose
Gauss residual stays bounded with it and drifts without."""
import numpy as np
import pytest
import torch

import psc_inputs
from tests.util import gpu_state, oracle_for, positions_f64, rel_maxnorm, smooth_fields

pytestmark = pytest.mark.gpu
TOL = 1e-5


def _sim(pl, **kw):
    from paper_1310_7866_b200.harness import Simulation

    return Simulation(pl, **kw)


def _cases(kind):
    if kind == "2d":
        return psc_inputs.make_config(1)
    if kind == "2d-o2":
        return psc_inputs.thermal((1, 24, 40), 9, seed=14, order=2, dx=(1.0, 0.5, 2.0), name="o2")
    if kind == "3d":
        return psc_inputs.thermal((12, 20, 8), 5, seed=12, dx=(0.8, 1.25, 0.5), name="3d")
    return psc_inputs.make_config(5, scale=(8, 8, 32))


def _rho_interior(sim):
    rho = torch.zeros(sim.psc.field_shape[1:], dtype=torch.float32, device="cuda")
    sim.psc.charge_density(rho)
    g, n = sim.g, sim.n
    full = rho.cpu().numpy()
    inner = full[g[2]:g[2] + n[2], g[1]:g[1] + n[1], g[0]:g[0] + n[0]]
    return full, inner


@pytest.mark.parametrize("kind", ["2d", "2d-o2", "3d", "beam"])
def test_charge_density_matches_oracle(kind):
    """rho on the nodes from the cell store, after a few steps (residents + records waiting in
    the exchange rows), against orc_rho of the same particles; ghosts are periodic images"""
    pl = _cases(kind)
    smooth_fields(pl, 0.05, seed=21)
    sim = _sim(pl)
    sim.step(3)
    st = gpu_state(sim)
    pos = positions_f64(st, pl)
    orc = oracle_for(pl)
    f64 = lambda a: np.ascontiguousarray(a.astype(np.float64))
    m = st["species"] == 0
    want_e = orc.rho(*[np.ascontiguousarray(p[m]) for p in pos], f64(st["qw"][m]))
    want = orc.rho(pos[0], pos[1], pos[2], f64(st["qw"]))
    full, got = _rho_interior(sim)
    assert np.abs(got - want).max() <= TOL * np.abs(want_e).max()     # vs the density of one species
    g, n = sim.g, sim.n
    ez, ey, ex = full.shape
    kk, jj, ii = np.meshgrid(np.arange(ez), np.arange(ey), np.arange(ex), indexing="ij")
    img = got[(kk - g[2]) % n[2], (jj - g[1]) % n[1], (ii - g[0]) % n[0]]
    assert np.array_equal(full, img)
    assert sim.psc.status() == 0


@pytest.mark.parametrize("kind", ["2d", "3d", "beam"])
def test_marder_matches_oracle(kind):
    """three passes of E += D grad+ (div- E - rho) on a state with a deliberately broken Gauss law"""
    pl = _cases(kind)
    smooth_fields(pl, 0.05, seed=33)                 # E not consistent with rho: a large residual
    sim = _sim(pl)
    sim.psc.particles_sort()
    st = gpu_state(sim)
    pos = positions_f64(st, pl)
    orc = oracle_for(pl)
    f64 = lambda a: np.ascontiguousarray(a.astype(np.float64))
    rho = orc.rho(pos[0], pos[1], pos[2], f64(st["qw"]))
    E = f64(sim.interior(sim.E).cpu().numpy())
    D = 0.8 / sum(4.0 / pl.dx[d] ** 2 for d in range(3) if pl.n[d] > 1)
    r0 = np.abs(orc.div_minus(E) - rho).max()
    orc.marder(E, rho, D, 3)
    r1 = np.abs(orc.div_minus(E) - rho).max()
    assert r1 < r0
    sim.psc.marder(D, 3)
    assert rel_maxnorm(sim.interior(sim.E).cpu().numpy(), E) < TOL
    # ghost points stay periodic images of the interior
    G = sim.E.clone()
    sim.psc.fill_ghosts(0)
    assert torch.equal(G, sim.E)
    # an over-large diffusion number is refused (PSC_ERR_CFL), nothing else is touched
    import paper_1310_7866_b200 as psc
    assert psc.lib().psc_marder(sim.psc._h, None, 1.3 * D / 0.8, 1) == -4


def test_marder_keeps_gauss_law_over_a_long_fp32_run():
    """config 1 for 3000 steps.  Without the correction the Gauss residual
    div- E - rho random-walks upwards with the fp32 rounding of j; with one Marder pass every
    ten steps it stays at its early level."""
    pl = psc_inputs.make_config(1)
    orc = oracle_for(pl)
    f64 = lambda a: np.ascontiguousarray(a.astype(np.float64))
    D = 0.5 / sum(4.0 / pl.dx[d] ** 2 for d in range(3) if pl.n[d] > 1)

    def residual(sim):
        st = gpu_state(sim)
        pos = positions_f64(st, pl)
        rho = orc.rho(pos[0], pos[1], pos[2], f64(st["qw"]))
        m = st["species"] == 0
        rho_e = orc.rho(*[np.ascontiguousarray(p[m]) for p in pos], f64(st["qw"][m]))
        E = f64(sim.interior(sim.E).cpu().numpy())
        return np.abs(orc.div_minus(E) - rho).max() / np.abs(rho_e).max()

    free, kept = _sim(pl), _sim(pl)
    free.step(300)
    early = residual(free)
    free.step(2700)
    for _ in range(300):
        kept.step(10)
        kept.psc.marder(D, 1)
    r_free, r_kept = residual(free), residual(kept)
    assert free.psc.status() == 0 and kept.psc.status() == 0
    assert r_kept < 0.5 * r_free, (early, r_free, r_kept)
    assert r_kept < 3 * early, (early, r_free, r_kept)
