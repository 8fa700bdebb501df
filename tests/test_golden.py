"""tests/golden/t0_two_steps.txt (written by tests/golden/make_golden.py from the definition-level
brute force only): the stencil oracle must reproduce it to round-off (CPU), the CUDA path within
the parity tolerance (GPU)."""
import importlib.util
import os

import numpy as np
import pytest

from oracle.psc_oracle import Oracle

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
mg = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(mg)


def _stored():
    out = {}
    with open(os.path.join(HERE, "golden", "t0_two_steps.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            name, key, *vals = line.split()
            out[(name, key)] = np.array([float(v) for v in vals])
    return out


@pytest.mark.parametrize("case", mg.CASES, ids=[c[0] for c in mg.CASES])
def test_stencil_oracle_reproduces_the_stored_brute_force_result(case):
    name, order, n = case
    g = _stored()
    pos, u, qw, species, E, B, dt = mg.inputs(order, n)
    orc = Oracle(n, mg.DX, dt, order, mg.Q, mg.M)
    J = orc.zeros_field()
    p = [np.ascontiguousarray(pos[:, d]) for d in range(3)]
    v = [np.ascontiguousarray(u[:, d]) for d in range(3)]
    E, B = np.ascontiguousarray(E), np.ascontiguousarray(B)
    orc.step(E, B, J, *p, *v, np.ascontiguousarray(qw), species, mg.NSTEPS)
    for d in range(3):
        L = n[d] * mg.DX[d]
        dd = np.abs((p[d] - g[(name, "x")].reshape(-1, 3)[:, d] + 0.5 * L) % L - 0.5 * L)
        assert dd.max() < 1e-12
        assert np.abs(v[d] - g[(name, "u")].reshape(-1, 3)[:, d]).max() < 1e-12
    for key, arr in (("E", E), ("B", B), ("J", J)):
        assert np.abs(arr.ravel() - g[(name, key)]).max() < 1e-12, key


@pytest.mark.gpu
@pytest.mark.parametrize("case", mg.CASES, ids=[c[0] for c in mg.CASES])
def test_cuda_path_matches_the_stored_brute_force_result(case):
    import torch

    import psc_inputs
    from paper_1310_7866_b200.harness import Simulation

    name, order, n = case
    g = _stored()
    pos, u, qw, species, E, B, dt = mg.inputs(order, n)
    t32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
    pl = psc_inputs.Plasma("golden-" + name, n, mg.DX, dt, order, mg.Q, mg.M, mg.NSTEPS,
                           x=t32(pos[:, 0]), y=t32(pos[:, 1]), z=t32(pos[:, 2]),
                           ux=t32(u[:, 0]), uy=t32(u[:, 1]), uz=t32(u[:, 2]), qw=t32(qw),
                           species=torch.from_numpy(species.copy()),
                           id=torch.arange(mg.NPART, dtype=torch.int32), E=t32(E), B=t32(B))
    sim = Simulation(pl)
    sim.step(mg.NSTEPS)
    assert sim.psc.status() == 0
    sim.psc.particles_export()
    cur = {k: v.cpu().numpy() for k, v in sim.current().items()}
    o = np.argsort(cur["id"], kind="stable")
    gx, gu = g[(name, "x")].reshape(-1, 3), g[(name, "u")].reshape(-1, 3)
    for d, c in enumerate(("x", "y", "z")):
        if n[d] == 1:
            continue
        L = n[d] * mg.DX[d]
        dd = np.abs((cur[c][o].astype(np.float64) - gx[:, d] + 0.5 * L) % L - 0.5 * L)
        assert dd.max() / L < 1e-5
    for d, c in enumerate(("ux", "uy", "uz")):
        assert np.abs(cur[c][o] - gu[:, d]).max() < 1e-5 * np.abs(gu).max()
    for key, F in (("E", sim.E), ("B", sim.B), ("J", sim.J)):
        got = sim.interior(F).cpu().numpy().astype(np.float64).ravel()
        want = g[(name, key)]
        assert np.abs(got - want).max() <= 1e-5 * np.abs(want).max(), key
