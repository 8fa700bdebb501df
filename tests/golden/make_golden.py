"""Writes tests/golden/t0_two_steps.txt: two PIC steps of eight particles on a 1x6x5 (order 1)
and a 4x5x6 (order 2) periodic grid, computed by the DEFINITION-LEVEL brute force only
(oracle/brute_force.py: gather over all grid points with Eq. 29-31 typed out, PAPER.md:183-193;
currents from the flux definition / whole-grid density decomposition; FDTD of
Eq. 17-18 with np.roll).  The paper prints no numeric worked example for this path, so this
fixture is a stored result of the oracle's slowest, most literal tier -- a guard against the
stencil oracle and the brute force drifting together.  Nothing here touches the CUDA path.

    python tests/golden/make_golden.py        # rewrites the fixture (inputs are fp32-exact)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle.brute_force import BruteForce  # noqa: E402

CASES = [("o1_2d", 1, (1, 6, 5)), ("o2_3d", 2, (4, 5, 6))]
Q, M = [-1.0, 1.0], [1.0, 4.0]
DX = (1.0, 1.0, 1.0)
NPART, NSTEPS = 8, 2


def inputs(order, n):
    """seeded inputs, rounded to fp32 so that the fp32 CUDA path can take exactly the same"""
    rng = np.random.default_rng(13107866 + order)
    f32 = lambda a: np.asarray(a, dtype=np.float32).astype(np.float64)
    pos = np.stack([f32(rng.random(NPART) * n[d] * DX[d]) if n[d] > 1 else np.zeros(NPART)
                    for d in range(3)], axis=1)
    u = f32(0.4 * rng.standard_normal((NPART, 3)))
    qw = f32(np.where(np.arange(NPART) % 2 == 0, -1.0, 1.0) * (0.5 + rng.random(NPART)))
    species = (np.arange(NPART) % 2).astype(np.int32)
    shape = (3, n[2], n[1], n[0])
    E = f32(0.2 * rng.standard_normal(shape))
    B = f32(0.2 * rng.standard_normal(shape))
    dt = 0.5 / np.sqrt(sum(1.0 / DX[d] ** 2 for d in range(3) if n[d] > 1))
    return pos, u, qw, species, E, B, float(np.float32(dt))


def run(order, n):
    pos, u, qw, species, E, B, dt = inputs(order, n)
    bf = BruteForce(n, DX, dt, order, Q, M)
    xs, us = pos.copy(), u.copy()
    for _ in range(NSTEPS):
        J = bf.step(E, B, xs, us, qw, species)
    return xs, us, E, B, J


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "t0_two_steps.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py (oracle/brute_force.py only); see its docstring\n")
        for name, order, n in CASES:
            xs, us, E, B, J = run(order, n)
            for key, arr in (("x", xs), ("u", us), ("E", E), ("B", B), ("J", J)):
                f.write("%s %s %s\n" % (name, key, " ".join("%.17g" % v for v in np.asarray(arr).ravel())))
    print("wrote", out)


if __name__ == "__main__":
    main()
