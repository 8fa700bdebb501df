"""Pins of the oracle's grid part: discrete operators, FDTD leap-frog, B-splines, gather.

Each test checks oracle/psc_oracle.c against something the paper or the mathematics fixes, never
against itself (citations are PAPER.md lines)."""
import numpy as np
import pytest

from oracle.brute_force import BruteForce, b0, b1, b2
from oracle.psc_oracle import Oracle

GRIDS = [((6, 5, 7), (1.0, 0.8, 1.3)), ((1, 8, 6), (1.0, 1.0, 0.7)), ((8, 1, 1), (0.9, 1.0, 1.0))]


@pytest.mark.parametrize("n,dx", GRIDS)
def test_div_curl_identities(n, dx):
    """Eq. 23: div+ curl+ = 0 and div- curl- = 0 to round-off."""
    orc = Oracle(n, dx, 0.1, 1, [-1.0], [1.0])
    rng = np.random.default_rng(1)
    F = rng.standard_normal(orc.fshape)
    assert np.abs(orc.div_plus(orc.curl_plus(F))).max() < 1e-13 * 50
    assert np.abs(orc.div_minus(orc.curl_minus(F))).max() < 1e-13 * 50
    # and the operators are not trivially zero
    assert np.abs(orc.curl_plus(F)).max() > 0.1
    assert np.abs(orc.div_minus(F)).max() > 0.1


def test_curl_on_linear_combination_of_modes():
    """curl+ / curl- of a single Fourier mode sampled at the Yee points is i K x F with
    K_d = (2/dx_d) sin(k_d dx_d/2): fixes sign, component order and staggering of Eq. 12-13."""
    n, dx = (8, 6, 10), (1.0, 0.75, 1.25)
    orc = Oracle(n, dx, 0.1, 1, [-1.0], [1.0])
    mode = (1, 2, 3)
    k = [2 * np.pi * mode[d] / (n[d] * dx[d]) for d in range(3)]
    K = np.array([2 / dx[d] * np.sin(k[d] * dx[d] / 2) for d in range(3)])
    stagE = np.array([[0.5, 0, 0], [0, 0.5, 0], [0, 0, 0.5]])
    stagB = np.array([[0, 0.5, 0.5], [0.5, 0, 0.5], [0.5, 0.5, 0]])
    kk, jj, ii = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")

    def phase(stag):
        return (k[0] * (ii + stag[0]) * dx[0] + k[1] * (jj + stag[1]) * dx[1] + k[2] * (kk + stag[2]) * dx[2])

    A = np.array([0.3, -1.1, 0.7])
    # E-staggered field A cos(phase): curl+ gives -(K x A) sin(phase) at the B points
    F = np.stack([A[c] * np.cos(phase(stagE[c])) for c in range(3)])
    want = np.stack([-np.cross(K, A)[c] * np.sin(phase(stagB[c])) for c in range(3)])
    assert np.abs(orc.curl_plus(F) - want).max() < 1e-13
    # B-staggered field: curl- lands on the E points
    F = np.stack([A[c] * np.cos(phase(stagB[c])) for c in range(3)])
    want = np.stack([-np.cross(K, A)[c] * np.sin(phase(stagE[c])) for c in range(3)])
    assert np.abs(orc.curl_minus(F) - want).max() < 1e-13


@pytest.mark.parametrize("n,dx,mode", [((8, 6, 10), (1.0, 0.75, 1.25), (1, 2, -1)),
                                       ((1, 16, 12), (1.0, 1.0, 1.0), (0, 3, 2))])
def test_fdtd_vacuum_eigenmode(n, dx, mode):
    """Leap-frog Eq. 17-18 in vacuum: a plane wave with sin^2(W dt/2)/dt^2 = sum sin^2(k dx/2)/dx^2,
    E0 perp K, B0 = K x E0 / ((2/dt) sin(W dt/2)) stays on the analytic phase for any number of
    steps; div+ B stays 0."""
    dt = 0.5 / np.sqrt(sum(1 / dx[d] ** 2 for d in range(3) if n[d] > 1))
    orc = Oracle(n, dx, dt, 1, [-1.0], [1.0])
    k = [2 * np.pi * mode[d] / (n[d] * dx[d]) for d in range(3)]
    K = np.array([2 / dx[d] * np.sin(k[d] * dx[d] / 2) for d in range(3)])
    Wt = np.sqrt(K @ K)                       # (2/dt) sin(W dt/2)
    W = 2 / dt * np.arcsin(Wt * dt / 2)
    E0 = np.cross(K, [0.3, -0.4, 0.9])
    E0 /= np.linalg.norm(E0)
    B0 = np.cross(K, E0) / Wt
    stagE = np.array([[0.5, 0, 0], [0, 0.5, 0], [0, 0, 0.5]])
    stagB = np.array([[0, 0.5, 0.5], [0.5, 0, 0.5], [0.5, 0.5, 0]])
    kk, jj, ii = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")

    def wave(amp, stag, t):
        return np.stack([amp[c] * np.cos(k[0] * (ii + stag[c][0]) * dx[0] + k[1] * (jj + stag[c][1]) * dx[1]
                                         + k[2] * (kk + stag[c][2]) * dx[2] - W * t) for c in range(3)])

    E = wave(E0, stagE, 0.5 * dt)
    B = wave(B0, stagB, 0.0)
    J = orc.zeros_field()
    nsteps = 200
    for _ in range(nsteps):
        orc.push_b(E, B, 0.5)
        orc.push_b(E, B, 0.5)
        orc.push_e(E, B, J, 1.0)
    assert np.abs(E - wave(E0, stagE, (nsteps + 0.5) * dt)).max() < 1e-12
    assert np.abs(B - wave(B0, stagB, nsteps * dt)).max() < 1e-12
    assert np.abs(orc.div_plus(B)).max() < 1e-13


def test_push_e_current_sign_and_frac():
    """Eq. 17: a uniform J with no B lowers E by dt*J (frac scales it)."""
    orc = Oracle((4, 4, 4), (1, 1, 1), 0.25, 1, [-1.0], [1.0])
    E, B, J = orc.zeros_field(), orc.zeros_field(), orc.zeros_field()
    J[1] = 2.0
    orc.push_e(E, B, J, 1.0)
    assert np.allclose(E[1], -0.5) and np.all(E[0] == 0) and np.all(E[2] == 0)
    orc.push_e(E, B, J, 0.5)
    assert np.allclose(E[1], -0.75)


def test_bsplines_are_convolutions_of_b0():
    """Eq. 30 (read as a convolution, A2): b1 = b0 * b0, b2 = b0 * b1; partition of unity."""
    s = np.linspace(-3, 3, 240001)
    ds = s[1] - s[0]
    for xi in (-1.3, -0.7, -0.2, 0.0, 0.4, 0.9, 1.45):
        c1 = np.sum(b0(xi - s) * b0(s)) * ds
        c2 = np.sum(b0(xi - s) * b1(s)) * ds
        assert abs(c1 - b1(xi)) < 2e-4
        assert abs(c2 - b2(xi)) < 2e-4
    for f in np.linspace(-0.5, 0.5, 11):
        assert abs(sum(b1(f - i) for i in range(-2, 3)) - 1) < 1e-15
        assert abs(sum(b2(f - i) for i in range(-2, 3)) - 1) < 1e-15


@pytest.mark.parametrize("order", [1, 2])
@pytest.mark.parametrize("n", [(6, 7, 8), (1, 8, 6), (6, 1, 8)])
def test_gather_uniform_and_linear(order, n):
    """Eq. 11 with b1/b2 weights reproduces constants and functions linear in x exactly when the
    field is sampled at its own staggered points (weights sum to 1, first moment exact)."""
    dx = (1.0, 0.8, 1.25)
    orc = Oracle(n, dx, 0.1, order, [-1.0], [1.0])
    rng = np.random.default_rng(5)
    stagE = np.array([[0.5, 0, 0], [0, 0.5, 0], [0, 0, 0.5]])
    stagB = np.array([[0, 0.5, 0.5], [0.5, 0, 0.5], [0.5, 0.5, 0]])
    kk, jj, ii = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    a = rng.standard_normal(6)
    g = rng.standard_normal((6, 3))
    for d in range(3):
        if n[d] == 1:
            g[:, d] = 0

    def lin(c, stag):
        return a[c] + g[c, 0] * (ii + stag[0]) * dx[0] + g[c, 1] * (jj + stag[1]) * dx[1] + g[c, 2] * (kk + stag[2]) * dx[2]

    E = np.stack([lin(c, stagE[c]) for c in range(3)])
    B = np.stack([lin(3 + c, stagB[c]) for c in range(3)])
    # keep particles away from the periodic seam where the linear function jumps
    npart = 64
    pos = [np.ascontiguousarray((2.0 + rng.random(npart) * (n[d] - 4.5)) * dx[d]) if n[d] > 1
           else np.full(npart, 0.5 * dx[d]) for d in range(3)]
    EB = orc.gather(E, B, *pos)
    for c in range(6):
        want = a[c] + sum(g[c, d] * pos[d] for d in range(3) if n[d] > 1)
        assert np.abs(EB[:, c] - want).max() < 1e-13 * 20


@pytest.mark.parametrize("order", [1, 2])
@pytest.mark.parametrize("n", [(5, 6, 7), (1, 6, 5)])
def test_gather_t1_equals_t0(order, n):
    """stencil gather == sum over the whole grid with Eq. 31 evaluated directly (random fields,
    particles anywhere including next to the periodic seam)."""
    dx = (1.0, 0.8, 1.25)
    orc = Oracle(n, dx, 0.1, order, [-1.0], [1.0])
    bf = BruteForce(n, dx, 0.1, order, [-1.0], [1.0])
    rng = np.random.default_rng(7)
    E, B = rng.standard_normal(orc.fshape), rng.standard_normal(orc.fshape)
    npart = 12
    pos = [np.ascontiguousarray(rng.random(npart) * n[d] * dx[d]) for d in range(3)]
    pos[1][0] = 0.0            # exactly on a node / the seam
    pos[2][1] = 0.5 * dx[2]    # exactly on a staggered point
    EB = orc.gather(E, B, *pos)
    for a in range(npart):
        Ep, Bp = bf.gather(E, B, (pos[0][a], pos[1][a], pos[2][a]))
        assert np.abs(EB[a, :3] - Ep).max() < 1e-13
        assert np.abs(EB[a, 3:] - Bp).max() < 1e-13


# ------------------------------------------------------------------------------------------------
# Marder's Gauss-law correction

@pytest.mark.parametrize("n,dx", [((8, 6, 10), (1.0, 0.8, 1.25)), ((1, 12, 8), (1.0, 0.5, 2.0))])
def test_marder_fourier_mode_decays_by_the_closed_form_factor(n, dx):
    """a single Fourier mode of the Gauss residual f = div- E - rho is multiplied by
    1 - D sum_d K_d^2, K_d = (2/dx_d) sin(k_d dx_d/2), per pass (div- grad+ is the 7-point
    Laplacian); the residual shrinks (sign of the correction); a Gauss-consistent E is untouched"""
    orc = Oracle(n, dx, 0.1, 1, [-1.0], [1.0])
    rng = np.random.default_rng(3)
    nx, ny, nz = n
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    m = (1 if nx > 1 else 0, 2, 1)
    kv = [2 * np.pi * m[d] / (n[d] * dx[d]) for d in range(3)]
    K2 = sum((2 / dx[d] * np.sin(kv[d] * dx[d] / 2)) ** 2 for d in range(3) if n[d] > 1)
    mode = np.cos(kv[0] * i * dx[0] + kv[1] * j * dx[1] + kv[2] * k * dx[2] + 0.3)
    # a consistent pair (E0, rho0 = div- E0) plus a residual in the shape of the mode
    E = np.ascontiguousarray(rng.normal(size=orc.fshape))
    rho0 = orc.div_minus(E)
    rho = np.ascontiguousarray(rho0 - 0.7 * mode)           # f = div- E - rho = 0.7 mode
    D = 0.4 / sum(4 / dx[d] ** 2 for d in range(3) if n[d] > 1)
    f0 = orc.div_minus(E) - rho
    assert np.abs(f0 - 0.7 * mode).max() < 1e-12
    E1 = E.copy()
    orc.marder(E1, rho, D, 1)
    f1 = orc.div_minus(E1) - rho
    assert np.abs(f1 - (1 - D * K2) * f0).max() < 1e-12
    assert np.abs(f1).max() < np.abs(f0).max()
    orc.marder(E1, rho, D, 2)
    f3 = orc.div_minus(E1) - rho
    assert np.abs(f3 - (1 - D * K2) ** 3 * f0).max() < 1e-12
    # the correction is a pure gradient: it never changes curl+ E (Faraday's law is untouched)
    assert np.abs(orc.curl_plus(E1) - orc.curl_plus(E)).max() < 1e-12
    # div- E = rho: nothing to correct
    E2 = E.copy()
    orc.marder(E2, rho0, D, 5)
    assert np.abs(E2 - E).max() < 1e-13
    # a random residual decays monotonically in the max-norm of its spectrum: 30 passes at the
    # stability limit D sum 4/dx^2 = 1 remove at least the upper half of the spectrum
    rho_r = np.ascontiguousarray(rho0 + rng.normal(size=rho0.shape))
    rho_r -= (rho_r - rho0).mean()                           # (the mean of the residual cannot be removed)
    E3 = E.copy()
    r0 = np.abs(orc.div_minus(E3) - rho_r).max()
    orc.marder(E3, rho_r, 1.0 / sum(4 / dx[d] ** 2 for d in range(3) if n[d] > 1), 30)
    assert np.abs(orc.div_minus(E3) - rho_r).max() < 0.8 * r0


# ------------------------------------------------------------------------------------------------
# alternating-order gather ([22]; A29)

@pytest.mark.parametrize("order", [1, 2])
@pytest.mark.parametrize("n", [(5, 6, 7), (1, 6, 5)])
def test_alternating_gather_t1_equals_t0_and_closed_forms(order, n):
    """scheme 1: along a direction in which a component is half-staggered the weight is one order
    lower (b0 / b1 instead of b1 / b2).  T1 == the all-grid sum with those shapes; a uniform field
    is reproduced; order 2 still reproduces a field linear in x (b1 does), order 1 returns the
    value of the NEAREST staggered point along the staggered direction; and the unstaggered
    directions are untouched (a component that varies only along them equals the standard gather)."""
    dx = (1.0, 0.8, 1.25)
    orc = Oracle(n, dx, 0.1, order, [-1.0], [1.0], scheme=1)
    std = Oracle(n, dx, 0.1, order, [-1.0], [1.0], scheme=0)
    bf = BruteForce(n, dx, 0.1, order, [-1.0], [1.0], scheme=1)
    rng = np.random.default_rng(70 + order)
    E, B = rng.standard_normal(orc.fshape), rng.standard_normal(orc.fshape)
    npart = 12
    pos = [np.ascontiguousarray(rng.random(npart) * n[d] * dx[d]) for d in range(3)]
    EB = orc.gather(E, B, *pos)
    for a in range(npart):
        Ep, Bp = bf.gather(E, B, (pos[0][a], pos[1][a], pos[2][a]))
        assert np.abs(EB[a, :3] - Ep).max() < 1e-13
        assert np.abs(EB[a, 3:] - Bp).max() < 1e-13
    assert np.abs(EB - std.gather(E, B, *pos)).max() > 1e-3         # it IS a different scheme
    # uniform field
    U = np.ones(orc.fshape) * np.array([0.3, -1.0, 2.0])[:, None, None, None]
    EBu = orc.gather(U, 2 * U, *pos)
    assert np.abs(EBu[:, :3] - [0.3, -1.0, 2.0]).max() < 1e-14 and np.abs(EBu[:, 3:] - [0.6, -2.0, 4.0]).max() < 1e-14
    # E_z varying along z only (its staggered direction), particles away from the seam
    kk = np.arange(n[2])[:, None, None] * np.ones((1, n[1], n[0]))
    F = np.zeros(orc.fshape)
    F[2] = 1.5 + 0.25 * (kk + 0.5) * dx[2]                          # linear in z, sampled at k + 1/2
    z = np.ascontiguousarray((1.6 + rng.random(npart) * (n[2] - 3.5)) * dx[2])
    got = orc.gather(F, F, pos[0], pos[1], z)[:, 2]
    if order == 2:
        assert np.abs(got - (1.5 + 0.25 * z)).max() < 1e-13
    else:
        nearest = np.floor(z / dx[2]) + 0.5                          # the half point of the particle's cell
        assert np.abs(got - (1.5 + 0.25 * nearest * dx[2])).max() < 1e-13
    # E_z varying along y only (unstaggered for E_z): same as the standard scheme
    jj = np.arange(n[1])[None, :, None] * np.ones((n[2], 1, n[0]))
    G = np.zeros(orc.fshape)
    G[2] = np.sin(2 * np.pi * jj / n[1])
    assert np.abs(orc.gather(G, G, *pos)[:, 2] - std.gather(G, G, *pos)[:, 2]).max() < 1e-14
