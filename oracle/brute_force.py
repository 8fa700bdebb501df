"""T0: definition-level brute force of the PIC step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Pure numpy / Python loops over ALL grid points with periodic minimum-image distances; the
B-splines are Eq. 29-31 typed out; the order-1 current is the time integral
of the instantaneous flux that makes Eq. 25 hold for b1-assigned charge; nothing
here uses a stencil, a cell index or a closed-form deposit weight.  Used on 1-8 particles and
<= 8^3 cells to pin oracle/psc_oracle.c (T1).  Shares no code with T1 or with the CUDA path.

Fields: float64 [3, nz, ny, nx], periodic, no ghosts (same staggering as psc_oracle.c).
"""
from __future__ import annotations

import numpy as np

STAG_E = ((0.5, 0.0, 0.0), (0.0, 0.5, 0.0), (0.0, 0.0, 0.5))  # Eq. 20
STAG_B = ((0.0, 0.5, 0.5), (0.5, 0.0, 0.5), (0.5, 0.5, 0.0))  # Eq. 21


def b0(xi):
    xi = np.asarray(xi, dtype=np.float64)
    return np.where(np.abs(xi) < 0.5, 1.0, 0.0)  # Eq. 29


def b1(xi):
    xi = np.asarray(xi, dtype=np.float64)
    return np.where((xi >= -1) & (xi <= 0), 1 + xi, np.where((xi >= 0) & (xi <= 1), 1 - xi, 0.0))


def b2(xi):
    xi = np.asarray(xi, dtype=np.float64)
    return np.where(
        (xi >= -1.5) & (xi <= -0.5), 0.5 * (1.5 + xi) ** 2,
        np.where((xi >= -0.5) & (xi <= 0.5), 0.75 - xi ** 2,
                 np.where((xi >= 0.5) & (xi <= 1.5), 0.5 * (1.5 - xi) ** 2, 0.0)))


def _min_image(d, n):
    """distance in cells wrapped into [-n/2, n/2)"""
    return (d + 0.5 * n) % n - 0.5 * n


def _weights_1d(shape, n, xi, stag):
    """weights of all n staggered points (i + stag) for a particle at xi (cells).  n == 1: [1]."""
    if n == 1:
        return np.ones(1)
    nodes = np.arange(n, dtype=np.float64) + stag
    return shape(_min_image(xi - nodes, n))


class BruteForce:
    def __init__(self, n, dx, dt, order, q, m, scheme=0):
        self.n = tuple(int(v) for v in n)
        self.dx = tuple(float(v) for v in dx)
        self.dt = float(dt)
        self.order = int(order)
        self.q = list(q)
        self.m = list(m)
        self.s = b1 if order == 1 else b2  # weights are one order above the particle shape
        # alternating order: one order lower along half-staggered directions
        self.s_stag = (b0 if order == 1 else b1) if scheme == 1 else self.s
        self.dV = self.dx[0] * self.dx[1] * self.dx[2]

    # ---- Eq. 11 with piecewise-constant fields: E_p = sum_grid F * s s s -------------------
    def gather_one(self, F, c, stag, pos):
        nx, ny, nz = self.n
        sh = [self.s_stag if stag[d] != 0.0 else self.s for d in range(3)]
        wx = _weights_1d(sh[0], nx, pos[0] / self.dx[0], stag[0])
        wy = _weights_1d(sh[1], ny, pos[1] / self.dx[1], stag[1])
        wz = _weights_1d(sh[2], nz, pos[2] / self.dx[2], stag[2])
        tot = 0.0
        for k in range(nz):
            for j in range(ny):
                for i in range(nx):
                    tot += F[c, k, j, i] * wx[i] * wy[j] * wz[k]
        return tot

    def gather(self, E, B, pos):
        Ep = [self.gather_one(E, c, STAG_E[c], pos) for c in range(3)]
        Bp = [self.gather_one(B, c, STAG_B[c], pos) for c in range(3)]
        return np.array(Ep), np.array(Bp)

    # ---- rho on nodes ----------------------------------------------------------------------
    def rho(self, xs, qws):
        nx, ny, nz = self.n
        out = np.zeros((nz, ny, nx))
        for pos, qw in zip(xs, qws):
            wx = _weights_1d(self.s, nx, pos[0] / self.dx[0], 0.0)
            wy = _weights_1d(self.s, ny, pos[1] / self.dx[1], 0.0)
            wz = _weights_1d(self.s, nz, pos[2] / self.dx[2], 0.0)
            out += qw / self.dV * wz[:, None, None] * wy[None, :, None] * wx[None, None, :]
        return out

    # ---- Boris (Eq. 27-28, written independently of the C code: rotation-matrix-free form) --
    def boris(self, u, Ep, Bp, s):
        h = self.q[s] * self.dt / (2.0 * self.m[s])
        um = np.asarray(u, dtype=np.float64) + h * Ep
        gm = np.sqrt(1.0 + um @ um)
        t = h * Bp / gm
        up = um + np.cross(um, t)
        upl = um + np.cross(up, 2.0 * t / (1.0 + t @ t))
        return upl + h * Ep

    # ---- order 1 current: time integral of the instantaneous flux --------------------------
    #   j_c(i_c+1/2, i_e, i_f)(t) = (qw/dV) v_c 1[xi_c(t) in [i_c, i_c+1)] b1(xi_e(t)-i_e) b1(xi_f(t)-i_f)
    # (this is the only j for which d/dt of b1-assigned rho + div- j = 0 holds at every instant);
    # j^{n+1} is its average over the step along the straight line x0 -> x1.
    def _flux_integrand(self, c, xi, v):
        """instantaneous j_c on the whole grid, array [nz, ny, nx], for in-grid position xi (cells)"""
        w = []
        for d in range(3):
            n = self.n[d]
            if n == 1:
                w.append(np.ones(1))
            elif d == c:
                # indicator of xi_c in [i, i+1): b0 centred on i + 1/2 (closed below, open above)
                dist = _min_image(xi[d] - (np.arange(n) + 0.5), n)
                w.append(np.where((dist >= -0.5) & (dist < 0.5), 1.0, 0.0))
            else:
                w.append(b1(_min_image(xi[d] - np.arange(n, dtype=np.float64), n)))
        return v[c] * w[2][:, None, None] * w[1][None, :, None] * w[0][None, None, :]

    def vb_midpoint(self, x0, x1, v, qw, nsamples):
        """plain midpoint rule on the definition (error O(1/nsamples) from the indicator jump);
        the same integrand as _flux_integrand, evaluated for all sample times at once"""
        nx, ny, nz = self.n
        J = np.zeros((3, nz, ny, nx))
        xi0 = np.array([x0[d] / self.dx[d] for d in range(3)])
        xi1 = np.array([x1[d] / self.dx[d] for d in range(3)])
        t = (np.arange(nsamples) + 0.5) / nsamples
        for c in range(3):
            w = []
            for d in range(3):
                n = self.n[d]
                xi = xi0[d] + t * (xi1[d] - xi0[d])
                if n == 1:
                    w.append(np.ones((nsamples, 1)))
                elif d == c:
                    dist = _min_image(xi[:, None] - (np.arange(n) + 0.5)[None, :], n)
                    w.append(np.where((dist >= -0.5) & (dist < 0.5), 1.0, 0.0))
                else:
                    w.append(b1(_min_image(xi[:, None] - np.arange(n, dtype=np.float64)[None, :], n)))
            J[c] = v[c] * np.einsum("mk,mj,mi->kji", w[2], w[1], w[0])
        return J * (qw / self.dV / nsamples)

    def vb_exact(self, x0, x1, v, qw):
        """same integral, exact: the integrand is a polynomial of degree <= 2 in t between the
        times at which some xi_d(t) is an integer, so 3-point Gauss-Legendre per piece is exact."""
        nx, ny, nz = self.n
        J = np.zeros((3, nz, ny, nx))
        xi0 = np.array([x0[d] / self.dx[d] for d in range(3)])
        xi1 = np.array([x1[d] / self.dx[d] for d in range(3)])
        cuts = [0.0, 1.0]
        for d in range(3):
            if self.n[d] == 1 or xi1[d] == xi0[d]:
                continue
            lo, hi = sorted((xi0[d], xi1[d]))
            for node in range(int(np.floor(lo)), int(np.ceil(hi)) + 1):
                t = (node - xi0[d]) / (xi1[d] - xi0[d])
                if 0.0 < t < 1.0:
                    cuts.append(t)
        cuts = sorted(cuts)
        gx, gw = np.polynomial.legendre.leggauss(3)
        for ta, tb in zip(cuts[:-1], cuts[1:]):
            if tb <= ta:
                continue
            for g, wg in zip(gx, gw):
                t = 0.5 * (ta + tb) + 0.5 * (tb - ta) * g
                xi = xi0 + t * (xi1 - xi0)
                for c in range(3):
                    J[c] += 0.5 * (tb - ta) * wg * self._flux_integrand(c, xi, v)
        return J * (qw / self.dV)

    # ---- order 2 current: Esirkepov's density decomposition on the WHOLE grid ----------------
    def esirkepov(self, x0, x1, v, qw):
        nx, ny, nz = self.n
        J = np.zeros((3, nz, ny, nx))
        S0, S1 = [], []
        for d in range(3):
            S0.append(_weights_1d(b2, self.n[d], x0[d] / self.dx[d], 0.0))
            S1.append(_weights_1d(b2, self.n[d], x1[d] / self.dx[d], 0.0))
        DS = [S1[d] - S0[d] for d in range(3)]

        def axis(a, d):  # put a 1-d array on grid axis d (arrays are [z, y, x])
            sh = [1, 1, 1]
            sh[2 - d] = -1
            return a.reshape(sh)

        for c in range(3):
            e, f = (c + 1) % 3, (c + 2) % 3
            br = (axis(S0[e], e) * axis(S0[f], f) + 0.5 * axis(DS[e], e) * axis(S0[f], f)
                  + 0.5 * axis(S0[e], e) * axis(DS[f], f) + axis(DS[e], e) * axis(DS[f], f) / 3.0)
            if self.n[c] == 1:
                J[c] += qw / self.dV * v[c] * (br * axis(np.ones(1), c))
                continue
            W = axis(DS[c], c) * br  # [nz, ny, nx]
            # j_c(i+1/2) - j_c(i-1/2) = -(qw/dV)(dx_c/dt) W[i]; start the running sum half a grid
            # away from the particle, where every W vanishes (needs n_c >= 6)
            n = self.n[c]
            start = (int(np.floor(x0[c] / self.dx[c])) + n // 2 + 1) % n
            order_idx = [(start + a) % n for a in range(n)]
            Wm = np.moveaxis(W, 2 - c, 0)
            Jm = np.moveaxis(J[c], 2 - c, 0)
            run = np.zeros(Wm.shape[1:])
            for i in order_idx:
                run = run - qw / self.dV * (self.dx[c] / self.dt) * Wm[i]
                Jm[i] += run
        return J

    def deposit(self, x0, x1, v, qw):
        return self.vb_exact(x0, x1, v, qw) if self.order == 1 else self.esirkepov(x0, x1, v, qw)

    # ---- FDTD with np.roll (Eq. 12-13, 17-18) -----------------------------------------------
    def _d_fwd(self, a, d):  # (a[i+1] - a[i]) / dx_d
        return (np.roll(a, -1, axis=2 - d) - a) / self.dx[d]

    def _d_bwd(self, a, d):  # (a[i] - a[i-1]) / dx_d
        return (a - np.roll(a, 1, axis=2 - d)) / self.dx[d]

    def push_b(self, E, B, frac):
        h = frac * self.dt
        B[0] -= h * (self._d_fwd(E[2], 1) - self._d_fwd(E[1], 2))
        B[1] -= h * (self._d_fwd(E[0], 2) - self._d_fwd(E[2], 0))
        B[2] -= h * (self._d_fwd(E[1], 0) - self._d_fwd(E[0], 1))

    def push_e(self, E, B, J):
        h = self.dt
        E[0] += h * (self._d_bwd(B[2], 1) - self._d_bwd(B[1], 2) - J[0])
        E[1] += h * (self._d_bwd(B[0], 2) - self._d_bwd(B[2], 0) - J[1])
        E[2] += h * (self._d_bwd(B[1], 0) - self._d_bwd(B[0], 1) - J[2])

    # ---- one step, Fig. 8 ----------------------------------------------------------------------
    def step(self, E, B, xs, us, qws, species):
        """xs, us: float64 [N,3] (updated in place); returns J [3,nz,ny,nx]"""
        self.push_b(E, B, 0.5)
        J = np.zeros_like(E)
        for a in range(xs.shape[0]):
            Ep, Bp = self.gather(E, B, xs[a])
            u = self.boris(us[a], Ep, Bp, species[a])
            vel = u / np.sqrt(1.0 + u @ u)
            x1 = xs[a].copy()
            for d in range(3):
                if self.n[d] != 1:
                    x1[d] = xs[a, d] + self.dt * vel[d]
            J += self.deposit(xs[a], x1, vel, qws[a])
            for d in range(3):
                if self.n[d] != 1:
                    L = self.n[d] * self.dx[d]
                    x1[d] = x1[d] % L
                    if x1[d] >= L:
                        x1[d] = 0.0
            xs[a] = x1
            us[a] = u
        self.push_b(E, B, 0.5)
        self.push_e(E, B, J)
        return J
