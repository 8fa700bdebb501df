"""Seeded synthetic plasmas shaped like the paper's workloads.

This module serves BOTH the oracle-side tests and the CUDA path (tests, bench.py, smoke) and
therefore holds none of the method's arithmetic: it only draws random numbers and lays out
initial conditions.  Everything is generated in fp32 once ("rounded to fp32 once, then given to
both paths").  Units: c = eps0 = mu0 = 1, dx = 1 cell, e = 1, m_e = 1, d_e = 4 cells, so
omega_pe = 0.25 and n0 = omega_pe^2 = 0.0625; macro-particle weight w = n0 dV / ppc(n0).

The five configs are BASELINE.json's; the paper's own production decks (bubble reconnection,
Harris-sheet acceleration) are not available and these stand in for them.
Particles are created cell by cell (initial array cell-ordered in natural k,j,i order,
PAPER.md:577), positions uniform inside the cell, ions co-located with electrons so that
rho = 0 and E = 0 satisfies Gauss's law at t = 0 (A21).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import torch

N0 = 0.0625
SEED0 = 13107866


@dataclass
class Plasma:
    name: str
    n: tuple          # cells (nx, ny, nz); 1 = invariant
    dx: tuple
    dt: float
    order: int
    q: list
    m: list
    steps: int        # BASELINE.json's step count for this config
    x: torch.Tensor = None
    y: torch.Tensor = None
    z: torch.Tensor = None
    ux: torch.Tensor = None
    uy: torch.Tensor = None
    uz: torch.Tensor = None
    qw: torch.Tensor = None
    species: torch.Tensor = None
    id: torch.Tensor = None
    E: torch.Tensor = None   # [3, nz, ny, nx] interior values, Yee-staggered
    B: torch.Tensor = None
    extra: dict = field(default_factory=dict)

    @property
    def n_particles(self):
        return int(self.x.shape[0])

    def columns(self):
        return (self.x, self.y, self.z, self.ux, self.uy, self.uz, self.qw, self.species, self.id)

    def shuffled(self, seed=None):
        """a seeded random permutation of the particle list (so that a sort does real work)"""
        g = torch.Generator(device=self.x.device).manual_seed(SEED0 + 999 if seed is None else seed)
        p = torch.randperm(self.n_particles, generator=g, device=self.x.device)
        out = Plasma(self.name + "-shuffled", self.n, self.dx, self.dt, self.order, self.q, self.m,
                     self.steps, E=self.E.clone(), B=self.B.clone(), extra=dict(self.extra))
        for k in ("x", "y", "z", "ux", "uy", "uz", "qw", "species", "id"):
            setattr(out, k, getattr(self, k)[p].contiguous())
        return out


def cfl_dt(n, dx, frac=0.5):
    """'dt = 0.5 CFL' (A16): frac / sqrt(sum over non-invariant d of 1/dx_d^2)"""
    s = sum(1.0 / (dx[d] * dx[d]) for d in range(3) if n[d] > 1)
    return frac / math.sqrt(s)


def _cell_origin(n, device):
    """origins (x,y,z) of all cells in natural k,j,i order, int64 [ncells] each"""
    nx, ny, nz = n
    idx = torch.arange(nx * ny * nz, device=device)
    return idx % nx, (idx // nx) % ny, idx // (nx * ny)


def _place(n, dx, counts, gen, device):
    """uniform positions inside cells; counts: int64 [ncells] particles per cell -> x,y,z fp32"""
    ci, cj, ck = _cell_origin(n, device)
    ci = torch.repeat_interleave(ci, counts)
    cj = torch.repeat_interleave(cj, counts)
    ck = torch.repeat_interleave(ck, counts)
    out = []
    for d, c in enumerate((ci, cj, ck)):
        if n[d] == 1:
            out.append(torch.full(c.shape, 0.5 * dx[d], dtype=torch.float32, device=device))
            continue
        r = torch.rand(c.shape, generator=gen, device=device, dtype=torch.float32)
        p = (c.to(torch.float32) + r) * dx[d]
        # fp32 rounding may land exactly on the upper face of the cell / domain: pull it back
        hi = (c + 1).to(torch.float32) * dx[d]
        p = torch.where(p >= hi, torch.nextafter(hi, torch.zeros_like(hi)), p)
        out.append(p)
    return out[0], out[1], out[2], (ci, cj, ck)


def _maxwellian(nump, vth, drift, gen, device):
    u = torch.randn(nump, generator=gen, device=device, dtype=torch.float32) * vth
    return u + drift if isinstance(drift, torch.Tensor) or drift != 0.0 else u


def _pair(pl: Plasma, pos, u_e, u_i, w, s_e, s_i, parts):
    """append electrons (species s_e) and co-located ions (species s_i) with weights w"""
    x, y, z = pos
    nump = x.shape[0]
    dev = x.device
    for (u, s, sign) in ((u_e, s_e, -1.0), (u_i, s_i, +1.0)):
        parts.append(dict(x=x, y=y, z=z, ux=u[0], uy=u[1], uz=u[2],
                          qw=(sign * w).to(torch.float32) if isinstance(w, torch.Tensor)
                          else torch.full((nump,), sign * w, dtype=torch.float32, device=dev),
                          species=s if isinstance(s, torch.Tensor)
                          else torch.full((nump,), s, dtype=torch.int32, device=dev)))


def _finish(pl: Plasma, parts, per_cell_counts):
    """interleave the populations cell by cell: per cell, population 0's particles, then 1's, ...
    parts[k] covers counts per_cell_counts[k] (int64 [ncells]) in natural cell order."""
    dev = parts[0]["x"].device
    ncell = per_cell_counts[0].shape[0]
    tot = torch.zeros(ncell, dtype=torch.int64, device=dev)
    starts = []
    for c in per_cell_counts:
        starts.append(tot.clone())
        tot = tot + c
    cell_base = torch.cumsum(tot, 0) - tot
    ntot = int(tot.sum())
    dest = []
    for c, st in zip(per_cell_counts, starts):
        first = torch.repeat_interleave(cell_base + st, c)         # slot of the cell's first one
        pbase = torch.cumsum(c, 0) - c
        rank = torch.arange(int(c.sum()), device=dev) - torch.repeat_interleave(pbase, c)
        dest.append(first + rank)
    for k in ("x", "y", "z", "ux", "uy", "uz", "qw", "species"):
        buf = torch.empty(ntot, dtype=parts[0][k].dtype, device=dev)
        for prt, d in zip(parts, dest):
            buf[d] = prt[k]
        setattr(pl, k, buf)
    pl.id = torch.arange(ntot, dtype=torch.int32, device=dev)
    nx, ny, nz = pl.n
    if pl.E is None:
        pl.E = torch.zeros((3, nz, ny, nx), dtype=torch.float32, device=dev)
    if pl.B is None:
        pl.B = torch.zeros((3, nz, ny, nx), dtype=torch.float32, device=dev)
    return pl


def thermal(n, ppc, *, mass_ratio=100.0, vth_e=0.1, vth_i=0.01, order=1, steps=10, seed=SEED0,
            device="cpu", name="thermal", dx=(1.0, 1.0, 1.0)):
    """periodic two-species thermal plasma (configs 1, 2, 4): ppc electrons + ppc ions per cell"""
    dev = torch.device(device)
    gen = torch.Generator(device=dev).manual_seed(seed)
    pl = Plasma(name, tuple(n), tuple(dx), cfl_dt(n, dx), order, [-1.0, 1.0], [1.0, mass_ratio], steps)
    ncell = n[0] * n[1] * n[2]
    counts = torch.full((ncell,), ppc, dtype=torch.int64, device=dev)
    x, y, z, _ = _place(n, dx, counts, gen, dev)
    nump = x.shape[0]
    w = N0 * dx[0] * dx[1] * dx[2] / ppc
    u_e = [_maxwellian(nump, vth_e, 0.0, gen, dev) for _ in range(3)]
    u_i = [_maxwellian(nump, vth_i, 0.0, gen, dev) for _ in range(3)]
    parts = []
    _pair(pl, (x, y, z), u_e, u_i, w, 0, 1, parts)
    return _finish(pl, parts, [counts, counts])


def harris(n=(1, 512, 1024), *, ppc0=100, steps=200, seed=SEED0 + 3, device="cpu"):
    """config 3: double Harris sheet in the yz plane (DESIGN.md input recipe #3).
    Scales with n: sheets at z = nz/4 and 3nz/4, half-width L = 10 * nz/1024 cells."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev).manual_seed(seed)
    dx = (1.0, 1.0, 1.0)
    mi = 25.0
    pl = Plasma("harris", tuple(n), dx, cfl_dt(n, dx), 1, [-1.0, 1.0], [1.0, mi], steps)
    nx, ny, nz = n
    L = 10.0 * nz / 1024.0
    z1, z2 = 0.25 * nz, 0.75 * nz
    B0 = 0.0625
    Ttot = B0 * B0 / (2.0 * N0)
    Te, Ti = Ttot / 6.0, Ttot * 5.0 / 6.0
    vth_e, vth_i = math.sqrt(Te), math.sqrt(Ti / mi)
    drift = 2.0 * Ttot / (B0 * L)                      # |u_i - u_e| in the sheets
    ui_mag, ue_mag = drift * 5.0 / 6.0, drift / 6.0    # u_i/T_i = -u_e/T_e
    # per-cell counts: background 0.1 n0 (non-drifting) + sheet sech^2 (drifting), from cell centres
    ci, cj, ck = _cell_origin(n, dev)
    zc = ck.to(torch.float64) + 0.5
    s1 = 1.0 / torch.cosh((zc - z1) / L) ** 2
    s2 = 1.0 / torch.cosh((zc - z2) / L) ** 2
    c_bg = torch.full_like(ck, int(round(0.1 * ppc0)))
    c_s1 = torch.round(ppc0 * s1).to(torch.int64)
    c_s2 = torch.round(ppc0 * s2).to(torch.int64)
    w = N0 / ppc0
    parts, counts = [], []
    for cnt, sgn in ((c_bg, 0.0), (c_s1, -1.0), (c_s2, +1.0)):   # sheet 1: u_i - u_e < 0
        x, y, z, _ = _place(n, dx, cnt, gen, dev)
        nump = x.shape[0]
        u_e = [_maxwellian(nump, vth_e, -sgn * ue_mag if c == 0 else 0.0, gen, dev) for c in range(3)]
        u_i = [_maxwellian(nump, vth_i, sgn * ui_mag if c == 0 else 0.0, gen, dev) for c in range(3)]
        _pair(pl, (x, y, z), u_e, u_i, w, 0, 1, parts)
        counts += [cnt, cnt]
    # B_y at its Yee points (i+1/2, j, k+1/2): depends on z = k + 1/2 only
    zy = torch.arange(nz, device=dev, dtype=torch.float64) + 0.5
    by = B0 * (torch.tanh((zy - z1) / L) - torch.tanh((zy - z2) / L) - 1.0)
    pl.B = torch.zeros((3, nz, ny, nx), dtype=torch.float32, device=dev)
    pl.B[1] = by.to(torch.float32)[:, None, None]
    pl.extra.update(L=L, B0=B0)
    return _finish(pl, parts, counts)


def beam(n=(64, 64, 256), *, ppc_bg=32, ppc_beam=8, steps=100, seed=SEED0 + 5, device="cpu",
         order=2):
    """config 5: relativistic (gamma = 5) electron beam along x at 10 % density through a
    return-current background; three species (0 background e, 1 beam e, 2 ions m = 100)."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev).manual_seed(seed)
    dx = (1.0, 1.0, 1.0)
    pl = Plasma("beam", tuple(n), dx, cfl_dt(n, dx), order, [-1.0, -1.0, 1.0], [1.0, 1.0, 100.0], steps)
    ncell = n[0] * n[1] * n[2]
    gam = 5.0
    u_beam = math.sqrt(gam * gam - 1.0)
    beta_b = u_beam / gam
    v_bg = -0.1 * beta_b
    u_bg = v_bg / math.sqrt(1.0 - v_bg * v_bg)
    parts, counts = [], []
    for ppc, dens, drift, s_e in ((ppc_bg, 1.0, u_bg, 0), (ppc_beam, 0.1, u_beam, 1)):
        cnt = torch.full((ncell,), ppc, dtype=torch.int64, device=dev)
        x, y, z, _ = _place(n, dx, cnt, gen, dev)
        nump = x.shape[0]
        u_e = [_maxwellian(nump, 0.05, drift if c == 0 else 0.0, gen, dev) for c in range(3)]
        u_i = [_maxwellian(nump, 0.005, 0.0, gen, dev) for _ in range(3)]
        _pair(pl, (x, y, z), u_e, u_i, dens * N0 / ppc, s_e, 2, parts)
        counts += [cnt, cnt]
    return _finish(pl, parts, counts)


def make_config(k: int, *, device="cpu", scale=None):
    """BASELINE.json configs 1..5.  `scale` (optional) replaces the grid by a smaller one of the
    same dimensionality and keeps particles per cell (parity tests at sizes the oracle finishes
    in seconds); scale=None gives the full size."""
    if k == 1:
        return thermal(scale or (1, 64, 64), 16, steps=10, seed=SEED0 + 1, device=device, name="config1")
    if k == 2:
        return thermal(scale or (1, 1024, 1024), 100, steps=100, seed=SEED0 + 2, device=device, name="config2")
    if k == 3:
        pl = harris(scale or (1, 512, 1024), device=device)
        pl.name = "config3"
        return pl
    if k == 4:
        return thermal(scale or (128, 128, 128), 50, steps=50, seed=SEED0 + 4, device=device, name="config4")
    if k == 5:
        pl = beam(scale or (64, 64, 256), device=device)
        pl.name = "config5"
        return pl
    raise ValueError(k)
