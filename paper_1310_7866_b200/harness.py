"""Device-buffer plumbing around the binding: allocates the PyTorch tensors the library borrows
(two particle column sets, ghosted E/B/J, workspace) from a seeded synthetic plasma
(psc_inputs.Plasma) and maps the library's raw pointers back to tensors.  Layout only -- no
arithmetic of the method lives here."""
from __future__ import annotations

import weakref

import torch

from . import COLUMNS, PSC_B, PSC_E, PSC_GHOST, Psc


class Simulation:
    GUARD = 64               # sentinel entries behind the n entries of every dense column
    SENTINEL = 0x7FC0DEAD    # (a NaN pattern as fp32)
    live = weakref.WeakSet()  # the simulations alive in this process (tests check their guards)

    def __init__(self, plasma, block=(0, 0, 0), device="cuda:0", with_id=True, with_x=True, scheme=0):
        self.device = torch.device(device)
        self.plasma = plasma
        self.psc = Psc(plasma.n, plasma.dx, plasma.dt, plasma.order, plasma.q, plasma.m, block, scheme)
        self.n = tuple(plasma.n)
        self.g = tuple(PSC_GHOST if v > 1 else 0 for v in self.n)
        self.np = plasma.n_particles
        dev = self.device
        shp = self.psc.field_shape
        self.E = torch.zeros(shp, dtype=torch.float32, device=dev)
        self.B = torch.zeros(shp, dtype=torch.float32, device=dev)
        self.J = torch.zeros(shp, dtype=torch.float32, device=dev)
        self.interior(self.E).copy_(plasma.E.to(dev))
        self.interior(self.B).copy_(plasma.B.to(dev))
        self.capacity = self.psc.particle_capacity(self.np)
        self.sets = []
        for k in range(2):
            s = {}
            for c in COLUMNS:
                if (c == "id" and not with_id) or (c == "x" and not with_x):
                    s[c] = None       # optional columns (include/psc.h): not carried
                    continue
                dt = torch.int32 if c in ("species", "id") else torch.float32
                # set 0 is the dense set (n entries, include/psc.h) followed by GUARD sentinel
                # entries the library must never write; set 1 is the store set (capacity entries)
                if k == 0:
                    s[c] = torch.empty(self.np + self.GUARD, dtype=dt, device=dev)
                    s[c][self.np:].view(torch.int32).fill_(self.SENTINEL)
                else:
                    s[c] = torch.empty(self.capacity, dtype=dt, device=dev)
            self.sets.append(s)
        for c in COLUMNS:
            if self.sets[0][c] is not None and self.np:
                self.sets[0][c][: self.np].copy_(getattr(plasma, c).to(dev))
        self.ws = torch.empty(self.psc.workspace_bytes(self.np), dtype=torch.uint8, device=dev)
        self.psc.bind_workspace(self.ws)
        self.psc.bind_fields(self.E, self.B, self.J)
        self.psc.bind_particles(self.np, self.capacity, self.sets[0], self.sets[1])
        self.psc.fill_ghosts(PSC_E)
        self.psc.fill_ghosts(PSC_B)
        Simulation.live.add(self)

    def interior(self, F):
        g, n = self.g, self.n
        return F[:, g[2]:g[2] + n[2], g[1]:g[1] + n[1], g[0]:g[0] + n[0]]

    def guards_intact(self):
        """True while no entry behind the n entries of a dense-set column has been written"""
        for t in self.sets[0].values():
            if t is not None and not bool((t[self.np:].view(torch.int32) == self.SENTINEL).all()):
                return False
        return True

    def memory(self):
        """device bytes the library works in: particle columns of both sets (guards excluded),
        workspace, fields; `multiplier` = column bytes / (n * bytes of one dense particle)"""
        ncol = sum(1 for t in self.sets[0].values() if t is not None)
        cols = 4 * ncol * (self.np + self.capacity)
        return {"columns": cols, "workspace": self.ws.numel(), "fields": 3 * 4 * self.E.numel(),
                "bytes_per_particle": (cols + self.ws.numel()) / max(self.np, 1),
                "multiplier": cols / max(4 * ncol * self.np, 1)}

    def current(self):
        """the column set (dict of tensors, trimmed to n particles) that holds the particles now;
        only meaningful for absolute columns (after bind or psc_particles_export)"""
        assert self.psc.particles_form() == 0
        ptr = self.psc.particles_current()["y"]
        s = self.sets[0] if self.sets[0]["y"].data_ptr() == ptr else self.sets[1]
        assert s["y"].data_ptr() == ptr
        return {c: (None if t is None else t[: self.np]) for c, t in s.items()}

    def gather(self, absolute=False):
        """dense copy of the cell store (psc_particles_gather): dict of column tensors [n] plus
        "key" (int32 cell keys; the cell the in-cell offsets refer to).  State unchanged."""
        dev = self.device
        out = {}
        for c in COLUMNS:
            if self.sets[0][c] is None:
                out[c] = None
                continue
            dt = torch.int32 if c in ("species", "id") else torch.float32
            out[c] = torch.empty(max(self.np, 1), dtype=dt, device=dev)
        key = torch.empty(max(self.np, 1), dtype=torch.int32, device=dev)
        self.psc.particles_gather(out, key, absolute)
        out = {c: (None if t is None else t[: self.np]) for c, t in out.items()}
        out["key"] = key[: self.np]
        return out

    def _ws_view(self, ptr, count):
        off = ptr - self.ws.data_ptr()
        return self.ws[off: off + 4 * count].view(torch.int32)

    def sort_result(self):
        """(cell_idx[n], perm[n], cell_offsets[n_keys+1]) as int32 tensors viewing the workspace"""
        ci, pm, co, nk = self.psc.sort_result()
        return self._ws_view(ci, self.np), self._ws_view(pm, self.np), self._ws_view(co, nk + 1)

    def step(self, nsteps=1):
        for _ in range(nsteps):
            self.psc.step()
