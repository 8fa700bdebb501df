"""paper_1310_7866_b200 -- thin Python binding of the C-ABI CUDA library (include/psc.h).

Argument marshalling only: every step of the PIC hot path (sort, gather, Boris push, deposit,
ghost exchange, FDTD) runs in the hand-written sm_100a kernels of csrc/.  PyTorch supplies device
memory and streams.  There is no CPU fallback: if the library cannot be built or loaded, or no
CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

PSC_OK = 0
PSC_E, PSC_B, PSC_J = 0, 1, 2
PSC_F_OOB, PSC_F_NAN, PSC_F_SPECIES, PSC_F_OVERFLOW = 1, 4, 8, 32
PSC_GHOST = 2
PSC_ERR_SCRATCH_LIMIT = -9
MARDER_STATIC_MAX_POINTS = 327680
PSC_SCHEME_STANDARD, PSC_SCHEME_ALTERNATING = 0, 1
PHASES = {"sort": 0, "push": 1, "j_zero": 2, "field_b": 3, "j_exchange": 4, "field_e": 5,
          "sort_count": 6, "sort_scan": 7, "sort_rank": 8, "sort_reorder": 9, "marder": 10}
PSC_PH_COUNT = 16

EXPORTS = [
    "psc_create", "psc_destroy", "psc_workspace_bytes", "psc_bind_workspace", "psc_bind_fields",
    "psc_field_elems", "psc_particle_capacity", "psc_bind_particles", "psc_particles_sort",
    "psc_push_particles", "psc_push_fields", "psc_exchange_j", "psc_fill_ghosts", "psc_step",
    "psc_charge_density", "psc_marder", "psc_marder_static", "psc_patch_loads", "psc_hilbert_order", "psc_balance", "psc_balance_owners",
    "psc_step_host", "psc_sort_result", "psc_particles_current", "psc_particles_form",
    "psc_particles_gather", "psc_particles_export", "psc_store_info", "psc_status", "psc_launch_count",
    "psc_last_cuda_error", "psc_set_option", "psc_profile", "psc_strerror", "psc_version",
]

COLUMNS = ("x", "y", "z", "ux", "uy", "uz", "qw", "species", "id")


class PscParams(C.Structure):
    _fields_ = [
        ("n", C.c_int32 * 3),
        ("ghost", C.c_int32),
        ("dx", C.c_float * 3),
        ("dt", C.c_float),
        ("order", C.c_int32),
        ("n_species", C.c_int32),
        ("q", C.POINTER(C.c_float)),
        ("m", C.POINTER(C.c_float)),
        ("block", C.c_int32 * 3),
        ("scheme", C.c_int32),
    ]


class PscCols(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in COLUMNS]


class PscError(RuntimeError):
    def __init__(self, code, what, cuda=0):
        self.code = code
        msg = "%s failed: %s (%d)" % (what, lib().psc_strerror(code).decode(), code)
        if cuda:
            msg += " [cudaError %d]" % cuda
        super().__init__(msg)


_lib = None


def lib():
    """Loads (building first if needed) libpsc_b200.so.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.psc_create.argtypes = [C.POINTER(PscParams), C.POINTER(C.c_void_p)]
        L.psc_destroy.argtypes = [C.c_void_p]
        L.psc_destroy.restype = None
        L.psc_workspace_bytes.argtypes = [C.c_void_p, C.c_int64]
        L.psc_workspace_bytes.restype = C.c_size_t
        L.psc_bind_workspace.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        L.psc_bind_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.psc_field_elems.argtypes = [C.c_void_p, C.POINTER(C.c_int32 * 3)]
        L.psc_field_elems.restype = C.c_int64
        L.psc_particle_capacity.argtypes = [C.c_void_p, C.c_int64]
        L.psc_particle_capacity.restype = C.c_int64
        L.psc_bind_particles.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.POINTER(PscCols), C.POINTER(PscCols)]
        for f in ("psc_particles_sort", "psc_push_particles", "psc_exchange_j", "psc_step"):
            getattr(L, f).argtypes = [C.c_void_p, C.c_void_p]
        L.psc_push_fields.argtypes = [C.c_void_p, C.c_int, C.c_float, C.c_void_p]
        L.psc_fill_ghosts.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.psc_charge_density.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.psc_marder.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_int]
        L.psc_marder_static.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_int]
        L.psc_patch_loads.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_int32), C.c_void_p,
                                      C.POINTER(C.c_int32)]
        L.psc_hilbert_order.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.psc_balance.argtypes = [C.c_int64, C.POINTER(C.c_double), C.c_int32, C.POINTER(C.c_double),
                                  C.POINTER(C.c_int32)]
        L.psc_balance_owners.argtypes = [C.c_int64, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.psc_step_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(PscCols),
                                    C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.psc_sort_result.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p),
                                      C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                      C.POINTER(C.c_int64)]
        L.psc_particles_form.argtypes = [C.c_void_p]
        L.psc_particles_gather.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(PscCols), C.c_void_p, C.c_int]
        L.psc_store_info.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
        L.psc_particles_export.argtypes = [C.c_void_p, C.c_void_p]
        L.psc_particles_current.argtypes = [C.c_void_p, C.POINTER(PscCols)]
        L.psc_status.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_uint32)]
        L.psc_launch_count.argtypes = [C.c_void_p]
        L.psc_launch_count.restype = C.c_int64
        L.psc_last_cuda_error.argtypes = [C.c_void_p]
        L.psc_profile.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.psc_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int64]
        L.psc_strerror.argtypes = [C.c_int]
        L.psc_strerror.restype = C.c_char_p
        L.psc_version.restype = C.c_char_p
        _lib = L
    return _lib


def _stream(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    return C.c_void_p(int(stream))


def _cols(tensors) -> PscCols:
    """dict / sequence of per-column tensors (or None for id) -> PscCols of raw pointers"""
    c = PscCols()
    if not isinstance(tensors, dict):
        tensors = dict(zip(COLUMNS, tensors))
    for k in COLUMNS:
        t = tensors.get(k)
        setattr(c, k, None if t is None else t.data_ptr())
    return c


class Psc:
    """One psc_ctx.  Method names are the C names without the psc_ prefix."""

    def __init__(self, n, dx, dt, order, q, m, block=(0, 0, 0), scheme=0):
        self._h = None
        L = lib()
        p = PscParams()
        for d in range(3):
            p.n[d] = int(n[d])
            p.dx[d] = float(dx[d])
            p.block[d] = int(block[d])
        p.ghost = PSC_GHOST
        p.dt = float(dt)
        p.order = int(order)
        p.scheme = int(scheme)
        p.n_species = len(q)
        self._q = (C.c_float * len(q))(*[float(v) for v in q])
        self._m = (C.c_float * len(m))(*[float(v) for v in m])
        p.q = C.cast(self._q, C.POINTER(C.c_float))
        p.m = C.cast(self._m, C.POINTER(C.c_float))
        h = C.c_void_p()
        rc = L.psc_create(C.byref(p), C.byref(h))
        if rc:
            raise PscError(rc, "psc_create")
        self._h = h
        self._keep = {}
        self.n = tuple(int(v) for v in n)
        ext = (C.c_int32 * 3)()
        self.field_elems = int(L.psc_field_elems(h, C.byref(ext)))
        self.ext = tuple(int(v) for v in ext)
        self.field_shape = (3, self.ext[2], self.ext[1], self.ext[0])

    def _check(self, rc, what):
        if rc:
            raise PscError(rc, what, lib().psc_last_cuda_error(self._h))

    def close(self):
        if self._h is not None:
            lib().psc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- binding -------------------------------------------------------------------------------
    def workspace_bytes(self, max_particles):
        return int(lib().psc_workspace_bytes(self._h, int(max_particles)))

    def bind_workspace(self, ws):
        self._keep["ws"] = ws
        self._check(lib().psc_bind_workspace(self._h, ws.data_ptr(), ws.numel() * ws.element_size()),
                    "psc_bind_workspace")

    def bind_fields(self, E, B, J):
        self._keep["fields"] = (E, B, J)
        self._check(lib().psc_bind_fields(self._h, E.data_ptr(), B.data_ptr(), J.data_ptr()),
                    "psc_bind_fields")

    def particle_capacity(self, n):
        """entries every particle column needs for n particles (the cell store's spare room)"""
        return int(lib().psc_particle_capacity(self._h, int(n)))

    def bind_particles(self, n, capacity, primary, secondary):
        self._keep["particles"] = (primary, secondary)
        a, b = _cols(primary), _cols(secondary)
        self._check(lib().psc_bind_particles(self._h, int(n), int(capacity), C.byref(a), C.byref(b)),
                    "psc_bind_particles")

    # -- the hot path ----------------------------------------------------------------------------
    def particles_sort(self, stream=None):
        """psc_particles_sort: stable cell-key counting sort (include/psc.h)"""
        self._check(lib().psc_particles_sort(self._h, _stream(stream)), "psc_particles_sort")

    def push_particles(self, stream=None):
        """psc_push_particles: fused gather (Eq. 11) - Boris (Eq. 27-28) - move (Eq. 26) -
        charge-conserving deposit, the particle loop of Fig. 8"""
        self._check(lib().psc_push_particles(self._h, _stream(stream)), "psc_push_particles")

    def push_fields(self, which, frac, stream=None):
        """psc_push_fields: Yee FDTD update of E or B over frac*dt (Eq. 17-18)"""
        self._check(lib().psc_push_fields(self._h, int(which), float(frac), _stream(stream)),
                    "psc_push_fields")

    def exchange_j(self, stream=None):
        """psc_exchange_j: add_and_fill_ghosts_j of Fig. 8 on one GPU"""
        self._check(lib().psc_exchange_j(self._h, _stream(stream)), "psc_exchange_j")

    def fill_ghosts(self, which, stream=None):
        """psc_fill_ghosts: ghosts := periodic images"""
        self._check(lib().psc_fill_ghosts(self._h, int(which), _stream(stream)), "psc_fill_ghosts")

    def charge_density(self, rho, stream=None):
        """psc_charge_density: node charge density with the bound order's weights"""
        self._check(lib().psc_charge_density(self._h, _stream(stream), rho.data_ptr()), "psc_charge_density")

    def marder(self, diffusion, iters=1, stream=None):
        """psc_marder: E += diffusion * grad+ (div- E - rho), `iters` passes"""
        self._check(lib().psc_marder(self._h, _stream(stream), float(diffusion), int(iters)), "psc_marder")

    def marder_static(self, diffusion, iters=1, stream=None):
        """psc_marder_static: psc_marder with its scratch in a fixed device array of the library, for
        callers that cannot allocate device memory when they apply the correction (include/psc.h:
        grids up to MARDER_STATIC_MAX_POINTS points incl. ghosts; overlapping calls race)"""
        self._check(lib().psc_marder_static(self._h, _stream(stream), float(diffusion), int(iters)),
                    "psc_marder_static")

    def patch_loads(self, patch_blocks, loads, stream=None):
        """psc_patch_loads: particles + cells of every patch into the device int64
        tensor `loads`; returns the patch grid (npx, npy, npz)"""
        pb = (C.c_int32 * 3)(*[int(v) for v in patch_blocks])
        npo = (C.c_int32 * 3)()
        self._check(lib().psc_patch_loads(self._h, _stream(stream), pb, loads.data_ptr(), npo), "psc_patch_loads")
        return tuple(npo)

    def step(self, stream=None):
        """psc_step: one time step in the order of Fig. 8"""
        self._check(lib().psc_step(self._h, _stream(stream)), "psc_step")

    def step_host(self, n, host_cols, hE, hB, hJ=None, nsteps=1, stream=None):
        """psc_step_host: the same with HOST buffers (copies in, nsteps psc_step, copies out)"""
        h = _cols(host_cols)
        self._check(lib().psc_step_host(self._h, _stream(stream), int(n), C.byref(h), hE.data_ptr(),
                                        hB.data_ptr(), None if hJ is None else hJ.data_ptr(),
                                        int(nsteps)), "psc_step_host")

    # -- inspection ------------------------------------------------------------------------------
    def sort_result(self, stream=None):
        """raw device pointers (cell_idx, perm, cell_offsets) and n_keys"""
        ci, pm, co = C.c_void_p(), C.c_void_p(), C.c_void_p()
        nk = C.c_int64()
        self._check(lib().psc_sort_result(self._h, _stream(stream), C.byref(ci), C.byref(pm),
                                          C.byref(co), C.byref(nk)), "psc_sort_result")
        return ci.value, pm.value, co.value, int(nk.value)

    def particles_form(self):
        return int(lib().psc_particles_form(self._h))

    def particles_gather(self, dst, key=None, absolute=False, stream=None):
        """psc_particles_gather: dense copy of the cell store into the caller's columns `dst`
        (+ cell keys), state unchanged"""
        d = _cols(dst)
        self._check(lib().psc_particles_gather(self._h, _stream(stream), C.byref(d),
                                               None if key is None else key.data_ptr(),
                                               1 if absolute else 0), "psc_particles_gather")

    def store_info(self, stream=None):
        """{max_count, slots, relayouts, spilled, image_slots, tma_tiles} of the cell store (synchronises)"""
        a = (C.c_int64 * 8)()
        self._check(lib().psc_store_info(self._h, _stream(stream), a), "psc_store_info")
        return {"max_count": int(a[0]), "slots": int(a[1]), "relayouts": int(a[2]),
                "spilled": int(a[3]), "image_slots": int(a[4]), "tma_tiles": int(a[5]), "inserted": int(a[6])}

    def particles_export(self, stream=None):
        self._check(lib().psc_particles_export(self._h, _stream(stream)), "psc_particles_export")

    def particles_current(self):
        """raw device pointers of the column set that currently holds the particles"""
        c = PscCols()
        self._check(lib().psc_particles_current(self._h, C.byref(c)), "psc_particles_current")
        return {k: getattr(c, k) for k in COLUMNS}

    def status(self, stream=None):
        f = C.c_uint32()
        self._check(lib().psc_status(self._h, _stream(stream), C.byref(f)), "psc_status")
        return int(f.value)

    def profile(self, stream=None):
        """{phase: (total ms, brackets)} since the last call (needs set_option("profile", 1))"""
        ms = (C.c_double * PSC_PH_COUNT)()
        cnt = (C.c_int64 * PSC_PH_COUNT)()
        self._check(lib().psc_profile(self._h, _stream(stream), ms, cnt), "psc_profile")
        return {k: (float(ms[i]), int(cnt[i])) for k, i in PHASES.items()}

    def launch_count(self):
        return int(lib().psc_launch_count(self._h))

    def set_option(self, name, value):
        self._check(lib().psc_set_option(self._h, name.encode(), int(value)), "psc_set_option")


def version():
    return lib().psc_version().decode()


def hilbert_order(np3):
    """psc_hilbert_order: row-major patch indices in Hilbert-Peano curve order"""
    n = int(np3[0]) * int(np3[1]) * int(np3[2])
    a = (C.c_int32 * 3)(*[int(v) for v in np3])
    out = (C.c_int32 * n)()
    rc = lib().psc_hilbert_order(a, out)
    if rc:
        raise PscError(rc, "psc_hilbert_order")
    return list(out)


def balance(loads, capability):
    """psc_balance: Appendix A: patches per rank along the curve"""
    n, r = len(loads), len(capability)
    L = (C.c_double * n)(*[float(v) for v in loads])
    Cp = (C.c_double * r)(*[float(v) for v in capability])
    out = (C.c_int32 * r)()
    rc = lib().psc_balance(n, L, r, Cp, out)
    if rc:
        raise PscError(rc, "psc_balance")
    return list(out)


def balance_owners(count):
    """psc_balance_owners: rank of every patch along the curve for the counts psc_balance returned"""
    r, n = len(count), int(sum(count))
    cnt = (C.c_int32 * r)(*[int(v) for v in count])
    out = (C.c_int32 * max(n, 1))()
    rc = lib().psc_balance_owners(n, r, cnt, out)
    if rc:
        raise PscError(rc, "psc_balance_owners")
    return list(out)[:n]
