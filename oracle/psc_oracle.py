"""ctypes loader for oracle/psc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It holds no arithmetic of the method: it compiles the C oracle with gcc
(plain -O2, OpenMP) and marshals numpy arrays.  Field arrays are float64 [3, nz, ny, nx] without
ghosts; particle columns are float64 [N] (species int32 [N]).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "psc_oracle.c")
_LIB = os.path.join(_HERE, "libpsc_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle (gcc -O2 -fopenmp).  Returns the path of the shared library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


class OrcParams(C.Structure):
    _fields_ = [
        ("n", C.c_int32 * 3),
        ("order", C.c_int32),
        ("n_species", C.c_int32),
        ("block", C.c_int32 * 3),
        ("dx", C.c_double * 3),
        ("dt", C.c_double),
        ("q", C.c_double * 8),
        ("m", C.c_double * 8),
        ("scheme", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_sort.restype = C.c_int
        _lib.orc_sort_cells.restype = C.c_int
    return _lib


def _d(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f(a):
    assert a.dtype == np.float32 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _i(a):
    assert a.dtype == np.int32 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_int32))


class Oracle:
    """One grid + species table.  All methods call straight into the C oracle."""

    def __init__(self, n, dx, dt, order, q, m, block=None, scheme=0):
        self.n = tuple(int(v) for v in n)
        self.dx = tuple(float(v) for v in dx)
        self.dt = float(dt)
        self.order = int(order)
        self.q = [float(v) for v in q]
        self.m = [float(v) for v in m]
        self.block = tuple(int(v) for v in (block if block is not None else (1, 1, 1)))
        p = OrcParams()
        for d in range(3):
            p.n[d] = self.n[d]
            p.dx[d] = self.dx[d]
            p.block[d] = self.block[d]
            assert self.n[d] % self.block[d] == 0
        p.dt = self.dt
        p.order = self.order
        p.n_species = len(self.q)
        p.scheme = int(scheme)
        self.scheme = int(scheme)
        for s in range(len(self.q)):
            p.q[s] = self.q[s]
            p.m[s] = self.m[s]
        self.p = p
        self.fshape = (3, self.n[2], self.n[1], self.n[0])
        self.sshape = (self.n[2], self.n[1], self.n[0])

    # -- helpers ---------------------------------------------------------------------------
    def zeros_field(self):
        return np.zeros(self.fshape, dtype=np.float64)

    @staticmethod
    def num_threads():
        return int(lib().orc_num_threads())

    @staticmethod
    def set_num_threads(n):
        lib().orc_set_num_threads(C.c_int(int(n)))

    # -- grid operators --------------------------------------------------------------------
    def curl_plus(self, F):
        out = self.zeros_field()
        lib().orc_curl_plus(C.byref(self.p), _d(F), _d(out))
        return out

    def curl_minus(self, F):
        out = self.zeros_field()
        lib().orc_curl_minus(C.byref(self.p), _d(F), _d(out))
        return out

    def div_plus(self, F):
        out = np.zeros(self.sshape, dtype=np.float64)
        lib().orc_div_plus(C.byref(self.p), _d(F), _d(out))
        return out

    def div_minus(self, F):
        out = np.zeros(self.sshape, dtype=np.float64)
        lib().orc_div_minus(C.byref(self.p), _d(F), _d(out))
        return out

    def push_b(self, E, B, frac):
        lib().orc_push_b(C.byref(self.p), _d(E), _d(B), C.c_double(frac))

    def push_e(self, E, B, J, frac=1.0):
        lib().orc_push_e(C.byref(self.p), _d(E), _d(B), _d(J), C.c_double(frac))

    # -- particles -------------------------------------------------------------------------
    def gather(self, E, B, x, y, z):
        n = x.shape[0]
        EB = np.zeros((n, 6), dtype=np.float64)
        lib().orc_gather(C.byref(self.p), _d(E), _d(B), C.c_int64(n), _d(x), _d(y), _d(z), _d(EB))
        return EB

    def boris(self, ux, uy, uz, species, EB):
        n = ux.shape[0]
        lib().orc_boris(C.byref(self.p), C.c_int64(n), _d(ux), _d(uy), _d(uz), _i(species), _d(EB))

    def rho(self, x, y, z, qw):
        out = np.zeros(self.sshape, dtype=np.float64)
        lib().orc_rho(C.byref(self.p), C.c_int64(x.shape[0]), _d(x), _d(y), _d(z), _d(qw), _d(out))
        return out

    def deposit(self, J, x0, y0, z0, x1, y1, z1, vx, vy, vz, qw):
        lib().orc_deposit(C.byref(self.p), _d(J), C.c_int64(x0.shape[0]), _d(x0), _d(y0), _d(z0),
                          _d(x1), _d(y1), _d(z1), _d(vx), _d(vy), _d(vz), _d(qw))

    def push_particles(self, E, B, J, x, y, z, ux, uy, uz, qw, species):
        lib().orc_push_particles(C.byref(self.p), _d(E), _d(B), _d(J), C.c_int64(x.shape[0]),
                                 _d(x), _d(y), _d(z), _d(ux), _d(uy), _d(uz), _d(qw), _i(species))

    def step(self, E, B, J, x, y, z, ux, uy, uz, qw, species, nsteps=1):
        lib().orc_step(C.byref(self.p), _d(E), _d(B), _d(J), C.c_int64(x.shape[0]),
                       _d(x), _d(y), _d(z), _d(ux), _d(uy), _d(uz), _d(qw), _i(species),
                       C.c_int(int(nsteps)))

    def energy(self, E, B, ux, uy, uz, qw, species):
        out = np.zeros(3, dtype=np.float64)
        lib().orc_energy(C.byref(self.p), _d(E), _d(B), C.c_int64(ux.shape[0]), _d(ux), _d(uy),
                         _d(uz), _d(qw), _i(species), _d(out))
        return out

    def marder(self, E, rho, D, iters=1):
        """E += D grad+ (div- E - rho), `iters` passes"""
        lib().orc_marder(C.byref(self.p), _d(E), _d(rho), C.c_double(float(D)), C.c_int(int(iters)))

    def sort(self, x32, y32, z32):
        """fp32 positions in -> (cell_idx, key, perm, cell_offsets), all int32."""
        n = x32.shape[0]
        nk = self.n[0] * self.n[1] * self.n[2]
        cell_idx = np.zeros(n, dtype=np.int32)
        key = np.zeros(n, dtype=np.int32)
        perm = np.zeros(n, dtype=np.int32)
        offs = np.zeros(nk + 1, dtype=np.int32)
        rc = lib().orc_sort(C.byref(self.p), C.c_int64(n), _f(x32), _f(y32), _f(z32),
                            _i(cell_idx), _i(key), _i(perm), _i(offs))
        if rc != 0:
            raise ValueError("orc_sort: particle outside the domain")
        return cell_idx, key, perm, offs

    def sort_cells(self, cx, cy, cz):
        """int32 cell coordinates in -> (cell_idx, key, perm, cell_offsets), all int32."""
        n = cx.shape[0]
        nk = self.n[0] * self.n[1] * self.n[2]
        cell_idx = np.zeros(n, dtype=np.int32)
        key = np.zeros(n, dtype=np.int32)
        perm = np.zeros(n, dtype=np.int32)
        offs = np.zeros(nk + 1, dtype=np.int32)
        rc = lib().orc_sort_cells(C.byref(self.p), C.c_int64(n), _i(cx), _i(cy), _i(cz),
                                  _i(cell_idx), _i(key), _i(perm), _i(offs))
        if rc != 0:
            raise ValueError("orc_sort_cells: cell outside the grid")
        return cell_idx, key, perm, offs
