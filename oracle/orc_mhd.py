"""ctypes view of liborc_mhd.so (oracle/orc_mhd.cpp) -- TEST INFRASTRUCTURE ONLY, see oracle/orc_mhd.h."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liborc_mhd.so")
_SRC = [os.path.join(_HERE, f) for f in ("orc_mhd.cpp", "orc.cpp", "orc_mhd.h", "orc.h")]
_lib = None


def build(force: bool = False) -> str:
    if (not force and os.path.exists(_SO)
            and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC)):
        return _SO
    subprocess.run(["g++", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-Wall",
                    "-o", _SO, _SRC[0], _SRC[1]], check=True, cwd=_HERE)
    return _SO


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
    L.orcm_pack_create.restype = C.c_void_p
    L.orcm_pack_create.argtypes = [C.c_int] * 5 + [C.c_double] + [C.c_int] * 3 + [ip, dp, dp]
    L.orcm_pack_bind.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.orcm_set_threads.argtypes = [C.c_void_p, C.c_int]
    L.orcm_pack_set_recon.argtypes = [C.c_void_p, C.c_int]
    L.orcm_pack_set_integrator.argtypes = [C.c_void_p, C.c_int]
    L.orcm_fill_ghosts.argtypes = [C.c_void_p]
    L.orcm_stage.argtypes = [C.c_void_p, C.c_int, C.c_double]
    L.orcm_new_dt.argtypes = [C.c_void_p, C.c_double, dp]
    L.orcm_pack_current.restype = C.c_void_p
    L.orcm_pack_current.argtypes = [C.c_void_p]
    L.orcm_pack_floor_count.restype = C.c_longlong
    L.orcm_pack_floor_count.argtypes = [C.c_void_p]
    L.orcm_pack_destroy.argtypes = [C.c_void_p]
    L.orcm_last_error.restype = C.c_char_p
    for f in (L.orcm_hlld, L.orcm_llf, L.orcm_hlle):
        f.argtypes = [C.c_double, C.c_double, dp, dp, dp]
        f.restype = None
    L.orcm_pack_set_rsolver.argtypes = [C.c_void_p, C.c_int]
    _lib = L
    return L


class OrcError(RuntimeError):
    pass


def _chk(rc):
    if rc != 0:
        raise OrcError(lib().orcm_last_error().decode())


def hlld(gamma, bn, WL, WR, solver="hlld"):
    F = (C.c_double * 7)()
    a = (C.c_double * 7)(*[float(v) for v in WL])
    b = (C.c_double * 7)(*[float(v) for v in WR])
    getattr(lib(), "orcm_" + solver)(gamma, bn, a, b, F)
    return np.array(F[:])


class OrcMhdPack:
    """Oracle MHD pack over a uniform Mesh (paper_2409_16053_b200.inputs.Mesh); owns two numpy state buffers of 8 variables."""

    def __init__(self, mesh, gamma, threads=1, recon=0, nstages=2, rsolver=0):
        L = lib()
        self.mesh = mesh
        self.nstages = nstages
        lx = [v for (_, l1, l2, l3) in mesh.blocks for v in (l1, l2, l3)]
        self._h = L.orcm_pack_create(mesh.nmb, *mesh.nx, mesh.ng, gamma, *mesh.nrb, (C.c_int * len(lx))(*lx),
                                     (C.c_double * 3)(*mesh.xmin), (C.c_double * 3)(*mesh.xmax))
        if not self._h:
            raise OrcError(L.orcm_last_error().decode())
        shape = (mesh.nmb, 8) + tuple(mesh.state_shape()[2:])
        self.ua = np.zeros(shape)
        self.ub = np.zeros(shape)
        _chk(L.orcm_pack_bind(self._h, self.ua.ctypes.data, self.ub.ctypes.data))
        if threads != 1:
            _chk(L.orcm_set_threads(self._h, threads))
        _chk(L.orcm_pack_set_recon(self._h, recon))
        _chk(L.orcm_pack_set_integrator(self._h, nstages))
        _chk(L.orcm_pack_set_rsolver(self._h, rsolver))

    def load(self, U):
        self.ua[...] = np.asarray(U)
        _chk(lib().orcm_pack_bind(self._h, self.ua.ctypes.data, self.ub.ctypes.data))

    def current(self):
        return self.ua if lib().orcm_pack_current(self._h) == self.ua.ctypes.data else self.ub

    def fill_ghosts(self):
        _chk(lib().orcm_fill_ghosts(self._h))

    def stage(self, stage, dt):
        _chk(lib().orcm_stage(self._h, stage, dt))

    def new_dt(self, cfl):
        dt = C.c_double()
        _chk(lib().orcm_new_dt(self._h, cfl, C.byref(dt)))
        return dt.value

    def floor_count(self):
        return lib().orcm_pack_floor_count(self._h)

    def step(self, cfl, dt=None):
        if dt is None:
            dt = self.new_dt(cfl)
        for s in range(1, self.nstages + 1):
            self.fill_ghosts()
            self.stage(s, dt)
        return dt

    def close(self):
        if self._h:
            lib().orcm_pack_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
