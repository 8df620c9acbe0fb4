"""ctypes view of liborc.so (oracle/orc.cpp) -- TEST INFRASTRUCTURE ONLY, see oracle/orc.h.

build() compiles the oracle with g++ (-O2 -ffp-contract=off -fno-fast-math -fopenmp); OrcPack wraps
the orc_* calls on caller-owned numpy arrays laid out U[m][n][k][j][i].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liborc.so")
_SRC = [os.path.join(_HERE, "orc.cpp"), os.path.join(_HERE, "orc.h")]
_lib = None


def build(force: bool = False) -> str:
    if (not force and os.path.exists(_SO)
            and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC)):
        return _SO
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-Wall",
           "-o", _SO, _SRC[0]]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    dp = C.POINTER(C.c_double)
    L.orc_pack_create.restype = C.c_void_p
    L.orc_pack_create.argtypes = [C.c_int] * 5 + [C.c_double, C.c_int, C.c_int]
    L.orc_pack_set_mesh.argtypes = [C.c_void_p] + [C.c_int] * 3 + [C.c_double] * 6
    L.orc_pack_set_block.argtypes = [C.c_void_p] + [C.c_int] * 5
    L.orc_pack_bind.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.orc_pack_set_boundaries.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
    L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
    L.orc_set_flux_correction.argtypes = [C.c_void_p, C.c_int]
    L.orc_set_fofc.argtypes = [C.c_void_p, C.c_int]
    L.orc_pack_fofc_count.restype = C.c_longlong
    L.orc_pack_fofc_count.argtypes = [C.c_void_p]
    L.orc_set_integrator.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
    L.orc_fill_ghosts.argtypes = [C.c_void_p]
    L.orc_hydro_stage.argtypes = [C.c_void_p, C.c_int, C.c_double]
    L.orc_new_dt.argtypes = [C.c_void_p, C.c_double, dp]
    L.orc_pack_current.restype = C.c_void_p
    L.orc_pack_current.argtypes = [C.c_void_p]
    L.orc_pack_floor_count.restype = C.c_longlong
    L.orc_pack_floor_count.argtypes = [C.c_void_p]
    L.orc_pack_destroy.argtypes = [C.c_void_p]
    L.orc_last_error.restype = C.c_char_p
    L.orc_c2p.argtypes = [C.c_double, dp, dp, C.POINTER(C.c_int)]
    L.orc_c2p.restype = None
    L.orc_plm.argtypes = [C.c_double] * 3 + [dp, dp]
    L.orc_plm.restype = None
    for f in (L.orc_ppm4, L.orc_ppmx, L.orc_wenoz):
        f.argtypes = [dp, dp, dp]
        f.restype = None
    L.orc_ppm4_iface.argtypes = [C.c_double] * 4 + [dp]
    L.orc_ppm4_iface.restype = None
    L.orc_hllc.argtypes = [C.c_double, C.c_int, dp, dp, dp]
    L.orc_hllc.restype = None
    for f in (L.orc_llf, L.orc_hlle, L.orc_roe):
        f.argtypes = [C.c_double, C.c_int, dp, dp, dp]
        f.restype = None
    _lib = L
    return L


class OrcError(RuntimeError):
    pass


def _chk(rc):
    if rc != 0:
        raise OrcError(lib().orc_last_error().decode())


def _arr5(x):
    return (C.c_double * 5)(*[float(v) for v in x])


# ---- single-operation entry points --------------------------------------------------------------
def c2p(gamma, U):
    W = (C.c_double * 5)()
    fl = C.c_int(0)
    lib().orc_c2p(gamma, _arr5(U), W, C.byref(fl))
    return np.array(W[:]), fl.value


def plm(qm1, q0, qp1):
    a, b = C.c_double(), C.c_double()
    lib().orc_plm(qm1, q0, qp1, C.byref(a), C.byref(b))
    return a.value, b.value


def ppm4(q5):
    a, b = C.c_double(), C.c_double()
    lib().orc_ppm4(_arr5(q5), C.byref(a), C.byref(b))
    return a.value, b.value


def ppmx(q5):
    a, b = C.c_double(), C.c_double()
    lib().orc_ppmx(_arr5(q5), C.byref(a), C.byref(b))
    return a.value, b.value


def wenoz(q5):
    a, b = C.c_double(), C.c_double()
    lib().orc_wenoz(_arr5(q5), C.byref(a), C.byref(b))
    return a.value, b.value


def ppm4_iface(qm1, q0, qp1, qp2):
    a = C.c_double()
    lib().orc_ppm4_iface(qm1, q0, qp1, qp2, C.byref(a))
    return a.value


def hllc(gamma, direction, WL, WR):
    F = (C.c_double * 5)()
    lib().orc_hllc(gamma, direction, _arr5(WL), _arr5(WR), F)
    return np.array(F[:])


def llf(gamma, direction, WL, WR):
    F = (C.c_double * 5)()
    lib().orc_llf(gamma, direction, _arr5(WL), _arr5(WR), F)
    return np.array(F[:])


def roe(gamma, direction, WL, WR):
    F = (C.c_double * 5)()
    lib().orc_roe(gamma, direction, _arr5(WL), _arr5(WR), F)
    return np.array(F[:])


def hlle(gamma, direction, WL, WR):
    F = (C.c_double * 5)()
    lib().orc_hlle(gamma, direction, _arr5(WL), _arr5(WR), F)
    return np.array(F[:])


# ---- pack ---------------------------------------------------------------------------------------
class OrcPack:
    """Oracle pack over a Mesh (paper_2409_16053_b200.inputs.Mesh); owns two numpy state buffers."""

    def __init__(self, mesh, gamma, recon, rsolver=0, threads=1):
        L = lib()
        self.mesh = mesh
        self._h = L.orc_pack_create(mesh.nmb, *mesh.nx, mesh.ng, gamma, recon, rsolver)
        if not self._h:
            raise OrcError(L.orc_last_error().decode())
        _chk(L.orc_pack_set_mesh(self._h, *mesh.nrb, mesh.xmin[0], mesh.xmax[0], mesh.xmin[1], mesh.xmax[1],
                                 mesh.xmin[2], mesh.xmax[2]))
        for m, (lev, l1, l2, l3) in enumerate(mesh.blocks):
            _chk(L.orc_pack_set_block(self._h, m, lev, l1, l2, l3))
        bc = tuple(getattr(mesh, "bc", (0,) * 6))
        if any(bc):
            _chk(L.orc_pack_set_boundaries(self._h, (C.c_int * 6)(*bc)))
        self.ua = np.zeros(mesh.state_shape(), dtype=np.float64)
        self.ub = np.zeros(mesh.state_shape(), dtype=np.float64)
        _chk(L.orc_pack_bind(self._h, self.ua.ctypes.data, self.ub.ctypes.data))
        if threads != 1:
            _chk(L.orc_set_threads(self._h, threads))

    def set_integrator(self, nstages):
        """1 = forward Euler, 2 = SSPRK(2,2) (default), 3 = SSPRK(3,3) (allocates the third register)."""
        uc = np.zeros(self.mesh.state_shape(), dtype=np.float64) if nstages == 3 else None
        _chk(lib().orc_set_integrator(self._h, nstages, uc.ctypes.data if nstages == 3 else None))
        self.nstages, self.uc = nstages, uc

    def set_flux_correction(self, on=True):
        """f1 of SURVEY 8(f): coarse fluxes at level-boundary faces <- mean of the four fine fluxes (off by default)."""
        _chk(lib().orc_set_flux_correction(self._h, 1 if on else 0))

    def set_fofc(self, on=True):
        """f2 of SURVEY 8(f): first-order flux correction (off by default)."""
        _chk(lib().orc_set_fofc(self._h, 1 if on else 0))

    def fofc_count(self):
        return lib().orc_pack_fofc_count(self._h)

    def load(self, U):
        """Copy U^n (numpy or CPU torch tensor of the state shape) into buffer A and make it current."""
        self.ua[...] = np.asarray(U)
        _chk(lib().orc_pack_bind(self._h, self.ua.ctypes.data, self.ub.ctypes.data))

    def current(self):
        p = lib().orc_pack_current(self._h)
        if getattr(self, "uc", None) is not None and p == self.uc.ctypes.data:
            return self.uc
        return self.ua if p == self.ua.ctypes.data else self.ub

    def fill_ghosts(self):
        _chk(lib().orc_fill_ghosts(self._h))

    def hydro_stage(self, stage, dt):
        _chk(lib().orc_hydro_stage(self._h, stage, dt))

    def new_dt(self, cfl):
        dt = C.c_double()
        _chk(lib().orc_new_dt(self._h, cfl, C.byref(dt)))
        return dt.value

    def floor_count(self):
        return lib().orc_pack_floor_count(self._h)

    def step(self, cfl, dt=None):
        """One RK step in the call order of SURVEY section 3: dt; nstages x (fill, stage).  Returns dt."""
        if dt is None:
            dt = self.new_dt(cfl)
        for stage in range(1, getattr(self, "nstages", 2) + 1):
            self.fill_ghosts()
            self.hydro_stage(stage, dt)
        return dt

    def close(self):
        if self._h:
            lib().orc_pack_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
