"""ctypes binding of the MHD entry points of libak.so (include/ak_mhd.h): argument marshalling only.

PyTorch allocates the device buffers and supplies the stream; every step of the path runs in the CUDA kernels of
csrc/mhd/ak_mhd.cu.  There is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C

import torch

from . import ak as _ak

SYMBOLS = [
    "akm_pack_create", "akm_pack_state_bytes", "akm_pack_work_bytes", "akm_pack_bind", "akm_fill_ghosts", "akm_stage",
    "akm_new_dt", "akm_step", "akm_pack_current", "akm_pack_floor_count", "akm_pack_launch_count", "akm_pack_destroy",
    "akm_last_error", "akm_pack_set_exact", "akm_pack_set_recon", "akm_pack_set_integrator", "akm_pack_set_rsolver",
]
_ready = False


class AkmError(RuntimeError):
    pass


def lib():
    """libak.so with the akm_* signatures set."""
    global _ready
    L = _ak.lib()
    if not _ready:
        vp, i, d, sz, ll = C.c_void_p, C.c_int, C.c_double, C.c_size_t, C.c_longlong
        dp, ip = C.POINTER(d), C.POINTER(i)
        sig = {
            "akm_pack_create": (vp, [i, i, i, i, i, d, i, i, i, ip, dp, dp]),
            "akm_pack_state_bytes": (sz, [vp]), "akm_pack_work_bytes": (sz, [vp]),
            "akm_pack_bind": (i, [vp, vp, vp, vp, vp]),
            "akm_fill_ghosts": (i, [vp]), "akm_stage": (i, [vp, i, d]),
            "akm_new_dt": (i, [vp, d, dp]), "akm_step": (i, [vp, d, d, dp]),
            "akm_pack_current": (vp, [vp]), "akm_pack_floor_count": (ll, [vp]), "akm_pack_launch_count": (ll, [vp]),
            "akm_pack_destroy": (i, [vp]), "akm_last_error": (C.c_char_p, []), "akm_pack_set_exact": (i, [vp, i]),
            "akm_pack_set_recon": (i, [vp, i]), "akm_pack_set_integrator": (i, [vp, i]), "akm_pack_set_rsolver": (i, [vp, i]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _ready = True
    return L


def _chk(rc):
    if rc != 0:
        raise AkmError(f"akm error {rc}: {lib().akm_last_error().decode()}")


class MhdPack:
    """An MHD MeshBlockPack (uniform periodic mesh) bound to torch-owned device buffers; methods map 1:1 to akm_* calls."""

    def __init__(self, mesh, gamma, device="cuda:0", stream=None, exact=False, recon=0, nstages=2, rsolver=0):
        L = lib()
        if not torch.cuda.is_available():
            raise AkmError("no CUDA device: the MHD path has no CPU fallback")
        self.mesh, self.device = mesh, torch.device(device)
        lx = [v for (_, l1, l2, l3) in mesh.blocks for v in (l1, l2, l3)]
        self._h = L.akm_pack_create(mesh.nmb, *mesh.nx, mesh.ng, gamma, *mesh.nrb, (C.c_int * len(lx))(*lx),
                                    (C.c_double * 3)(*mesh.xmin), (C.c_double * 3)(*mesh.xmax))
        if not self._h:
            raise AkmError(L.akm_last_error().decode())
        shape = (mesh.nmb, 8) + tuple(mesh.state_shape()[2:])
        with torch.cuda.device(self.device):
            self.ua = torch.zeros(shape, dtype=torch.float64, device=self.device)
            self.ub = torch.zeros(shape, dtype=torch.float64, device=self.device)
            self.work = torch.zeros(L.akm_pack_work_bytes(self._h), dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            torch.cuda.synchronize(self.device)
        assert L.akm_pack_state_bytes(self._h) == self.ua.numel() * 8
        self._bind()
        if exact:
            _chk(L.akm_pack_set_exact(self._h, 1))
        if recon:
            _chk(L.akm_pack_set_recon(self._h, recon))
        if nstages != 2:
            _chk(L.akm_pack_set_integrator(self._h, nstages))
        if rsolver:
            _chk(L.akm_pack_set_rsolver(self._h, rsolver))
        self.nstages = nstages

    def _bind(self):
        _chk(lib().akm_pack_bind(self._h, self.ua.data_ptr(), self.ub.data_ptr(), self.work.data_ptr(), self.stream.cuda_stream))

    def load(self, U):
        with torch.cuda.stream(self.stream):
            self.ua.copy_(U.to(self.device, non_blocking=True))
        self.stream.synchronize()
        self._bind()

    def current(self) -> torch.Tensor:
        return self.ua if lib().akm_pack_current(self._h) == self.ua.data_ptr() else self.ub

    def fill_ghosts(self):
        _chk(lib().akm_fill_ghosts(self._h))

    def stage(self, stage, dt):
        _chk(lib().akm_stage(self._h, stage, dt))

    def new_dt(self, cfl):
        dt = C.c_double()
        _chk(lib().akm_new_dt(self._h, cfl, C.byref(dt)))
        return dt.value

    def step(self, cfl, dt=None):
        out = C.c_double()
        _chk(lib().akm_step(self._h, cfl, 0.0 if dt is None else dt, C.byref(out)))
        return out.value

    def floor_count(self):
        return lib().akm_pack_floor_count(self._h)

    def launch_count(self):
        return lib().akm_pack_launch_count(self._h)

    def close(self):
        if getattr(self, "_h", None):
            lib().akm_pack_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
