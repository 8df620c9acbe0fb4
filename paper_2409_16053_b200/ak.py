"""Thin binding over libak.so (include/ak.h): argument marshalling only.

Every step of the path runs inside the library's CUDA kernels; PyTorch is used here to allocate device
memory and to supply the stream (P:63 device-resident arrays, P:65 host drives / device computes).
There is no CPU fallback: if the library is missing or cannot be loaded, importing the symbols raises.
The function names mirror the C-ABI one to one.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libak.so")
_lib = None

AK_OK = 0
RECON_PLM, RECON_PPM4 = 0, 1
RSOLVER_HLLC, RSOLVER_LLF, RSOLVER_HLLE, RSOLVER_ROE = 0, 1, 2, 3

SYMBOLS = [
    "ak_last_error", "ak_pack_create", "ak_pack_set_mesh", "ak_pack_set_block", "ak_pack_state_bytes",
    "ak_pack_scratch_bytes", "ak_pack_bind", "ak_fill_ghosts", "ak_hydro_stage", "ak_new_dt", "ak_step",
    "ak_pack_current", "ak_pack_upload", "ak_pack_download", "ak_pack_download_async", "ak_pack_floor_count", "ak_pack_set_variant", "ak_pack_set_tile", "ak_pack_set_flux_correction", "ak_pack_set_ghost_push", "ak_pack_set_fofc", "ak_pack_fofc_count", "ak_pack_set_boundaries", "ak_pack_set_integrator",
    "ak_pack_launch_count", "ak_pack_destroy", "ak_new_dt_noalloc",
]


class AkError(RuntimeError):
    pass


def lib():
    """Load libak.so (built in-tree by paper_2409_16053_b200.build).  Raises if it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise AkError(f"{_SO} not found: run `python -m paper_2409_16053_b200.build` (no CPU fallback exists)")
    L = C.CDLL(_SO)
    vp, i, d, sz, ll = C.c_void_p, C.c_int, C.c_double, C.c_size_t, C.c_longlong
    sig = {
        "ak_last_error": (C.c_char_p, []),
        "ak_pack_create": (vp, [i, i, i, i, i, d, i, i]),
        "ak_pack_set_mesh": (i, [vp, i, i, i, d, d, d, d, d, d]),
        "ak_pack_set_block": (i, [vp, i, i, i, i, i]),
        "ak_pack_state_bytes": (sz, [vp]),
        "ak_pack_scratch_bytes": (sz, [vp]),
        "ak_pack_bind": (i, [vp, vp, vp, vp, vp]),
        "ak_fill_ghosts": (i, [vp]),
        "ak_hydro_stage": (i, [vp, i, d]),
        "ak_new_dt": (i, [vp, d, C.POINTER(d)]),
        "ak_step": (i, [vp, d, d, C.POINTER(d)]),
        "ak_pack_current": (vp, [vp]),
        "ak_pack_upload": (i, [vp, vp]),
        "ak_pack_download": (i, [vp, vp]),
        "ak_pack_download_async": (i, [vp, vp]),
        "ak_pack_floor_count": (ll, [vp]),
        "ak_pack_set_variant": (i, [vp, i]),
        "ak_pack_set_ghost_push": (i, [vp, i]),
        "ak_pack_set_fofc": (i, [vp, i, vp]),
        "ak_pack_fofc_count": (C.c_longlong, [vp]),
        "ak_pack_set_tile": (i, [vp, i]),
        "ak_pack_set_flux_correction": (i, [vp, i]),
        "ak_pack_set_boundaries": (i, [vp, C.POINTER(C.c_int)]),
        "ak_pack_set_integrator": (i, [vp, i, vp]),
        "ak_pack_launch_count": (ll, [vp]),
        "ak_pack_destroy": (i, [vp]),
        "ak_new_dt_noalloc": (i, [vp, i, i, i, i, i, d, d, d, d, d, vp, C.POINTER(d)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def _chk(rc):
    if rc != AK_OK:
        raise AkError(f"ak error {rc}: {lib().ak_last_error().decode()}")


def new_dt_noalloc(U, mesh, gamma, cfl, stream=None):
    """ak_new_dt_noalloc: the CFL reduction on a device tensor U of mesh.state_shape() (uniform single-level mesh) with
    the library's static scratch array -- no pack, no allocation (include/ak.h)."""
    assert U.is_cuda and U.is_contiguous() and U.dtype == torch.float64 and tuple(U.shape) == tuple(mesh.state_shape())
    st = stream if stream is not None else torch.cuda.current_stream(U.device)
    dx = mesh.dx(0)
    dt = C.c_double()
    _chk(lib().ak_new_dt_noalloc(U.data_ptr(), mesh.nmb, *mesh.nx, mesh.ng, gamma, dx[0], dx[1], dx[2], cfl,
                                 st.cuda_stream, C.byref(dt)))
    return dt.value


class Pack:
    """A MeshBlockPack bound to torch-owned device buffers.  Methods map 1:1 to the ak_* calls."""

    def __init__(self, mesh, gamma, recon, rsolver=RSOLVER_HLLC, device="cuda:0", stream=None, variant=0):
        L = lib()
        if not torch.cuda.is_available():
            raise AkError("no CUDA device: the hydro path has no CPU fallback")
        self.mesh = mesh
        self.device = torch.device(device)
        self._h = L.ak_pack_create(mesh.nmb, *mesh.nx, mesh.ng, gamma, recon, rsolver)
        if not self._h:
            raise AkError(L.ak_last_error().decode())
        _chk(L.ak_pack_set_mesh(self._h, *mesh.nrb, mesh.xmin[0], mesh.xmax[0], mesh.xmin[1], mesh.xmax[1],
                                mesh.xmin[2], mesh.xmax[2]))
        for m, (lev, l1, l2, l3) in enumerate(mesh.blocks):
            _chk(L.ak_pack_set_block(self._h, m, lev, l1, l2, l3))
        bc = tuple(getattr(mesh, "bc", (0,) * 6))
        if any(bc):
            _chk(L.ak_pack_set_boundaries(self._h, (C.c_int * 6)(*bc)))
        nbytes = L.ak_pack_state_bytes(self._h)
        assert nbytes == 8 * int(torch.tensor(mesh.state_shape()).prod())
        with torch.cuda.device(self.device):
            self.ua = torch.zeros(mesh.state_shape(), dtype=torch.float64, device=self.device)
            self.ub = torch.zeros(mesh.state_shape(), dtype=torch.float64, device=self.device)
            self.scratch = torch.zeros(L.ak_pack_scratch_bytes(self._h), dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            torch.cuda.synchronize(self.device)
            _chk(L.ak_pack_bind(self._h, self.ua.data_ptr(), self.ub.data_ptr(), self.scratch.data_ptr(),
                                self.stream.cuda_stream))
        if variant:
            _chk(L.ak_pack_set_variant(self._h, variant))

    # ---- state -----------------------------------------------------------------------------------
    def load(self, U):
        """Device-side load of U^n (tensor of mesh.state_shape()) into buffer A; A becomes current."""
        with torch.cuda.stream(self.stream):
            self.ua.copy_(U.to(self.device, non_blocking=True))
        self.stream.synchronize()
        _chk(lib().ak_pack_bind(self._h, self.ua.data_ptr(), self.ub.data_ptr(), self.scratch.data_ptr(),
                                self.stream.cuda_stream))
        if getattr(self, "_fofc", False):
            self.set_fofc(True)                  # (the spare and buffer A trade places every step: re-arm after the re-bind)

    def current(self) -> torch.Tensor:
        p = lib().ak_pack_current(self._h)
        if getattr(self, "uc", None) is not None and p == self.uc.data_ptr():
            return self.uc
        if getattr(self, "uf", None) is not None and p == self.uf.data_ptr():
            return self.uf
        return self.ua if p == self.ua.data_ptr() else self.ub

    def set_integrator(self, nstages):
        """1 = forward Euler, 2 = SSPRK(2,2) (default), 3 = SSPRK(3,3): allocates the third state register."""
        with torch.cuda.device(self.device):
            uc = torch.zeros(self.mesh.state_shape(), dtype=torch.float64, device=self.device) if nstages == 3 else None
        _chk(lib().ak_pack_set_integrator(self._h, nstages, uc.data_ptr() if nstages == 3 else None))
        self.nstages, self.uc = nstages, uc

    def upload(self, host_tensor):
        """ak_pack_upload: HOST (ideally pinned) tensor -> buffer A through the C-ABI."""
        assert host_tensor.device.type == "cpu" and host_tensor.is_contiguous() and host_tensor.dtype == torch.float64
        _chk(lib().ak_pack_upload(self._h, host_tensor.data_ptr()))

    def download_async(self, host_tensor):
        assert host_tensor.device.type == "cpu" and host_tensor.is_contiguous() and host_tensor.dtype == torch.float64
        _chk(lib().ak_pack_download_async(self._h, host_tensor.data_ptr()))

    def download(self, host_tensor):
        assert host_tensor.device.type == "cpu" and host_tensor.is_contiguous() and host_tensor.dtype == torch.float64
        _chk(lib().ak_pack_download(self._h, host_tensor.data_ptr()))

    # ---- the hot path ----------------------------------------------------------------------------
    def fill_ghosts(self):
        _chk(lib().ak_fill_ghosts(self._h))

    def hydro_stage(self, stage, dt):
        _chk(lib().ak_hydro_stage(self._h, stage, dt))

    def new_dt(self, cfl):
        dt = C.c_double()
        _chk(lib().ak_new_dt(self._h, cfl, C.byref(dt)))
        return dt.value

    def step(self, cfl, dt=None):
        out = C.c_double()
        _chk(lib().ak_step(self._h, cfl, 0.0 if dt is None else dt, C.byref(out)))
        return out.value

    def floor_count(self):
        n = lib().ak_pack_floor_count(self._h)
        if n < 0:
            raise AkError(lib().ak_last_error().decode())
        return n

    def launch_count(self):
        return lib().ak_pack_launch_count(self._h)

    def set_variant(self, v):
        _chk(lib().ak_pack_set_variant(self._h, v))

    def set_flux_correction(self, on=True):
        _chk(lib().ak_pack_set_flux_correction(self._h, 1 if on else 0))

    def set_fofc(self, on=True):
        """P:118 first-order flux correction: allocates the spare buffer the last stage of a step then writes."""
        if on and getattr(self, "uf", None) is None:
            with torch.cuda.device(self.device):
                self.uf = torch.zeros(self.mesh.state_shape(), dtype=torch.float64, device=self.device)
        self._fofc = bool(on)
        _chk(lib().ak_pack_set_fofc(self._h, 1 if on else 0, self.uf.data_ptr() if on else None))

    def fofc_count(self):
        n = lib().ak_pack_fofc_count(self._h)
        if n < 0:
            raise AkError(lib().ak_last_error().decode())
        return n

    def set_ghost_push(self, on=True):
        _chk(lib().ak_pack_set_ghost_push(self._h, 1 if on else 0))

    def set_tile(self, t):
        _chk(lib().ak_pack_set_tile(self._h, t))

    def close(self):
        if getattr(self, "_h", None):
            lib().ak_pack_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
