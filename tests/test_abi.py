"""Host-side checks of the C-ABI library that need no GPU: it builds, loads, exports every symbol that
include/ak.h declares, validates arguments, and fails loudly (AK_ECUDA) instead of falling back when no
CUDA device is present."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2409_16053_b200 import ak, build, inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return ak.lib()


def test_every_symbol_of_the_mhd_header_is_exported(L):
    from paper_2409_16053_b200 import ak_mhd
    hdr = open(os.path.join(ROOT, "include", "ak_mhd.h")).read()
    declared = set(re.findall(r"\b(akm_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(ak_mhd.SYMBOLS), declared ^ set(ak_mhd.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name
    # argument checks that need no device
    h = L.akm_pack_create
    h.restype = C.c_void_p
    lx = (C.c_int * 3)(0, 0, 0)
    lo, hi = (C.c_double * 3)(0, 0, 0), (C.c_double * 3)(1, 1, 1)
    assert not h(1, 8, 8, 8, 2, C.c_double(5 / 3), 1, 1, 1, lx, lo, hi)          # ng < 3
    L.akm_last_error.restype = C.c_char_p
    assert b"ng" in L.akm_last_error()
    assert not h(2, 8, 8, 8, 3, C.c_double(5 / 3), 1, 1, 1, lx, lo, hi)          # nmb != nrb1 nrb2 nrb3


def test_every_declared_symbol_is_exported(L):
    hdr = open(os.path.join(ROOT, "include", "ak.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ak_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(ak.SYMBOLS), declared ^ set(ak.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name


def test_no_oracle_or_torch_symbols_in_library():
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", os.path.join(ROOT, "paper_2409_16053_b200", "libak.so")],
                         capture_output=True, text=True).stdout
    names = " ".join(line.split()[-1] for line in out.splitlines() if line.split())   # symbol names, not addresses
    assert "orc_" not in names and "at::" not in names and "c10" not in names and "torch" not in names


def test_create_rejects_bad_arguments(L):
    bad = [
        (0, 8, 8, 8, 2, 5 / 3, 0, 0),      # nmb < 1
        (1, 7, 8, 8, 2, 5 / 3, 0, 0),      # odd nx
        (1, 8, 8, 8, 1, 5 / 3, 0, 0),      # ng too small for PLM
        (1, 8, 8, 8, 2, 5 / 3, 1, 0),      # ng too small for PPM4
        (1, 8, 8, 8, 2, 1.0, 0, 0),        # gamma <= 1
        (1, 8, 8, 8, 2, 5 / 3, 7, 0),      # unknown recon
        (1, 8, 8, 8, 2, 5 / 3, 0, 4),      # unknown rsolver
        (1, 2, 8, 8, 3, 5 / 3, 1, 0),      # nx < ng
    ]
    for args in bad:
        assert not L.ak_pack_create(*args), args
        assert L.ak_last_error()
    h = L.ak_pack_create(1, 8, 8, 8, 2, 5 / 3, 0, 0)
    assert h
    assert L.ak_pack_state_bytes(h) == 5 * 12 ** 3 * 8
    assert L.ak_pack_set_block(h, 0, 0, 0, 0, 0) == -2          # AK_ESTATE: mesh not set
    assert L.ak_pack_set_mesh(h, 1, 1, 1, 0., 1., 0., 1., 0., 0.) == -1
    assert L.ak_pack_set_mesh(h, 1, 1, 1, 0., 1., 0., 1., 0., 1.) == 0
    assert L.ak_pack_set_block(h, 0, 0, 1, 0, 0) == -1          # location out of range
    assert L.ak_pack_set_block(h, 0, 2, 0, 0, 0) == -3          # AK_EUNSUPPORTED: level 2
    assert L.ak_pack_set_block(h, 0, 0, 0, 0, 0) == 0
    assert L.ak_pack_scratch_bytes(h) >= 256 + 16 + 4 + 32
    assert L.ak_fill_ghosts(h) == -2 and L.ak_hydro_stage(h, 1, 1e-3) == -2      # not bound
    assert L.ak_pack_bind(h, 0, 0, 0, 0) == -1
    assert L.ak_pack_bind(h, 0x1000080, 0x2000000, 0x3000000, 0) == -1           # misaligned
    assert L.ak_pack_set_variant(h, 3) == -1 and L.ak_pack_set_variant(h, 2) == 0 and L.ak_pack_set_variant(h, 0) == 0
    assert L.ak_pack_set_tile(h, 4) == -1 and L.ak_pack_set_tile(h, -2) == -1
    assert L.ak_pack_set_tile(h, 3) == 0 and L.ak_pack_set_tile(h, -1) == 0
    assert L.ak_pack_destroy(h) == 0


def test_bind_validates_tiling_before_touching_the_device(L):
    # 2x1x1 root grid with only one block registered twice / a hole / overlapping levels
    def mk(blocks, nmb, ng=2):
        h = L.ak_pack_create(nmb, 4, 4, 4, ng, 5 / 3, 0, 0)
        assert L.ak_pack_set_mesh(h, 2, 1, 1, 0., 1., 0., 1., 0., 1.) == 0
        for m, b in enumerate(blocks):
            assert L.ak_pack_set_block(h, m, *b) == 0
        return h
    fake = (0x10000000, 0x20000000, 0x30000000, 0)
    h = mk([(0, 0, 0, 0), (0, 0, 0, 0)], 2)
    assert L.ak_pack_bind(h, *fake) == -1 and b"duplicate" in L.ak_last_error()
    h = mk([(0, 0, 0, 0)], 2)
    assert L.ak_pack_bind(h, *fake) == -2                        # a block was never set
    h = mk([(0, 0, 0, 0)] + [(1, 2 + (c & 1), (c >> 1) & 1, c >> 2) for c in range(7)], 8)
    assert L.ak_pack_bind(h, *fake) == -1 and b"cover" in L.ak_last_error()
    h = mk([(0, 0, 0, 0), (0, 1, 0, 0), (1, 0, 0, 0)], 3)
    assert L.ak_pack_bind(h, *fake) == -1 and b"overlap" in L.ak_last_error()


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback_without_a_device(L):
    w = I.config0()
    with pytest.raises(ak.AkError):
        ak.Pack(w.mesh, w.gamma, w.recon)
    h = L.ak_pack_create(1, 4, 4, 4, 2, 5 / 3, 0, 0)
    L.ak_pack_set_mesh(h, 1, 1, 1, 0., 1., 0., 1., 0., 1.)
    L.ak_pack_set_block(h, 0, 0, 0, 0, 0)
    assert L.ak_pack_bind(h, 0x10000000, 0x20000000, 0x30000000, 0) == -4      # AK_ECUDA, loudly
    assert L.ak_last_error()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2409_16053_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "orc_" not in src and "import oracle" not in src and "from oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r'#include\s+"[^"]*ak[_.]', src) and "libak" not in src and "ak_pack" not in src, f
            assert not re.search(r"import\s+ak\b|\.ak\b", src), f
