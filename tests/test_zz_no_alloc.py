"""ak_new_dt_noalloc (include/ak.h): the CFL reduction for callers that may not allocate device memory.  Its scratch is a
128 KiB static device array inside libak.so that every call shares and that keeps the last call's contents, so the test makes
TWO calls in a row on DIFFERENT states and mesh shapes and compares each with the existing path (ak_new_dt on a pack with
caller-allocated scratch), with the tolerance the dt tests use: bit-identical.  In a file of its own that pytest collects
last; passes alone in a fresh process and after the other tests.
"""
import ctypes as C

import pytest
import torch

from paper_2409_16053_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ak():
    from paper_2409_16053_b200 import ak as _ak
    _ak.lib()
    assert torch.cuda.is_available()
    return _ak


def existing_path_dt(ak, w, U):
    """ak_new_dt on a freshly loaded pack: the stand-alone reduction kernel with the pack's own scratch buffer."""
    pg = ak.Pack(w.mesh, w.gamma, w.recon)
    pg.load(U)
    l0 = pg.launch_count()
    dt = pg.new_dt(w.cfl)
    assert pg.launch_count() - l0 == 2                      # dt_init + new_dt kernels ran (not the cached fused path)
    pg.close()
    return dt


def test_two_calls_in_a_row_match_the_existing_path_bit_for_bit(ak):
    # call 1: 8 blocks of 16^3, ng = 2 (short rows: several rows per warp); call 2: 27 ragged blocks, ng = 3, another
    # state, with MORE blocks than call 1 (table entries beyond call 1's are stale or never written before) and a
    # smaller dt (the minimum cell left by call 1 must not survive)
    w1 = I.config1(nrb=2, nx=16)
    w2 = I.config3(nrb=1, nx=16)
    w2.mesh = I.uniform_mesh((3, 3, 3), (34, 10, 6), 3)
    dev = torch.device("cuda", 0)
    U1, U2 = w1.state(device=dev), w2.state(device=dev)
    ref1, ref2 = existing_path_dt(ak, w1, U1), existing_path_dt(ak, w2, U2)
    assert ref1 != ref2
    got1 = ak.new_dt_noalloc(U1, w1.mesh, w1.gamma, w1.cfl)
    got2 = ak.new_dt_noalloc(U2, w2.mesh, w2.gamma, w2.cfl)
    assert got1 == ref1 and got2 == ref2, (got1, ref1, got2, ref2)
    # and back again: the larger table and the smaller minimum of call 2 are stale now
    assert ak.new_dt_noalloc(U1, w1.mesh, w1.gamma, w1.cfl) == ref1
    # after a step the pack's dt comes from the reduction fused into stage 2: the same bits again
    pg = ak.Pack(w1.mesh, w1.gamma, w1.recon)
    pg.load(U1)
    pg.step(w1.cfl)
    assert ak.new_dt_noalloc(pg.current(), w1.mesh, w1.gamma, w1.cfl) == pg.new_dt(w1.cfl)
    # a side stream
    s = torch.cuda.Stream(device=dev)
    s.wait_stream(torch.cuda.current_stream(dev))
    assert ak.new_dt_noalloc(U2, w2.mesh, w2.gamma, w2.cfl, stream=s) == ref2


def test_limits_and_errors(ak):
    L = ak.lib()
    dev = torch.device("cuda", 0)
    w = I.config1(nrb=1, nx=16)
    U = w.state(device=dev)
    dt = C.c_double()
    dx = w.mesh.dx(0)
    st = torch.cuda.current_stream(dev).cuda_stream
    args = lambda nmb: (U.data_ptr(), nmb, 16, 16, 16, 2, w.gamma, dx[0], dx[1], dx[2], w.cfl, st, C.byref(dt))
    # beyond the static array: a clear error, nothing launched (the pointer would be far too small for 8177 blocks)
    assert L.ak_new_dt_noalloc(*args(8177)) == -3
    assert b"8176" in L.ak_last_error() and b"128 KiB" in L.ak_last_error()
    assert L.ak_new_dt_noalloc(*args(0)) == -1
    host = torch.zeros(w.mesh.state_shape(), dtype=torch.float64)
    assert L.ak_new_dt_noalloc(host.data_ptr(), 1, 16, 16, 16, 2, w.gamma, dx[0], dx[1], dx[2], w.cfl, st, C.byref(dt)) != 0
    # a NaN momentum is reported like ak_new_dt reports it, and the next call on a healthy state is unaffected
    bad = U.clone()
    bad[0, 2, 5, 7, 9] = float("nan")
    with pytest.raises(ak.AkError) as ei:
        ak.new_dt_noalloc(bad, w.mesh, w.gamma, w.cfl)
    assert "non-finite" in str(ei.value)
    assert ak.new_dt_noalloc(U, w.mesh, w.gamma, w.cfl) == existing_path_dt(ak, w, U)
    # the entry point allocates nothing: device memory in use is unchanged across calls
    torch.cuda.synchronize(dev)
    free0 = torch.cuda.mem_get_info(dev)[0]
    for _ in range(5):
        ak.new_dt_noalloc(U, w.mesh, w.gamma, w.cfl)
    assert torch.cuda.mem_get_info(dev)[0] == free0
