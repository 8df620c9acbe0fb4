"""Pins for the oracle's higher-order reconstructions (paper P:101): WENOZ (Q29) and
PPMX (Q30).  Nothing here compares the oracle with itself: polynomial exactness, formal order on a smooth function,
behaviour at a step and at a smooth extremum (where PPMX must differ from PPM4), mirror symmetry, and -- what the
paper states -- fourth-order (or better) convergence of the 1-D linear wave with SSPRK(3,3).
"""
import json
import math
import os

import numpy as np
import pytest

from paper_2409_16053_b200 import inputs as I
from tests.test_oracle_scheme import act

GOLD_C = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "appendix_c.json")))
GOLD_R = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "recon.json")))    # tests/golden/make_recon.py
RECON_PPMX, RECON_WENOZ = 2, 3


def poly_avg(c, i):
    """Cell average over [i-1/2, i+1/2] of sum_k c[k] x^k."""
    return sum(ck * ((i + 0.5) ** (k + 1) - (i - 0.5) ** (k + 1)) / (k + 1) for k, ck in enumerate(c))


def poly_val(c, x):
    return sum(ck * x ** k for k, ck in enumerate(c))


def test_worked_numbers_of_the_stand_alone_script(orc):
    # a second, vectorised numpy implementation of readings Q29 / Q30 on the 9-point sequence of SURVEY A.3 (steps, an
    # extremum, a monotone ramp): a wrong branch or coefficient in either implementation shows at O(0.1)
    q = GOLD_R["recon_q"]
    for name, fn in (("ppmx", orc.ppmx), ("wenoz", orc.wenoz)):
        for i, (qm, qp) in GOLD_R[name].items():
            i = int(i)
            a, b = fn(q[i - 2:i + 3])
            assert a == pytest.approx(qm, rel=0, abs=1e-14) and b == pytest.approx(qp, rel=0, abs=1e-14), (name, i)


# ------------------------------------------------------------------ WENOZ -------------------------
def test_wenoz_is_exact_for_quadratics_whatever_the_weights(orc):
    # every candidate stencil reproduces a parabola's face value from its cell averages exactly, so any convex
    # combination does; a wrong coefficient in a candidate polynomial breaks this at O(1)
    rng = np.random.default_rng(5)
    for _ in range(200):
        c = rng.normal(size=3)
        q = [poly_avg(c, i) for i in range(-2, 3)]
        qm, qp = orc.wenoz(q)
        scale = max(abs(x) for x in q) + 1.0
        assert abs(qp - poly_val(c, 0.5)) <= 64 * np.spacing(scale)
        assert abs(qm - poly_val(c, -0.5)) <= 64 * np.spacing(scale)


def test_wenoz_is_fifth_order_on_a_smooth_function(orc):
    # cell averages of sin(x): the face value converges at h^5 (ratio 32 per halving) where the solution is smooth
    errs = []
    for h in (0.2, 0.1, 0.05, 0.025):
        x0 = 0.7
        avg = lambda i: (math.cos(x0 + (i - 0.5) * h) - math.cos(x0 + (i + 0.5) * h)) / h
        qm, qp = orc.wenoz([avg(i) for i in range(-2, 3)])
        errs.append(max(abs(qp - math.sin(x0 + 0.5 * h)), abs(qm - math.sin(x0 - 0.5 * h))))
    for a, b in zip(errs, errs[1:]):
        assert 24.0 <= a / b <= 40.0, errs


def test_wenoz_step_uniform_and_mirror(orc):
    # at a step the weights collapse onto the smooth stencil: no oscillation (the face value is that of the flat side)
    qm, qp = orc.wenoz([0.0, 0.0, 0.0, 1.0, 1.0])
    assert abs(qp) < 1e-30 and abs(qm) < 1e-30             # (the other stencils keep weights of order eps^2)
    qm, qp = orc.wenoz([0.0, 0.0, 1.0, 1.0, 1.0])
    assert abs(qp - 1.0) < 1e-15 and abs(qm - 1.0) < 1e-15
    assert orc.wenoz([2.5] * 5) == (2.5, 2.5)
    rng = np.random.default_rng(6)
    for _ in range(200):
        q = rng.normal(size=5)
        a, b = orc.wenoz(q)
        b2, a2 = orc.wenoz(q[::-1].copy())
        assert a == a2 and b == b2                          # bit-exact mirror symmetry


# ------------------------------------------------------------------ PPMX --------------------------
def test_ppmx_linear_and_cubic_data(orc):
    rng = np.random.default_rng(7)
    for _ in range(100):
        a0, s = rng.normal(), rng.normal()
        q = [a0 + s * i for i in range(-2, 3)]
        qm, qp = orc.ppmx(q)
        assert abs(qm - (a0 - 0.5 * s)) <= 8 * np.spacing(abs(a0) + abs(s) + 1) and abs(qp - (a0 + 0.5 * s)) <= 8 * np.spacing(abs(a0) + abs(s) + 1)
    # a monotone cubic: the fourth-order interface values are exact and no limiter acts
    c = [0.3, 10.0, 0.2, 1.0]
    q = [poly_avg(c, i) for i in range(-2, 3)]
    qm, qp = orc.ppmx(q)
    assert abs(qp - poly_val(c, 0.5)) <= 1e-13 and abs(qm - poly_val(c, -0.5)) <= 1e-13


def test_ppmx_keeps_a_smooth_extremum_where_ppm4_flattens_it(orc):
    # cell averages of a parabola with its maximum inside the middle cell: PPMX returns the parabola's own edge
    # values (the limited second derivative equals the parabola's), PPM4 (CW84) sets both edges to the cell average
    for x0 in (0.0, 0.2, -0.35):
        c = [1.0 - x0 * x0, 2.0 * x0, -1.0]                 # 1 - (x - x0)^2
        q = [poly_avg(c, i) for i in range(-2, 3)]
        qm, qp = orc.ppmx(q)
        assert abs(qm - poly_val(c, -0.5)) <= 1e-14 and abs(qp - poly_val(c, 0.5)) <= 1e-14
        m4, p4 = orc.ppm4(q)
        assert m4 == q[2] and p4 == q[2]
    # a non-smooth extremum (a single spike) is still flattened
    assert orc.ppmx([0.0, 0.0, 1.0, 0.0, 0.0]) == (1.0, 1.0)


def test_ppmx_step_no_new_extrema_and_mirror(orc):
    for q in ([0.0, 0.0, 0.0, 1.0, 1.0], [0.0, 0.0, 1.0, 1.0, 1.0], [0.0, 0.1, 0.5, 0.9, 1.0], [1.0, 2.0, 4.0, 7.0, 8.0]):
        qm, qp = orc.ppmx(q)
        lo, hi = min(q[1:4]), max(q[1:4])
        assert lo - 1e-15 <= qm <= hi + 1e-15 and lo - 1e-15 <= qp <= hi + 1e-15, (q, qm, qp)
        # the parabola through (qm, a, qp) is monotone inside the cell: each edge increment at most twice the other
        dm, dp = q[2] - qm, qp - q[2]
        assert abs(dm) <= 2 * abs(dp) + 1e-15 and abs(dp) <= 2 * abs(dm) + 1e-15
    rng = np.random.default_rng(8)
    for _ in range(300):
        q = rng.normal(size=5)
        a, b = orc.ppmx(q)
        b2, a2 = orc.ppmx(q[::-1].copy())
        assert a == a2 and b == b2


# ------------------------------------------------------------------ scheme order (paper P:130) ----
def wave_error_rk3(orc, N, recon, cfl):
    mesh = I.uniform_mesh((1, 1, 1), (N, 4, 4), 3)
    U0 = I.make_state(mesh, I.sound_wave_prim()).numpy()
    p = orc.OrcPack(mesh, I.GAMMA, recon)
    p.set_integrator(3)
    p.load(U0)
    t = 0.0
    while t < 1.0:
        dt = p.new_dt(cfl)
        if t + dt > 1.0:
            dt = 1.0 - t
        p.step(cfl, dt)
        t += dt
    a = act(mesh)
    U = p.current()
    return math.sqrt(sum(np.abs(U[a][0, n] - U0[a][0, n]).mean() ** 2 for n in range(5)))


@pytest.mark.parametrize("recon,key", [(RECON_WENOZ, "wenoz_rk3"), (RECON_PPMX, "ppmx_rk3")])
def test_linear_wave_converges_at_fourth_order_or_better(orc, recon, key):
    """'fourth-order convergence is observed for ... PPMX and WENOZ' on the 1-D linear wave.  SSPRK(3,3), dt scaled as
    dx^(4/3) (CFL 0.4 at N = 16) so that the third-order time error falls at the same fourth order; L1 error per
    doubling of N falls by >= 2^3.5 up to N = 64 (then round-off and the A^2 nonlinear terms of a 1e-6 wave
    approach).  No second-order scheme passes (PLM / PPM4: factor 4)."""
    e = {N: wave_error_rk3(orc, N, recon, 0.4 * (16.0 / N) ** (1.0 / 3.0)) for N in (16, 32, 64)}
    for N in (16, 32):
        assert e[N] / e[2 * N] >= 2 ** 3.5, (key, e)
    for N, ref in GOLD_C[key].items():                      # the stand-alone 1-D script's numbers (tests/golden/make_appendix_c.py)
        if int(N) in e:
            assert e[int(N)] == pytest.approx(ref, rel=2e-2), (key, N)
