#!/usr/bin/env python
"""Writes tests/golden/appendix_c.json: L1 errors of a 1-D sound wave after one period (paper P:130, Fig.1 left).

Stand-alone 1-D numpy evaluation of the scheme of DESIGN.md section 2 (PLM van Leer / PPM4-CW84 on W = (rho, v, u_g),
HLLC with Davis's wave speeds -- the round-2 reading Q2 --, SSPRK(2,2), CFL rule of Eq.(3)); it imports nothing from
oracle/ or from the CUDA package.  Vectorised over the line, so it is a second, independently written implementation
of the same formulas: the 3-D oracle on an N x 4 x 4 box must reproduce these errors (tests/test_oracle_scheme.py).
The paper prints no error values, only the convergence order.

    python tests/golden/make_appendix_c.py
"""
import json, math, os
import numpy as np

G = 5.0 / 3.0

def c2p(U):
    rho = U[0]; v = U[1] / rho
    return np.array([rho, v, U[2] - 0.5 * rho * v * v])          # (rho, v, u_g), 1-D: one velocity

def plm(q):
    dL = q - np.roll(q, 1); dR = np.roll(q, -1) - q
    prod = dL * dR
    with np.errstate(divide="ignore", invalid="ignore"):
        h = np.where(prod > 0.0, prod / (dL + dR), 0.0)
    return q - h, q + h

def ppm4(q):
    qm1, qp1, qp2 = np.roll(q, 1), np.roll(q, -1), np.roll(q, -2)
    f = (7.0 * (q + qp1) - (qm1 + qp2)) / 12.0                   # interface i+1/2
    f = np.maximum(np.minimum(q, qp1), np.minimum(f, np.maximum(q, qp1)))
    aR, aL = f.copy(), np.roll(f, 1)
    flat = (aR - q) * (q - aL) <= 0.0
    d = aR - aL; mu = q - 0.5 * (aL + aR)
    c1 = d * mu > d * d / 6.0
    c2 = -d * d / 6.0 > d * mu
    nL = np.where(c1, 3.0 * q - 2.0 * aR, aL)
    nR = np.where(~c1 & c2, 3.0 * q - 2.0 * aL, aR)
    return np.where(flat, q, nL), np.where(flat, q, nR)

def wenoz(q):
    """WENO-Z, Q29: (q-, q+) of every cell from q[i-2..i+2] (periodic)."""
    def upper(a, b, c, d, e):
        d1, d2, d3, d4 = b - a, c - b, d - c, e - d
        P0, P1, P2 = 5 * d2 - 2 * d1, 2 * d3 + d2, 4 * d3 - d4
        b0 = 13 / 12 * (d2 - d1) ** 2 + 0.25 * (3 * d2 - d1) ** 2
        b1 = 13 / 12 * (d3 - d2) ** 2 + 0.25 * (d2 + d3) ** 2
        b2 = 13 / 12 * (d4 - d3) ** 2 + 0.25 * (d4 - 3 * d3) ** 2
        tau = np.abs(b0 - b2)
        a0, a1, a2 = (w * (1 + (tau / (b + 1e-40)) ** 2) for w, b in ((0.1, b0), (0.6, b1), (0.3, b2)))
        return c + (a0 * P0 + (a1 * P1 + a2 * P2)) / (6 * (a0 + (a1 + a2)))
    m2, m1, p1, p2 = np.roll(q, 2), np.roll(q, 1), np.roll(q, -1), np.roll(q, -2)
    return upper(p2, p1, q, m1, m2), upper(m2, m1, q, p1, p2)

def ppmx(q):
    """PPMX, Q30: fourth-order interfaces + Colella-Sekora / McCorquodale-Colella limiters (C = 5/4)."""
    C = 1.25
    m2, m1, p1, p2 = np.roll(q, 2), np.roll(q, 1), np.roll(q, -1), np.roll(q, -2)
    def lim3(dc, dl, dr):
        pos = (dc > 0) & (dl > 0) & (dr > 0); neg = (dc < 0) & (dl < 0) & (dr < 0)
        return np.where(pos, np.minimum(dc, C * np.minimum(dl, dr)), np.where(neg, -np.minimum(-dc, C * np.minimum(-dl, -dr)), 0.0))
    v = (7.0 * (q + p1) - (m1 + p2)) / 12.0                        # interface i+1/2
    bad = (v - q) * (p1 - v) < 0.0
    D = lim3(3.0 * ((q + p1) - 2.0 * v), (m1 + p1) - 2.0 * q, (q + p2) - 2.0 * p1)
    v = np.where(bad, 0.5 * (q + p1) - D / 6.0, v)
    aR, aL = v, np.roll(v, 1)
    dm, dp = q - aL, aR - q
    ext = (dm * dp <= 0.0) | ((p1 - q) * (q - m1) <= 0.0)
    df = 6.0 * ((aL + aR) - 2.0 * q)
    d1, d2, d3 = (m2 + q) - 2.0 * m1, (m1 + p1) - 2.0 * q, (q + p2) - 2.0 * p1
    pos = (df > 0) & (d1 > 0) & (d2 > 0) & (d3 > 0); neg = (df < 0) & (d1 < 0) & (d2 < 0) & (d3 < 0)
    Dl = np.where(pos, np.minimum(df, C * np.minimum(d1, np.minimum(d2, d3))),
                  np.where(neg, -np.minimum(-df, C * np.minimum(-d1, np.minimum(-d2, -d3))), 0.0))
    with np.errstate(divide="ignore", invalid="ignore"):
        rho = np.where(df != 0.0, Dl / df, 0.0)
    use = rho <= 1.0 - 1e-12
    eL = np.where(use, q - rho * dm, aL); eR = np.where(use, q + rho * dp, aR)
    mL = np.where(np.abs(dm) >= 2.0 * np.abs(dp), q - 2.0 * dp, aL)
    mR = np.where(np.abs(dp) >= 2.0 * np.abs(dm), q + 2.0 * dm, aR)
    return np.where(ext, eL, mL), np.where(ext, eR, mR)

def hllc(WL, WR):
    rL, uL, eL = WL; rR, uR, eR = WR
    pL, pR = (G - 1) * eL, (G - 1) * eR
    cL, cR = np.sqrt(G * pL / rL), np.sqrt(G * pR / rR)
    SL, SR = np.minimum(uL - cL, uR - cR), np.maximum(uL + cL, uR + cR)
    mL, mR = rL * (uL - SL), rR * (SR - uR)
    Ss = ((pL - pR) + (mL * uL + mR * uR)) / (mL + mR)
    ps = np.maximum(0.5 * ((pL + rL * (SL - uL) * (Ss - uL)) + (pR + rR * (SR - uR) * (Ss - uR))), 0.0)
    left = Ss >= 0.0
    rK, uK, eK, pK = (np.where(left, a, b) for a, b in ((rL, rR), (uL, uR), (eL, eR), (pL, pR)))
    b = np.where(left, np.minimum(SL, 0.0), np.maximum(SR, 0.0))
    EK = eK + 0.5 * rK * uK * uK
    UK = np.array([rK, rK * uK, EK]); FK = np.array([rK * uK, rK * uK * uK + pK, (EK + pK) * uK])
    D = np.array([np.zeros_like(Ss), np.ones_like(Ss), Ss])
    return (Ss * (FK - b * UK) - b * ps * D) / (Ss - b)

def rhs(U, recon):
    W = c2p(U)
    qm, qp = zip(*(recon(W[n]) for n in range(3)))
    WL = np.array([np.roll(q, 1) for q in qp])                   # q+ of cell i-1 at face i-1/2
    WR = np.array(qm)
    F = hllc(WL, WR)                                             # flux at the lower face of cell i
    return -(np.roll(F, -1, axis=1) - F)

def run(N, recon, cfl, amp=1e-6, rk3=False):
    x = (np.arange(N) + 0.5) / N
    s = np.sin(2 * math.pi * x)
    rho, v, P = 1.0 + amp * s, amp * s, 1.0 / G + amp * s
    U0 = np.array([rho, rho * v, P / (G - 1) + 0.5 * rho * v * v])
    U, t, dx = U0.copy(), 0.0, 1.0 / N
    while t < 1.0:
        W = c2p(U)
        dt = cfl * np.min(dx / (np.abs(W[1]) + np.sqrt(G * ((G - 1) * W[2]) / W[0])))
        if t + dt > 1.0: dt = 1.0 - t
        U1 = U + dt / dx * rhs(U, recon)
        if rk3:                                                  # SSPRK(3,3), Q27
            U2 = 0.75 * U + 0.25 * (U1 + dt / dx * rhs(U1, recon))
            U = (1.0 / 3.0) * U + (2.0 / 3.0) * (U2 + dt / dx * rhs(U2, recon))
        else:
            U = 0.5 * U + 0.5 * (U1 + dt / dx * rhs(U1, recon))
        t += dt
    return math.sqrt(sum(np.abs(U[n] - U0[n]).mean() ** 2 for n in range(3)))

if __name__ == "__main__":
    out = {"source": "tests/golden/make_appendix_c.py (stand-alone 1-D numpy scheme; Davis wave speeds, DESIGN.md Q2); "
                     "sound wave A=1e-6, gamma=5/3, one period",
           "plm_cfl0.3": {str(N): run(N, plm, 0.3) for N in (16, 32, 64, 128, 256)},
           "ppm4_cfl0.1": {str(N): run(N, ppm4, 0.1) for N in (32, 64, 128)},
           # P:130 "fourth-order convergence ... for PPMX and WENOZ": SSPRK(3,3), CFL = 0.4 (16/N)^(1/3) so that the
           # time error falls at fourth order too
           "wenoz_rk3": {str(N): run(N, wenoz, 0.4 * (16.0 / N) ** (1.0 / 3.0), rk3=True) for N in (16, 32, 64, 128)},
           "ppmx_rk3": {str(N): run(N, ppmx, 0.4 * (16.0 / N) ** (1.0 / 3.0), rk3=True) for N in (16, 32, 64, 128)}}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "appendix_c.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out, indent=1))
