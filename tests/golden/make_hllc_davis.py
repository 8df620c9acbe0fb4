#!/usr/bin/env python
"""Writes tests/golden/hllc_davis.json: worked HLLC fluxes for the round-2 wave-speed reading (Q2).

Stand-alone on purpose: plain Python floats, imports nothing from oracle/ or the CUDA package.  It evaluates the
HLLC flux by a DIFFERENT algebraic route than oracle/orc.cpp: Toro (2013) Eqs.(10.37)-(10.39), the star STATE
    U*_K = rho_K (S_K - u_K)/(S_K - S*) [1, S*, v_K, w_K, E_K/rho_K + (S* - u_K)(S* + p_K/(rho_K (S_K - u_K)))]
and F*_K = F_K + S_K (U*_K - U_K), with Davis's direct wave speeds, Eq.(10.48):
    S_L = min(u_L - c_L, u_R - c_R),  S_R = max(u_L + c_L, u_R + c_R),
and S* from Eq.(10.37).  (The oracle uses the flux form with the mean of the two star pressures; for exact
arithmetic the two coincide, so agreement is to rounding, a few 1e-16 relative.)

    python tests/golden/make_hllc_davis.py
"""
import json, math, os

def hllc_star_state_form(g, WL, WR):
    rL, uL, vL, wL, eL = WL
    rR, uR, vR, wR, eR = WR
    pL, pR = (g - 1) * eL, (g - 1) * eR
    cL, cR = math.sqrt(g * pL / rL), math.sqrt(g * pR / rR)
    SL, SR = min(uL - cL, uR - cR), max(uL + cL, uR + cR)
    Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR))
    def side(r, u, v, w, e, p, S):
        E = e + 0.5 * r * (u * u + v * v + w * w)
        U = [r, r * u, r * v, r * w, E]
        F = [r * u, r * u * u + p, r * u * v, r * u * w, (E + p) * u]
        f = r * (S - u) / (S - Ss)
        Us = [f, f * Ss, f * v, f * w, f * (E / r + (Ss - u) * (Ss + p / (r * (S - u))))]
        return U, F, Us
    UL, FL, UsL = side(rL, uL, vL, wL, eL, pL, SL)
    UR, FR, UsR = side(rR, uR, vR, wR, eR, pR, SR)
    if SL >= 0: return FL, (SL, Ss, SR)
    if SR <= 0: return FR, (SL, Ss, SR)
    if Ss >= 0: return [FL[n] + SL * (UsL[n] - UL[n]) for n in range(5)], (SL, Ss, SR)
    return [FR[n] + SR * (UsR[n] - UR[n]) for n in range(5)], (SL, Ss, SR)

CASES = [
    # SURVEY Appendix A.2 state pairs (Sod-like jump at rest; a general 3-D pair), now with Davis speeds
    (1.4, [1.0, 0.0, 0.0, 0.0, 2.5], [0.125, 0.0, 0.0, 0.0, 0.25]),
    (5.0 / 3.0, [1.0, 0.3, -0.2, 0.1, 1.5], [0.8, -0.1, 0.4, 0.25, 0.9]),
    # S* < 0 branch, with shear
    (5.0 / 3.0, [0.5, -0.2, 0.3, -0.1, 0.6], [1.5, 0.1, -0.4, 0.2, 2.4]),
    # the two halves of Toro's two-strong-shocks tube (his test 4 class): both estimates positive -> upwind F_L
    (1.4, [5.99924, 19.5975, 0.0, 0.0, 460.894 / 0.4], [5.99242, -6.19633, 0.0, 0.0, 46.0950 / 0.4]),
    # head-on Mach-3 collision with a density asymmetry (round-1 reading returned the upwind F_R here)
    (5.0 / 3.0, [1.0, 3.0 * math.sqrt(5.0 / 3.0), 0.2, 0.0, 1.5], [1.001, -3.0 * math.sqrt(5.0 / 3.0), -0.1, 0.3, 1.5]),
]

if __name__ == "__main__":
    out = {"source": "tests/golden/make_hllc_davis.py (stand-alone star-state form, Toro Eqs. 10.37-10.39, 10.48)",
           "cases": []}
    for g, WL, WR in CASES:
        F, S = hllc_star_state_form(g, WL, WR)
        out["cases"].append({"gamma": g, "WL": WL, "WR": WR, "F": F, "SL": S[0], "Sstar": S[1], "SR": S[2]})
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "hllc_davis.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)
