"""Helpers shared by the GPU parity tests: the difference metric of DESIGN.md, conserved
totals, and lock-step / free-running drivers that advance the oracle and the CUDA path side by side."""
from __future__ import annotations

import math
import os

import numpy as np
import torch

from paper_2409_16053_b200 import inputs as I

NTHREADS = max(1, os.cpu_count() or 1)     # oracle OpenMP threads: bit-identical to 1 thread (orc.h)

MARGINS = []                               # one line per parity run; tests/conftest.py prints them in the summary


def report(line: str) -> None:
    """Record how far inside its bar a parity run ended (shown after the dots of `pytest -q`)."""
    MARGINS.append(line)
    print(line)


def active(mesh):
    g = mesh.ng
    return (slice(None), slice(None), slice(g, -g), slice(g, -g), slice(g, -g))


def q14(U_gpu: np.ndarray, U_orc: np.ndarray, gamma: float) -> float:
    """max over cells of max(|d rho|/rho, |d(rho v_d)|/(rho(|v|+c_s)), |dE|/E); denominators from the oracle."""
    rho, m, E = U_orc[:, 0], U_orc[:, 1:4], U_orc[:, 4]
    ke = 0.5 * (m ** 2).sum(1) / rho
    p = (gamma - 1.0) * (E - ke)
    cs = np.sqrt(gamma * np.maximum(p, 0.0) / rho)
    vmag = np.sqrt((m ** 2).sum(1)) / rho
    d = np.abs(U_gpu - U_orc)
    e = np.maximum(d[:, 0] / rho, d[:, 4] / E)
    e = np.maximum(e, d[:, 1:4].max(1) / (rho * (vmag + cs)))
    return float(e.max())


def totals(mesh, U: np.ndarray):
    """Volume-weighted totals of the 5 conserved variables over active cells (exact summation)."""
    a = active(mesh)
    out = np.zeros(5)
    for n in range(5):
        out[n] = math.fsum(float(np.sum(U[m][a[1:]][n], dtype=np.longdouble)) * mesh.cell_volume(m) for m in range(mesh.nmb))
    return out


def momentum_norm(mesh, U: np.ndarray, gamma: float) -> float:
    a = active(mesh)
    s = 0.0
    for m in range(mesh.nmb):
        u = U[m][a[1:]]
        rho, mom, E = u[0], u[1:4], u[4]
        p = (gamma - 1.0) * (E - 0.5 * (mom ** 2).sum(0) / rho)
        s += float(np.sum(np.sqrt((mom ** 2).sum(0)) + rho * np.sqrt(gamma * p / rho))) * mesh.cell_volume(m)
    return s


def make_pair(orc, ak, w: I.Workload, U0: torch.Tensor, variant=0, rsolver=0):
    po = orc.OrcPack(w.mesh, w.gamma, w.recon, rsolver=rsolver, threads=NTHREADS)
    po.load(U0.numpy())
    pg = ak.Pack(w.mesh, w.gamma, w.recon, rsolver=rsolver, variant=variant)
    pg.load(U0)
    return po, pg


def gpu_state(pg) -> np.ndarray:
    return pg.current().cpu().numpy()
