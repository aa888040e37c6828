"""Calibration of the full Eq. (9) momentum parameterisation on toy tracks.

    q/p = dSlope / F(tx, ty, dSlope),   F = sum_{i=0..4} c_i(tx, ty) dSlope^i,
    c_i(tx, ty) = sum_{k,m} c_i^{km} tx^k ty^m,  k + m <= 6,

"a set of toy tracks ... equi-populate the acceptance of tx, ty, and have a flat q/p spectrum"; "only even/odd
combinations of m, k" that respect the field symmetries are kept.  For a dipole B_y: F is even in ty, and
mirroring x flips tx, dSlope and q/p together, so c_i is even in tx for even i and odd in tx for odd i.  That leaves
10 terms for even i and 6 for odd i, in the order of `EVEN_TERMS` / `ODD_TERMS` (the layout of `lf_geometry.qop_poly2d`).

This module is an INPUT generator (a calibration the detector would ship with), like `datagen`: it holds none of the
algorithm's steps and serves the oracle and the CUDA path with the same coefficient table.  The paper fits per-bin
polynomials first and the 2-D polynomials second; here all 42 coefficients come from ONE linear least-squares problem
(F * q/p = dSlope is linear in them), which needs no binning.
"""
from __future__ import annotations

from typing import List

import numpy as np

from . import datagen as dg

EVEN_TERMS = ((0, 0), (2, 0), (0, 2), (4, 0), (2, 2), (0, 4), (6, 0), (4, 2), (2, 4), (0, 6))  # (k, m): tx^k ty^m
ODD_TERMS = ((1, 0), (3, 0), (1, 2), (5, 0), (3, 2), (1, 4))


def terms_of(i: int):
    return EVEN_TERMS if i % 2 == 0 else ODD_TERMS


def toy_dslope(tx, ty, qop, field_ax: float, field_ay: float):
    """What the algorithm measures on a perfect track: slope at z_ref (incl. the TOY quadratic term) minus the seed slope."""
    dtx = dg.toy_dtx(tx, ty, qop, field_ax, field_ay)
    return dg.toy_tx_at(tx + dtx, dtx, dg.TOY_Z_REF) - tx


def fit_qop_poly2d(field_ax: float, field_ay: float, n_toys: int = 200_000, seed: int = 7, p_min: float = 1.5) -> List[List[float]]:
    """Coefficients c_i^{km} as a 5 x 10 table (unused slots 0), from toys flat in tx, ty and q/p."""
    rng = np.random.Generator(np.random.PCG64(seed))
    tx = rng.uniform(-0.25, 0.25, n_toys)
    ty = rng.uniform(-0.2, 0.2, n_toys)
    qop = rng.uniform(-1.0 / p_min, 1.0 / p_min, n_toys)
    qop = np.where(np.abs(qop) < 1e-3, 1e-3, qop)
    ds = toy_dslope(tx, ty, qop, field_ax, field_ay)
    # keep the toys that stay inside the acceptance at the last layer (the tracks the algorithm can find)
    dtx = dg.toy_dtx(tx, ty, qop, field_ax, field_ay)
    x_last = dg.toy_x_at(tx * dg.TOY_Z_MAG, tx + dtx, dtx, dg.TOY_Z[-1])
    keep = np.abs(x_last) < dg.TOY_X_HALF
    tx, ty, qop, ds = tx[keep], ty[keep], qop[keep], ds[keep]
    # relative residuals: F * (q/p) / dSlope = 1, every toy with the same weight whatever its momentum
    cols, index = [], []
    for i in range(5):
        for j, (k, m) in enumerate(terms_of(i)):
            cols.append(tx ** k * ty ** m * ds ** i * (qop / ds))
            index.append((i, j))
    A = np.stack(cols, axis=1)
    scale = np.abs(A).max(axis=0)
    sol, *_ = np.linalg.lstsq(A / scale, np.ones(ds.shape[0]), rcond=None)
    sol = sol / scale
    table = [[0.0] * 10 for _ in range(5)]
    for (i, j), c in zip(index, sol):
        table[i][j] = float(c)
    return table


def evaluate_F(table, tx, ty, ds):
    """F(tx, ty, dSlope) in float64 from a coefficient table (for tests and studies)."""
    F = 0.0
    for i in range(5):
        c = 0.0
        for j, (k, m) in enumerate(terms_of(i)):
            c = c + table[i][j] * tx ** k * ty ** m
        F = F + c * ds ** i
    return F
