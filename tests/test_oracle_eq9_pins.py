"""Pins of the full Eq. (9) momentum parameterisation (C18b).  All CPU-only.

q/p = dSlope / F(tx, ty, dSlope), F = sum_i c_i(tx, ty) dSlope^i, c_i 2-D polynomials in the seed slopes with the terms
the field symmetries allow.  The coefficient table is an INPUT (momentum_fit.fit_qop_poly2d, a calibration on toys);
what is pinned here is the oracle's evaluation of it.
"""
import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

from paper_2402_14670_b200 import datagen as dg
from paper_2402_14670_b200 import momentum_fit as mf

AX, AY = 0.8, 1.5  # non-uniform toy field (datagen.toy_dtx)


@pytest.fixture(scope="module")
def table():
    return mf.fit_qop_poly2d(AX, AY)


def _field_cfg(n, seed, **kw):
    return dg.with_overrides(dg.single_track_config(n, seed=seed, sigma=0.0, smear=0.0), field_ax=AX, field_ay=AY, **kw)


def test_reduces_to_constants(oracle, geometry, params):
    """A table holding only the slope-independent terms of even i is the constant-coefficient mode, bit for bit."""
    b = dg.generate_config(0)
    c0, c2, c4 = geometry["qop_poly"][0], 0.37, -0.11
    t = [[0.0] * 10 for _ in range(5)]
    t[0][0], t[2][0], t[4][0] = c0, c2, c4
    a = oracle.run(dict(geometry, qop_poly=[c0, 0.0, c2, 0.0, c4]), params, b)
    c = oracle.run(dict(geometry, qop_mode=1, qop_poly2d=t), params, b)
    assert a.n_tracks == c.n_tracks > 150
    assert np.array_equal(a.state.view(np.uint32), c.state.view(np.uint32))


@pytest.mark.parametrize("real,tol", [("f64", 1e-6), ("f32", 2e-5)])
def test_against_polyval2d(oracle, geometry, params, table, real, tol):
    """q/p from the table equals dSlope / F with F evaluated by numpy.polynomial (polyval2d per power of dSlope);
    dSlope itself is recovered from a second oracle run with a constant F = 1 (then q/p = dSlope)."""
    b = dg.generate_config(1, n_events=30)
    r1 = oracle.run(dict(geometry, qop_poly=[1.0, 0.0, 0.0, 0.0, 0.0]), params, b, real=real)
    r2 = oracle.run(dict(geometry, qop_mode=1, qop_poly2d=table), params, b, real=real)
    assert np.array_equal(r1.seed_idx, r2.seed_idx) and np.array_equal(r1.hit_idx, r2.hit_idx)
    ds = r1.state[:, 4].astype(np.float64)
    tx = b.seed_tx[r1.seed_idx].astype(np.float64)
    ty = b.seed_ty[r1.seed_idx].astype(np.float64)
    tab32 = np.asarray(np.float32(table), np.float64)   # the oracle receives float32 coefficients
    F = np.zeros_like(ds)
    for i in range(5):
        cm = np.zeros((7, 7))
        for j, (k, m) in enumerate(mf.terms_of(i)):
            cm[k, m] = tab32[i][j]
        F += npoly.polyval2d(tx, ty, cm) * ds ** i
    want = ds / F
    assert np.max(np.abs(r2.state[:, 4] / want - 1.0)) < tol
    # the slope-dependent terms matter on this sample: the constant mode differs by several per cent
    r0 = oracle.run(geometry, params, b, real=real)
    assert np.max(np.abs(r0.state[:, 4] / r2.state[:, 4] - 1.0)) > 0.02


@pytest.mark.parametrize("real", ["f64", "f32"])
def test_truth_momentum_in_nonuniform_field(oracle, geometry, params, table, real):
    """Noise-free single tracks in the non-uniform toy field: with the calibrated table q/p equals the truth to the
    accuracy of the parameterisation (< 0.1 %); with the constant F of the uniform field it is off by up to 20-30 %."""
    b = dg.generate(_field_cfg(500, 41))
    G1 = dict(geometry, qop_mode=1, qop_poly2d=table)
    r = oracle.run(G1, params, b, real=real)
    tid = b.seed_track[r.seed_idx]
    full = np.bincount(b.hit_track[b.hit_track >= 0], minlength=b.n_tracks) == 12
    sel = full[tid] & (r.n_hits == 12)
    assert sel.sum() > 250
    rel = np.abs(r.state[sel, 4] / b.trk_qop[tid[sel]] - 1.0)
    assert rel.max() < 1e-3, rel.max()
    r0 = oracle.run(geometry, params, b, real=real)
    tid0 = b.seed_track[r0.seed_idx]
    rel0 = np.abs(r0.state[:, 4] / b.trk_qop[tid0] - 1.0)
    assert rel0.max() > 0.1 and np.median(rel0) > 10 * np.median(rel)


def test_twin_with_table(oracle, geometry, params, table):
    from oracle import brute_twin
    b = dg.generate(dg.with_overrides(dg.CONFIGS[0], field_ax=AX, field_ay=AY, seed=1234))
    G1 = dict(geometry, qop_mode=1, qop_poly2d=table)
    r = oracle.run(G1, params, b, real="f64")
    tw = brute_twin.run(G1, params, b)
    assert tw.n_tracks == r.n_tracks > 100
    assert np.array_equal(tw.hit_idx, r.hit_idx)
    assert np.max(np.abs(tw.state[:, 4] / r.state[:, 4] - 1.0)) < 1e-6


def test_mirror_symmetry(oracle, geometry, params, table):
    """x -> -x with the magnet polarity and the stereo angles flipped maps every track onto its mirror image: same hits (mirrored indices),
    x, tx and q/p change sign, y, ty and Q do not.  Fails if an odd term sits in an even coefficient (or the reverse),
    or if any left/right asymmetry in windows, seeding or fit has the wrong sign."""
    b = dg.generate(dg.with_overrides(dg.CONFIGS[0], field_ax=AX, field_ay=AY, seed=1235))
    G1 = dict(geometry, qop_mode=1, qop_poly2d=table)
    seg = b.seg_offsets.astype(np.int64)
    hx = b.hit_x.copy()
    mirror_of = np.empty(b.n_hits, np.int64)
    for s in range(seg.shape[0] - 1):
        a, e = seg[s], seg[s + 1]
        hx[a:e] = -b.hit_x[a:e][::-1]
        mirror_of[a:e] = np.arange(e - 1, a - 1, -1)
    bm = dg.Batch(**{**b.__dict__, "hit_x": hx, "seed_x": -b.seed_x, "seed_tx": -b.seed_tx, "seed_qop": -b.seed_qop})
    r = oracle.run(G1, params, b, real="f64")
    # the mirror image of a +5 degree stereo layer is a -5 degree one: s = x + y tan(alpha) -> -s needs tan(alpha) -> -tan(alpha)
    Gm = dict(G1, polarity=-geometry["polarity"], tan_alpha=[-t for t in geometry["tan_alpha"]])
    rm = oracle.run(Gm, params, bm, real="f64")
    assert r.n_tracks == rm.n_tracks > 100 and np.array_equal(r.seed_idx, rm.seed_idx)
    want = np.where(r.hit_idx >= 0, mirror_of[np.maximum(r.hit_idx, 0)], -1)
    assert np.array_equal(rm.hit_idx, want)
    sgn = np.array([-1.0, 1.0, -1.0, 1.0, -1.0])
    assert np.max(np.abs(rm.state * sgn - r.state)[:, :2]) < 1e-3
    assert np.max(np.abs(rm.state * sgn - r.state)[:, 2:4]) < 1e-7
    assert np.max(np.abs(rm.state[:, 4] * -1.0 / r.state[:, 4] - 1.0)) < 1e-6
    assert np.max(np.abs(rm.quality - r.quality)) < 1e-6
