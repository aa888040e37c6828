"""Pins of the oracle's no-UT mode (N1..N9).  All CPU-only.

Same devices as test_oracle_pins.py: the constants the paper prints (Table 3 second column, Table 5),
the brute-force twin, the generator's truth on noise-free single tracks, special cases of Eq. (7)/(8)
(zero slopes, window overlap, numpy.searchsorted), invariants, the fp64 build and statistical sanity.
"""
import os

import numpy as np
import pytest

from paper_2402_14670_b200 import datagen as dg
from paper_2402_14670_b200 import truth

HERE = os.path.dirname(os.path.abspath(__file__))
NL = 12
X_LAYERS = [0, 3, 4, 7, 8, 11]


@pytest.fixture(scope="module")
def nparams():
    return dg.no_ut_params()


def _assumed_p(b, P):
    """PAPER.md:289 in float64: the tighter of p_min and pT_min / sin(theta)."""
    s2 = b.seed_tx.astype(np.float64) ** 2 + b.seed_ty.astype(np.float64) ** 2
    with np.errstate(divide="ignore"):
        return np.maximum(P["velo_p_min"], P["velo_pt_min"] * np.sqrt(1.0 + s2) / np.sqrt(s2))


def _eq7(tx, ty, p, c):
    """Eq. (7) as printed, float64."""
    return (c[0] + tx * (c[1] + c[2] * tx) + ty ** 2 * (c[3] + tx * (c[4] + c[5] * tx)) + (c[6] * tx + c[7] / p) / p) / p


def test_paper_constants_noUT_fixture(nparams):
    for line in open(os.path.join(HERE, "golden", "paper_constants_noUT.txt")):
        line = line.split("#")[0].split()
        if len(line) != 2:
            continue
        k, v = line[0], float(line[1])
        if k.startswith("xtol_poly_"):
            assert nparams["xtol_poly"][int(k.split("_")[-1])] == v
        else:
            assert nparams[k] == v, k
    assert nparams["mode"] == 1
    # no momentum, no charge: the same-bend filter cannot exist; the tolerance at the magnet is a constant
    assert nparams["p_same_bend"] == 0.0 and nparams["mag_tol_inv_p"] == 0.0 and nparams["mag_tol_tx"] == 0.0


# ------------------------------------------------------------------------------------------------ twin
def _assert_twin_equal(oracle, G, P, b):
    from oracle import brute_twin
    r = oracle.run(G, P, b, real="f64", debug=True)
    tw = brute_twin.run(G, P, b)
    assert r.debug.win_count.shape[0] == 2 * b.n_seeds  # one row per (seed, window side)
    assert np.array_equal(tw.win_count, r.debug.win_count)
    m = tw.win_count > 0
    assert np.array_equal(tw.win_first[m], r.debug.win_first[m])
    assert len(tw.triplets) == 2 * b.n_seeds
    for row, trips in enumerate(tw.triplets):
        assert len(trips) == r.debug.n_triplets[row]
        for k, (chi2, s, i0, i2, i1) in enumerate(trips):
            assert tuple(r.debug.trip_hits[row, k]) == (i0, i1, i2) and r.debug.trip_set[row, k] == s
            assert abs(r.debug.trip_chi2[row, k] - chi2) <= 1e-5 * max(1.0, chi2)
    assert tw.n_tracks == r.n_tracks
    assert np.array_equal(tw.seed_idx, r.seed_idx)
    assert np.array_equal(tw.hit_idx, r.hit_idx)
    assert np.array_equal(tw.n_hits, r.n_hits)
    assert np.array_equal(tw.event_offsets, r.event_offsets)
    if r.n_tracks:
        assert np.max(np.abs(tw.state[:, :2] - r.state[:, :2])) < 3e-4
        assert np.max(np.abs(tw.state[:, 2:4] - r.state[:, 2:4])) < 1e-7
        assert np.max(np.abs(tw.state[:, 4] / r.state[:, 4] - 1)) < 1e-6
        assert np.max(np.abs(tw.quality - r.quality)) < 1e-6
    return r


def test_twin_config0_noUT(oracle, geometry, nparams):
    r = _assert_twin_equal(oracle, geometry, nparams, dg.generate_config(0))
    assert r.n_tracks > 100


def test_twin_dense_event_caps_bind_noUT(oracle, geometry, nparams):
    """Dense tiny events with a small window cap and few triplets: both caps bind on both window sides."""
    cfg = dg.GenConfig("dense", 2, 79, true_fixed=25, fake_mean=5.0, noise_fixed=450, p_min=4.0)
    b = dg.generate(cfg)
    P = dict(nparams, n_window=17, n_triplets=3, T_triplet=8.0, T_x=2.0, x_overlap=40.0, mag_tol_base=25.0, mag_tol_max=25.0)
    r = _assert_twin_equal(oracle, geometry, P, b)
    assert (r.debug.win_count >= 16).mean() > 0.3
    assert (r.debug.n_triplets == 3).sum() > 5
    # the paper's caps (64 hits, 20 triplets) on the same events, and a non-zero dRatio
    _assert_twin_equal(oracle, geometry, nparams, b)
    _assert_twin_equal(oracle, dict(geometry, d_ratio=-2.0e-5), nparams, b)


# ------------------------------------------------------------------------------------------------ truth
@pytest.mark.parametrize("real,tol_x,tol_t,tol_q", [("f64", 2.5e-4, 1e-6, 1e-5), ("f32", 1.5e-3, 3e-6, 1e-4)])
def test_truth_exact_hits_noise_free_noUT(oracle, geometry, nparams, real, tol_x, tol_t, tol_q):
    """sigma = 0, one particle per event, momentum above the assumed minimum: all 12 true hits, Q ~ 0,
    charge and momentum from the pT-kick equal the truth; the seed's q/p is never read."""
    b = dg.generate(dg.single_track_config(500, seed=21, sigma=0.0, smear=0.0, p_min=5.0))
    b.seed_qop = np.full_like(b.seed_qop, np.nan)  # VELO tracks carry no momentum estimate
    r = oracle.run(geometry, nparams, b, real=real, debug=True)
    cnt = np.bincount(b.hit_track[b.hit_track >= 0], minlength=b.n_tracks)
    p_true = 1.0 / np.abs(b.trk_qop)
    inside = (cnt == NL) & (p_true[:] > 1.3 * _assumed_p(b, nparams)[np.argsort(b.seed_track)])
    tid = b.seed_track[r.seed_idx]
    found = np.zeros(b.n_tracks, bool)
    found[tid] = True
    assert inside.sum() > 200
    assert np.all(found[inside]), "a fully measured noise-free track above the momentum threshold was not found"
    sel = inside[tid]
    assert np.all(b.hit_track[r.hit_idx[sel]] == tid[sel][:, None]) and np.all(r.n_hits[sel] == NL)
    assert np.max(r.quality[sel]) < (1e-7 if real == "f64" else 1e-5)
    t = tid[sel]
    st = r.state[sel].astype(np.float64)
    zs = geometry["z_state"]
    x_mag = b.trk_x[t] + b.trk_tx[t] * (dg.TOY_Z_MAG - dg.TOY_Z_SEED)
    dtx = dg.TOY_KICK * b.trk_qop[t]
    assert np.max(np.abs(st[:, 0] - dg.toy_x_at(x_mag, b.trk_tx[t] + dtx, dtx, zs))) < tol_x
    assert np.max(np.abs(st[:, 2] - dg.toy_tx_at(b.trk_tx[t] + dtx, dtx, zs))) < tol_t
    assert np.max(np.abs(st[:, 4] / b.trk_qop[t] - 1.0)) < tol_q
    assert np.all(np.sign(st[:, 4]) == np.sign(b.trk_qop[t]))
    # Eq. (8): with kick > 0 a positive particle bends to +x, i.e. it is found in the RIGHT window (side 1)
    cq = r.debug.cand_quality.reshape(b.n_seeds, 2, -1)
    ok = np.where(cq >= 0, cq, np.inf).min(2)           # best accepted Q per (seed, side)
    far = sel & (np.abs(dg.TOY_KICK * b.trk_qop[tid]) * 2600.0 > 3 * nparams["x_overlap"])  # outside the overlap at layer 0
    side_found = np.argmin(ok[r.seed_idx], axis=1)
    assert np.array_equal(side_found[far], (b.trk_qop[tid][far] > 0).astype(int))
    assert np.all(np.isinf(ok[r.seed_idx][far, 1 - side_found[far]]))


def test_zero_slope_seed_has_only_the_overlap(oracle, geometry, nparams):
    """tx = ty = 0: sin(theta) = 0, the pT threshold gives infinite momentum, x_tol = 0 (Eq. 7): every
    x window is [x, x + overlap] on the LEFT side and [x - overlap, x] on the RIGHT (Eq. 8)."""
    b = dg.generate(dg.GenConfig("z", 3, 31, true_fixed=4, noise_fixed=2500))
    b.seed_tx[:] = 0.0
    b.seed_ty[:] = 0.0
    d = oracle.run(geometry, dict(nparams, n_window=1 << 20), b, debug=True).debug
    ev = np.searchsorted(b.seed_offsets, np.arange(b.n_seeds), side="right") - 1
    n_nonempty = 0
    for si in range(b.n_seeds):
        for l in X_LAYERS:
            s0, s1 = b.seg_offsets[ev[si] * 24 + l * 2 + 1], b.seg_offsets[ev[si] * 24 + l * 2 + 2]  # ty >= 0: zone 1
            seg = b.hit_x[s0:s1].astype(np.float64)
            x = float(b.seed_x[si])
            for side, (lo, hi) in enumerate(((x, x + 5.0), (x - 5.0, x))):
                want = np.nonzero((seg >= lo) & (seg <= hi))[0]
                assert d.win_count[2 * si + side, l] == want.size
                if want.size:
                    n_nonempty += 1
                    assert d.win_first[2 * si + side, l] == s0 + want[0]
    assert n_nonempty > 20


def test_windows_eq7_eq8_against_searchsorted(oracle, geometry, nparams):
    """Uncapped windows: edges = numpy.searchsorted of Eq. (8) about the straight line, x_tol from Eq. (7)
    evaluated independently in float64; the two sides overlap by exactly the hits within +-x_overlap."""
    b = dg.generate_config(1, n_events=6)
    P = dict(nparams, n_window=1 << 20)
    d = oracle.run(geometry, P, b, debug=True).debug
    z = np.asarray(geometry["z"], np.float64)
    tana = np.asarray(geometry["tan_alpha"], np.float64)
    ev = np.searchsorted(b.seed_offsets, np.arange(b.n_seeds), side="right") - 1
    zone = (b.seed_ty >= 0).astype(np.int64)
    pa = _assumed_p(b, P)
    checked = 0
    for si in range(0, b.n_seeds, 5):
        x, y, tx, ty = (float(v[si]) for v in (b.seed_x, b.seed_y, b.seed_tx, b.seed_ty))
        x_tol = _eq7(tx, ty, pa[si], P["xtol_poly"])
        for l in (0, 5, 11):
            dz = z[l] - geometry["z_seed"]
            ctr = x + tx * dz + (y + ty * dz) * tana[l]
            tol = P["uv_half_width"] if tana[l] != 0 else x_tol
            s0, s1 = b.seg_offsets[ev[si] * 24 + l * 2 + zone[si]], b.seg_offsets[ev[si] * 24 + l * 2 + zone[si] + 1]
            seg = b.hit_x[s0:s1].astype(np.float64)
            edges = np.array([ctr - tol, ctr + 5.0, ctr - 5.0, ctr + tol])
            if seg.size and np.min(np.abs(seg[:, None] - edges[None, :])) < 2e-3:
                continue  # a hit within fp32 rounding of an edge: the float64 evaluation cannot decide it
            fl, ll = s0 + np.searchsorted(seg, edges[0], "left"), s0 + np.searchsorted(seg, edges[1], "right")
            fr, lr = s0 + np.searchsorted(seg, edges[2], "left"), s0 + np.searchsorted(seg, edges[3], "right")
            L, R = 2 * si, 2 * si + 1
            assert d.win_count[L, l] == ll - fl and d.win_count[R, l] == lr - fr
            if ll > fl:
                assert d.win_first[L, l] == fl
            if lr > fr:
                assert d.win_first[R, l] == fr
            assert ll - fr == np.count_nonzero(np.abs(seg - ctr) <= 5.0)
            checked += 1
    assert checked > 200


# ------------------------------------------------------------------------------------------------ invariants
def _check_invariants(b, P, r):
    n = r.n_tracks
    assert r.hit_idx.shape == (n, NL)
    assert np.all(np.diff(r.seed_idx) > 0), "tracks must be in seed order, at most one per seed"
    ev_of_seed = np.searchsorted(b.seed_offsets, r.seed_idx, side="right") - 1
    assert np.array_equal(np.bincount(ev_of_seed, minlength=b.n_events), np.diff(r.event_offsets.astype(np.int64)))
    assert np.array_equal((r.hit_idx >= 0).sum(1), r.n_hits) and np.all(r.n_hits >= P["min_hits"])
    for st in range(3):
        assert np.all((r.hit_idx[:, 4 * st + 1] >= 0) | (r.hit_idx[:, 4 * st + 2] >= 0))
    assert np.all(r.quality < P["T_Q"]) and np.all(r.quality >= 0)
    assert np.all(np.abs(r.state[:, 3] - b.seed_ty[r.seed_idx]) < P["T_ty"])
    assert np.all(np.isfinite(r.state))
    d = r.debug
    assert np.all(d.win_count <= P["n_window"]) and np.all(d.n_triplets <= P["n_triplets"])
    c = d.trip_chi2
    assert np.all(c[c >= 0] < P["T_triplet"])
    for k in range(P["n_triplets"] - 1):
        both = d.n_triplets > k + 1
        assert np.all(c[both, k] <= c[both, k + 1])
    # every hit of a track lies in ONE side's windows of its seed (a candidate never mixes the two sides)
    have = r.hit_idx >= 0
    inside = []
    for side in (0, 1):
        wf, wc = d.win_first[2 * r.seed_idx + side], d.win_count[2 * r.seed_idx + side]
        inside.append(np.all(((r.hit_idx >= wf) & (r.hit_idx < wf + wc)) | ~have, axis=1))
    assert np.all(inside[0] | inside[1])


@pytest.mark.parametrize("cid,n_events", [(0, None), (1, 40), (4, 12)])
def test_invariants_noUT(oracle, geometry, nparams, cid, n_events):
    b = dg.generate_config(cid, n_events=n_events)
    r = oracle.run(geometry, nparams, b, debug=True, threads=4)
    _check_invariants(b, nparams, r)
    assert r.n_tracks > 0


def test_statistical_sanity_noUT(oracle, geometry, nparams):
    """Run-3-like events: particles above the assumed momentum are found, ghosts stay rare (tight chi2 cuts,
    PAPER.md:323), fake seeds give almost nothing, and the with-UT tuning finds more (it sees p < 5 GeV)."""
    b = dg.generate_config(1, n_events=120)
    r = oracle.run(geometry, nparams, b, threads=4)
    e = truth.evaluate(b, r.hit_idx, r.n_hits)
    rec = truth.reconstructible(b)
    pa = np.zeros(b.n_tracks)
    true_seed = b.seed_track >= 0
    pa[b.seed_track[true_seed]] = _assumed_p(b, nparams)[true_seed]
    above = rec & (1.0 / np.abs(b.trk_qop) > 1.3 * pa)
    found = np.zeros(b.n_tracks, bool)
    found[e.matched_track[e.matched_track >= 0]] = True
    assert above.sum() > 5000
    assert found[above].mean() > 0.97, found[above].mean()
    assert e.ghost_rate < 0.01
    fake = b.seed_track[r.seed_idx] < 0
    assert fake.sum() / max(int((b.seed_track < 0).sum()), 1) < 0.02
    r_ut = oracle.run(geometry, dg.default_params(), b, threads=4)
    assert r_ut.n_tracks > r.n_tracks


def test_f32_build_matches_f64_build_noUT(oracle, geometry, nparams):
    b = dg.generate_config(1, n_events=100)
    a = oracle.run(geometry, nparams, b, threads=4)
    c = oracle.run(geometry, nparams, b, real="f64", threads=4)
    common, ia, ic = np.intersect1d(a.seed_idx, c.seed_idx, return_indices=True)
    assert len(common) >= 0.998 * max(a.n_tracks, c.n_tracks)
    assert (a.hit_idx[ia] == c.hit_idx[ic]).all(1).mean() > 0.998


def test_thread_sharding_and_ignored_qop_noUT(oracle, geometry, nparams):
    b = dg.generate_config(1, n_events=24)
    a = oracle.run(geometry, nparams, b, debug=True)
    b2 = dg.Batch(**{**b.__dict__, "seed_qop": -3.0 * b.seed_qop})
    c = oracle.run(geometry, nparams, b2, debug=True, threads=4)
    for k in ("hit_idx", "seed_idx", "n_hits", "state", "quality", "event_offsets"):
        assert np.array_equal(getattr(a, k), getattr(c, k)), k
    for k in ("win_first", "win_count", "n_triplets", "trip_hits", "trip_chi2", "cand_hits", "cand_quality"):
        assert np.array_equal(getattr(a.debug, k), getattr(c.debug, k)), k
