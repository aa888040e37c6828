"""Pins of the CPU oracle.  All CPU-only.

The oracle is pinned to things other than itself:
  1. a brute-force twin written from the definitions (membership tests, argmin, full sorts, lstsq);
  2. the generator's truth on noise-free single tracks + closed forms of the TOY field;
  3. invariants every output must satisfy;
  4. textbook reductions: numpy.linalg.lstsq on the oracle's own hit lists, numpy.searchsorted;
  5. its own fp64 build (rounding only) and statistical sanity against the truth.
"""
import os

import numpy as np
import pytest

from paper_2402_14670_b200 import datagen as dg
from paper_2402_14670_b200 import truth

HERE = os.path.dirname(os.path.abspath(__file__))
NL = 12


# ------------------------------------------------------------------------------------------------
def test_paper_constants_fixture(params, geometry):
    vals = {}
    for line in open(os.path.join(HERE, "golden", "paper_constants.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            vals[line[0]] = float(line[1])
    for k, v in vals.items():
        if k.startswith("C_nhits_"):
            assert params["C_nhits"][int(k.split("_")[-1]) - 9] == v
        elif k == "z_ref":
            assert geometry["z_ref"] == v
        else:
            assert params[k] == v, k


# ------------------------------------------------------------------------------------------------
# Pin 1: brute-force twin
# ------------------------------------------------------------------------------------------------
def _assert_twin_equal(oracle, G, P, b):
    from oracle import brute_twin
    r = oracle.run(G, P, b, real="f64", debug=True)
    tw = brute_twin.run(G, P, b)
    assert np.array_equal(tw.win_count, r.debug.win_count)
    m = tw.win_count > 0
    assert np.array_equal(tw.win_first[m], r.debug.win_first[m])
    for si, trips in enumerate(tw.triplets):
        assert len(trips) == r.debug.n_triplets[si]
        for k, (chi2, s, i0, i2, i1) in enumerate(trips):
            assert tuple(r.debug.trip_hits[si, k]) == (i0, i1, i2) and r.debug.trip_set[si, k] == s
            assert abs(r.debug.trip_chi2[si, k] - chi2) <= 1e-5 * max(1.0, chi2)
    assert tw.n_tracks == r.n_tracks
    assert np.array_equal(tw.seed_idx, r.seed_idx)
    assert np.array_equal(tw.hit_idx, r.hit_idx)
    assert np.array_equal(tw.n_hits, r.n_hits)
    assert np.array_equal(tw.event_offsets, r.event_offsets)
    # oracle writes float32 outputs: compare to output rounding
    assert np.max(np.abs(tw.state[:, 0] - r.state[:, 0])) < 3e-4
    assert np.max(np.abs(tw.state[:, 1] - r.state[:, 1])) < 3e-4
    assert np.max(np.abs(tw.state[:, 2:4] - r.state[:, 2:4])) < 1e-7
    assert np.max(np.abs(tw.state[:, 4] / r.state[:, 4] - 1)) < 1e-6
    assert np.max(np.abs(tw.quality - r.quality)) < 1e-6
    return r


def test_twin_config0(oracle, geometry, params):
    r = _assert_twin_equal(oracle, geometry, params, dg.generate_config(0))
    assert r.n_tracks > 150


def test_twin_dense_event_caps_bind(oracle, geometry, params):
    """Dense tiny events: n_window cap and the top-12 cut both bind; both magnet polarities."""
    cfg = dg.GenConfig("dense", 2, 77, true_fixed=25, fake_mean=5.0, noise_fixed=450, p_min=1.5, smear=0.2)
    b = dg.generate(cfg)
    r = _assert_twin_equal(oracle, geometry, params, b)
    assert (r.debug.win_count == params["n_window"]).mean() > 0.3
    assert (r.debug.n_triplets == params["n_triplets"]).sum() > 5
    G2 = dict(geometry, polarity=-1)
    _assert_twin_equal(oracle, G2, params, b)


def test_twin_nondefault_params(oracle, geometry, params):
    """Odd window cap, fewer triplets, non-zero dRatio: the twin still agrees."""
    P = dict(params, n_window=9, n_triplets=5, T_x=1.0, T_triplet=4.0, x_asym=60.0)
    G = dict(geometry, d_ratio=-2.0e-5)
    cfg = dg.GenConfig("dense2", 2, 78, true_fixed=20, fake_mean=3.0, noise_fixed=300)
    _assert_twin_equal(oracle, G, P, dg.generate(cfg))


# ------------------------------------------------------------------------------------------------
# Pin 2: generator truth and closed forms
# ------------------------------------------------------------------------------------------------
def _full_tracks(b):
    """Track ids whose 12 hits were all generated."""
    cnt = np.bincount(b.hit_track[b.hit_track >= 0], minlength=b.n_tracks)
    return cnt == NL


@pytest.mark.parametrize("real,tol_x,tol_t,tol_q", [("f64", 2.5e-4, 1e-6, 1e-5), ("f32", 1.5e-3, 3e-6, 1e-4)])
def test_truth_exact_hits_noise_free(oracle, geometry, params, real, tol_x, tol_t, tol_q):
    """sigma = 0, exact seeds: all 12 true hits, Q ~ 0, state and q/p reproduce the truth model."""
    b = dg.generate(dg.single_track_config(400, seed=11, sigma=0.0, smear=0.0))
    r = oracle.run(geometry, params, b, real=real, debug=True)
    full = _full_tracks(b)
    tid = b.seed_track[r.seed_idx]
    found = np.zeros(b.n_tracks, bool)
    found[tid] = True
    assert np.all(found[full]), "a fully measured noise-free track was not found"
    sel = full[tid]
    assert sel.sum() > 250
    hit_t = b.hit_track[r.hit_idx[sel]]
    assert np.all(hit_t == tid[sel][:, None])
    assert np.all(r.n_hits[sel] == NL)
    assert np.max(r.quality[sel]) < (1e-7 if real == "f64" else 1e-5)  # hits are fp32-rounded (ulp 2.4e-4 mm)
    # closed forms of the TOY field at z_state
    zs = geometry["z_state"]
    t = tid[sel]
    x_mag = b.trk_x[t] + b.trk_tx[t] * (dg.TOY_Z_MAG - dg.TOY_Z_SEED)
    dtx = dg.TOY_KICK * b.trk_qop[t]
    x_true = dg.toy_x_at(x_mag, b.trk_tx[t] + dtx, dtx, zs)
    tx_true = dg.toy_tx_at(b.trk_tx[t] + dtx, dtx, zs)
    y_true = b.trk_y[t] + b.trk_ty[t] * (zs - dg.TOY_Z_SEED)
    st = r.state[sel].astype(np.float64)
    assert np.max(np.abs(st[:, 0] - x_true)) < tol_x
    assert np.max(np.abs(st[:, 1] - y_true)) < 10 * tol_x     # y = residual / tan(5 deg): 11x lever
    assert np.max(np.abs(st[:, 2] - tx_true)) < tol_t
    assert np.max(np.abs(st[:, 3] - b.trk_ty[t])) < 10 * tol_t
    assert np.max(np.abs(st[:, 4] / b.trk_qop[t] - 1.0)) < tol_q   # pins C18 (Eq. 9 reduced)
    # K_x1 (C5): the true triplet's residual is < 0.01 mm
    first = r.debug.trip_chi2[r.seed_idx[sel], 0]
    assert np.max(first) < 0.01 ** 2


def test_truth_reversed_field(oracle, params):
    """Reading C7 with the field reversed (kick < 0, polarity -1): the same-bend filter compares the doublet's slope
    change with the sign of kick * q/p (Eq. 2), so low-momentum truth is still found with exactly its hits.  A filter
    written as (t - tx) * q/p > 0 would reject every true doublet below p_same_bend here."""
    G = dg.toy_geometry(polarity=-1, kick_sign=-1.0)
    cfg = dg.with_overrides(dg.single_track_config(400, seed=13, sigma=0.0, smear=0.0), kick_sign=-1.0, p_max=4.5)
    b = dg.generate(cfg)
    assert np.all(1.0 / np.abs(b.trk_qop) < params["p_same_bend"])
    r = oracle.run(G, params, b, debug=True)
    full = _full_tracks(b)
    tid = b.seed_track[r.seed_idx]
    found = np.zeros(b.n_tracks, bool)
    found[tid] = True
    assert full.sum() > 150 and np.all(found[full])
    sel = full[tid]
    assert np.all(b.hit_track[r.hit_idx[sel]] == tid[sel][:, None])
    assert np.max(np.abs(r.state[sel, 4].astype(np.float64) / b.trk_qop[tid[sel]] - 1.0)) < 1e-4


def test_truth_measured_hits_found(oracle, geometry, params):
    """sigma = 0.08 mm, 5 % q/p smear, no noise: exactly the generated hits of each >=9-hit track."""
    b = dg.generate(dg.with_overrides(dg.single_track_config(600, seed=12, sigma=0.08, smear=0.05), eff=0.98))
    r = oracle.run(geometry, params, b)
    rec = truth.reconstructible(b)
    tid = b.seed_track[r.seed_idx]
    found = np.zeros(b.n_tracks, bool)
    found[tid] = True
    assert found[rec].mean() > 0.995
    # every output hit belongs to the seed's particle, and none of its in-window hits is missed
    hit_t = np.where(r.hit_idx >= 0, b.hit_track[np.maximum(r.hit_idx, 0)], tid[:, None])
    assert np.all(hit_t == tid[:, None])
    n_true = np.bincount(b.hit_track, minlength=b.n_tracks)
    assert (r.n_hits == n_true[tid]).mean() > 0.99
    # momentum resolution is far below the paper's 1 % on this noise-free sample
    assert np.median(np.abs(r.state[:, 4] / b.trk_qop[tid] - 1.0)) < 2e-3


def test_charge_asymmetry_follows_eq3(oracle, geometry, params):
    """Eq. (3): q>0 with MU (or q<0 with MD) widens the LEFT edge by x_asym, else the right edge."""
    b = dg.generate(dg.GenConfig("asym", 4, 5, true_fixed=30, noise_fixed=600))
    P = dict(params, n_window=4096)       # no cap, so edges are visible
    P0 = dict(P, x_asym=0.0)
    for pol in (+1, -1):
        G = dict(geometry, polarity=pol)
        r1 = oracle.run(G, P, b, debug=True).debug
        r0 = oracle.run(G, P0, b, debug=True).debug
        xl = [0, 3, 4, 7, 8, 11]
        left_grew = (r1.win_first[:, xl] < r0.win_first[:, xl]).any(1)
        right_grew = ((r1.win_first + r1.win_count)[:, xl] > (r0.win_first + r0.win_count)[:, xl]).any(1)
        assert not np.any(left_grew & right_grew)
        qpos = b.seed_qop > 0
        want_left = qpos if pol > 0 else ~qpos
        assert np.all(left_grew[~want_left] == False) and np.all(right_grew[want_left] == False)
        assert left_grew[want_left].mean() > 0.9 and right_grew[~want_left].mean() > 0.9
        # u/v windows do not depend on the asymmetry
        uv = [1, 2, 5, 6, 9, 10]
        assert np.array_equal(r1.win_first[:, uv], r0.win_first[:, uv])


# ------------------------------------------------------------------------------------------------
# Pin 3: invariants
# ------------------------------------------------------------------------------------------------
def _check_invariants(b, P, r):
    n = r.n_tracks
    assert r.hit_idx.shape == (n, NL)
    assert np.all(np.diff(r.seed_idx) > 0), "tracks must be in seed order, at most one per seed"
    ev_of_seed = np.searchsorted(b.seed_offsets, r.seed_idx, side="right") - 1
    assert np.array_equal(np.bincount(ev_of_seed, minlength=b.n_events), np.diff(r.event_offsets.astype(np.int64)))
    # every hit sits in the right (event, layer, zone) segment
    zone = (b.seed_ty[r.seed_idx] >= 0).astype(np.int64)
    for l in range(NL):
        h = r.hit_idx[:, l].astype(np.int64)
        have = h >= 0
        seg = ev_of_seed * 24 + l * 2 + zone
        assert np.all(h[have] >= b.seg_offsets[seg[have]]) and np.all(h[have] < b.seg_offsets[seg[have] + 1])
    assert np.array_equal((r.hit_idx >= 0).sum(1), r.n_hits)
    assert np.all(r.n_hits >= P["min_hits"])
    for st in range(3):
        assert np.all((r.hit_idx[:, 4 * st + 1] >= 0) | (r.hit_idx[:, 4 * st + 2] >= 0))
    assert np.all(r.quality < P["T_Q"]) and np.all(r.quality >= 0)
    assert np.all(np.abs(r.state[:, 3] - b.seed_ty[r.seed_idx]) < P["T_ty"])
    assert np.all(np.isfinite(r.state))
    if r.debug is not None:
        d = r.debug
        assert np.all(d.win_count <= P["n_window"]) and np.all(d.win_count >= 0)
        assert np.all(d.n_triplets <= P["n_triplets"])
        # kept triplets are in (chi2, set, i0, i2) order and below the cut
        c = d.trip_chi2
        for k in range(P["n_triplets"] - 1):
            both = (d.n_triplets > k + 1)
            assert np.all(c[both, k] <= c[both, k + 1])
        assert np.all(c[c >= 0] < P["T_triplet"])
        # hits on a track lie inside that seed's window of the layer
        wf, wc = d.win_first[r.seed_idx], d.win_count[r.seed_idx]
        have = r.hit_idx >= 0
        assert np.all((r.hit_idx >= wf)[have]) and np.all((r.hit_idx < wf + wc)[have])


@pytest.mark.parametrize("cid,n_events", [(0, None), (1, 60), (4, 25)])
def test_invariants(oracle, geometry, params, cid, n_events):
    b = dg.generate_config(cid, n_events=n_events)
    r = oracle.run(geometry, params, b, debug=True)
    _check_invariants(b, params, r)
    # fake seeds (random states that match no hits) produce almost nothing
    fake = b.seed_track[r.seed_idx] < 0
    n_fake = max(int((b.seed_track < 0).sum()), 1)
    assert fake.sum() / n_fake < (0.02 if cid != 4 else 0.12)


def test_windows_against_searchsorted(oracle, geometry, params):
    """Uncapped window edges are numpy.searchsorted(lo,'left') / (hi,'right') on the sorted segment."""
    b = dg.generate_config(1, n_events=8)
    P = dict(params, n_window=1 << 20)
    d = oracle.run(geometry, P, b, debug=True).debug
    z = np.asarray(geometry["z"])
    ev = np.searchsorted(b.seed_offsets, np.arange(b.n_seeds), side="right") - 1
    zone = (b.seed_ty >= 0).astype(np.int64)
    f = np.float32
    for si in range(0, b.n_seeds, 7):
        aq = max(abs(f(b.seed_qop[si])), f(1e-6))
        x_mag = f(b.seed_x[si]) + f(b.seed_tx[si]) * f(f(geometry["z_mag"]) - f(geometry["z_seed"]))
        txp = f(b.seed_tx[si]) + f(geometry["kick"]) * f(b.seed_qop[si])
        l = 5  # a u layer: centre x_c + y*tan(alpha), +-800 mm
        xc = x_mag + txp * f(f(z[l]) - f(geometry["z_mag"]))
        yl = f(b.seed_y[si]) + f(b.seed_ty[si]) * f(f(z[l]) - f(geometry["z_seed"]))
        ctr = xc + yl * f(geometry["tan_alpha"][l])
        s0, s1 = b.seg_offsets[ev[si] * 24 + l * 2 + zone[si]], b.seg_offsets[ev[si] * 24 + l * 2 + zone[si] + 1]
        seg = b.hit_x[s0:s1]
        lo, hi = ctr - f(800.0), ctr + f(800.0)
        assert d.win_first[si, l] == s0 + np.searchsorted(seg, lo, side="left")
        assert d.win_first[si, l] + d.win_count[si, l] == s0 + np.searchsorted(seg, hi, side="right")


# ------------------------------------------------------------------------------------------------
# Pin 4: least-squares fits against numpy.linalg.lstsq in float64 on the oracle's own hit lists
# ------------------------------------------------------------------------------------------------
def test_fit_against_lstsq(oracle, geometry, params):
    b = dg.generate_config(1, n_events=40)
    r = oracle.run(geometry, params, b)
    z = np.asarray(geometry["z"], float)
    tana = np.asarray(geometry["tan_alpha"], float)
    z_ref, zs = geometry["z_ref"], geometry["z_state"]
    T_x, T_y = params["T_x"], params["T_y"]
    worst = np.zeros(6)
    for i in range(0, r.n_tracks, 5):
        si = r.seed_idx[i]
        y0, ty, tx = float(b.seed_y[si]), float(b.seed_ty[si]), float(b.seed_tx[si])
        lay = np.nonzero(r.hit_idx[i] >= 0)[0]
        s = b.hit_x[r.hit_idx[i, lay]].astype(float)
        dz = z[lay] - z_ref
        yl = y0 + ty * (z[lay] - geometry["z_seed"])
        A = np.stack([np.ones_like(dz), dz, dz * dz], 1)
        m = s - yl * tana[lay]
        par, *_ = np.linalg.lstsq(A, m, rcond=None)
        res = m - A @ par
        uv = tana[lay] != 0
        T_uv = max(params["T_uv_min"], params["T_uv_slope"] * (abs(tx) + abs(ty)))
        Qx = np.sum(res[~uv] ** 2) / T_x + np.sum(res[uv] ** 2) / T_uv
        yi = (s[uv] - A[uv] @ par) / tana[lay][uv]
        Ay = np.stack([np.ones(uv.sum()), dz[uv]], 1)
        yp, *_ = np.linalg.lstsq(Ay, yi, rcond=None)
        Qy = np.sum((yi - Ay @ yp) ** 2) / T_y
        n, nuv = len(lay), int(uv.sum())
        Q = (Qx / (n - 3) + Qy / (nuv - 2)) * params["C_nhits"][n - 9]
        dzs = zs - z_ref
        ref = np.array([par[0] + par[1] * dzs + par[2] * dzs ** 2, yp[0] + yp[1] * dzs,
                        par[1] + 2 * par[2] * dzs, yp[1], (par[1] - tx) / geometry["qop_poly"][0], Q])
        got = np.array(list(r.state[i]) + [r.quality[i]], float)
        worst = np.maximum(worst, np.abs(got - ref) / np.array([1, 1, 1, 1, abs(ref[4]), max(ref[5], 1e-3)]))
    # fp32 oracle vs float64 textbook solve
    assert worst[0] < 2e-3 and worst[1] < 2e-2 and worst[2] < 3e-6 and worst[3] < 3e-5
    assert worst[4] < 2e-4 and worst[5] < 2e-2


# ------------------------------------------------------------------------------------------------
# Pin 5: fp32 reference build vs fp64 build; statistical sanity; harness sharding
# ------------------------------------------------------------------------------------------------
def test_f32_build_matches_f64_build(oracle, geometry, params):
    b = dg.generate_config(1, n_events=150)
    a = oracle.run(geometry, params, b, threads=4)
    c = oracle.run(geometry, params, b, real="f64", threads=4)
    common, ia, ic = np.intersect1d(a.seed_idx, c.seed_idx, return_indices=True)
    assert len(common) >= 0.999 * max(a.n_tracks, c.n_tracks)
    same = (a.hit_idx[ia] == c.hit_idx[ic]).all(1)
    assert same.mean() > 0.998
    d = np.abs(a.state[ia][same].astype(float) - c.state[ic][same].astype(float))
    assert d[:, 0].max() < 2e-3 and d[:, 1].max() < 2e-2 and d[:, 2].max() < 3e-6 and d[:, 3].max() < 3e-5


@pytest.mark.parametrize("cid,n_events,eff_lo,eff_hi,ghost_hi", [(0, None, 0.98, 1.0, 0.01), (1, 200, 0.985, 1.0, 0.005),
                                                               (4, 60, 0.70, 0.83, 0.06)])
def test_statistical_sanity(oracle, geometry, params, cid, n_events, eff_lo, eff_hi, ghost_hi):
    b = dg.generate_config(cid, n_events=n_events)
    r = oracle.run(geometry, params, b, threads=4)
    e = truth.evaluate(b, r.hit_idx, r.n_hits)
    assert eff_lo <= e.efficiency <= eff_hi, e.efficiency
    assert e.ghost_rate <= ghost_hi, e.ghost_rate


def test_thread_sharding_is_transparent(oracle, geometry, params):
    b = dg.generate_config(1, n_events=30)
    a = oracle.run(geometry, params, b, debug=True)
    c = oracle.run(geometry, params, b, debug=True, threads=4)
    for k in ("hit_idx", "seed_idx", "n_hits", "state", "quality", "event_offsets"):
        assert np.array_equal(getattr(a, k), getattr(c, k)), k
    for k in ("win_first", "win_count", "n_triplets", "trip_hits", "trip_chi2", "cand_hits", "cand_quality"):
        assert np.array_equal(getattr(a.debug, k), getattr(c.debug, k)), k


def test_edge_cases(oracle, geometry, params):
    # no events; events without seeds; events without hits
    empty = dg.generate(dg.GenConfig("e", 0, 1))
    r = oracle.run(geometry, params, empty)
    assert r.n_tracks == 0 and r.event_offsets.tolist() == [0]
    noseed = dg.generate(dg.GenConfig("ns", 3, 2, true_fixed=0, noise_fixed=50))
    r = oracle.run(geometry, params, noseed)
    assert r.n_tracks == 0 and r.event_offsets.tolist() == [0, 0, 0, 0]
    b = dg.generate_config(0)
    nohits = dg.Batch(**{**b.__dict__, "hit_x": np.zeros(0, np.float32),
                        "seg_offsets": np.zeros(b.n_events * 24 + 1, np.uint32),
                        "hit_track": np.zeros(0, np.int32)})
    r = oracle.run(geometry, params, nohits)
    assert r.n_tracks == 0


def test_golden_config0_regression(oracle, geometry, params):
    """Oracle output on configs[0] equals the stored file written by tests/golden/make_golden.py."""
    r = oracle.run(geometry, params, dg.generate_config(0))
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "cfg0_oracle_tracks.txt")) if not l.startswith("#")]
    assert len(rows) == r.n_tracks
    for i, row in enumerate(rows):
        assert int(row[0]) == r.seed_idx[i] and int(row[1]) == r.n_hits[i]
        assert [int(v) for v in row[2:14]] == r.hit_idx[i].tolist()
        bits = [np.float32(r.quality[i]).view(np.uint32).item()] + [np.float32(v).view(np.uint32).item() for v in r.state[i]]
        assert [int(v, 16) for v in row[14:20]] == bits
