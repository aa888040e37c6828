"""Generator: determinism, layout, occupancy (BASELINE.json configs)."""
import numpy as np

from paper_2402_14670_b200 import datagen as dg


def _sorted_in_segments(b):
    d = np.diff(b.hit_x)
    bad = np.nonzero(d < 0)[0] + 1
    return np.all(np.isin(bad, b.seg_offsets))


def test_layout_and_sortedness():
    b = dg.generate_config(0)
    assert b.n_events == 10 and b.n_seeds == 200
    assert b.seed_offsets.dtype == np.uint32 and b.seg_offsets.dtype == np.uint32
    assert b.seed_offsets.shape == (11,) and b.seg_offsets.shape == (10 * 24 + 1,)
    assert b.seed_offsets[-1] == b.n_seeds and b.seg_offsets[-1] == b.n_hits
    assert b.hit_x.dtype == np.float32 and b.seed_qop.dtype == np.float32
    assert _sorted_in_segments(b)
    assert np.all(np.abs(b.hit_x[b.hit_track < 0]) <= dg.TOY_X_HALF)
    # 20 true tracks per event, none fake
    assert np.all(np.diff(b.seed_offsets) == 20) and np.all(b.seed_track >= 0)


def test_deterministic_and_worker_independent():
    a = dg.generate_config(1, n_events=600, workers=1)
    b = dg.generate_config(1, n_events=600, workers=3)
    for k in ("seed_x", "seed_qop", "seed_offsets", "hit_x", "seg_offsets", "hit_track", "seed_track"):
        assert np.array_equal(getattr(a, k), getattr(b, k)), k
    # a prefix of whole chunks is identical to the shorter run
    c = dg.generate_config(1, n_events=250)
    assert np.array_equal(c.hit_x, a.hit_x[: c.n_hits]) and np.array_equal(c.seed_x, a.seed_x[: c.n_seeds])


def test_occupancy_matches_baseline_configs():
    b = dg.generate_config(1, n_events=500)
    assert abs(b.n_hits / b.n_events - 5000) < 100          # "about 5,000 SciFi hits"
    assert abs(b.n_seeds / b.n_events - 180) < 4            # Poisson(150) + Poisson(30)
    assert abs((b.seed_track < 0).sum() / b.n_events - 30) < 2
    b4 = dg.generate_config(4, n_events=250)
    assert abs(b4.n_hits / b4.n_events - 12000) < 250       # "about 12,000 hits per event"
    assert abs(b4.n_seeds / b4.n_events - 360) < 8
    p_true = 1.0 / np.abs(b4.trk_qop)
    assert p_true.min() >= 1.5 and p_true.max() <= 100.0
    assert _sorted_in_segments(b) and _sorted_in_segments(b4)


def test_zone_is_sign_of_y_and_stereo_sign():
    cfg = dg.single_track_config(200, seed=7)
    b = dg.generate(cfg)
    seg_of_hit = np.repeat(np.arange(b.seg_offsets.shape[0] - 1), np.diff(b.seg_offsets.astype(np.int64)))
    layer, zone = (seg_of_hit % 24) // 2, seg_of_hit % 2
    t = b.hit_track
    assert np.all(zone == (b.trk_ty[t] >= 0))
    # stored coordinate = x + y*tan(alpha): recompute from the truth model
    z = np.asarray(dg.TOY_Z)[layer]
    x_mag = b.trk_x[t] + b.trk_tx[t] * (dg.TOY_Z_MAG - dg.TOY_Z_SEED)
    dtx = dg.TOY_KICK * b.trk_qop[t]
    x = dg.toy_x_at(x_mag, b.trk_tx[t] + dtx, dtx, z)
    y = b.trk_y[t] + b.trk_ty[t] * (z - dg.TOY_Z_SEED)
    s = x + y * np.asarray(dg.TOY_TAN)[layer]
    assert np.max(np.abs(s - b.hit_x)) < 5e-4


def test_slice_events_rebases():
    b = dg.generate_config(1, n_events=20)
    s = b.slice_events(5, 9)
    assert s.n_events == 4 and s.seed_offsets[0] == 0 and s.seg_offsets[0] == 0
    assert s.seed_offsets[-1] == s.n_seeds and s.seg_offsets[-1] == s.n_hits
    h0 = int(b.seg_offsets[5 * 24])
    assert np.array_equal(s.hit_x, b.hit_x[h0:h0 + s.n_hits])


def test_toy_k_closed_form_against_simulation():
    """K_x1 for the TOY field (C5): chord through layers a,c + K correction hits layer b."""
    G = dg.toy_geometry()
    rng = np.random.default_rng(5)
    qop = rng.choice([-1, 1], 2000) / np.exp(rng.uniform(np.log(2), np.log(100), 2000))
    tx = rng.uniform(-0.25, 0.25, 2000)
    x_mag = tx * dg.TOY_Z_MAG
    dtx = dg.TOY_KICK * qop
    for (a, bb, c), K in (((0, 4, 8), G["k_first"]), ((3, 7, 11), G["k_last"])):
        za, zb, zc = dg.TOY_Z[a], dg.TOY_Z[bb], dg.TOY_Z[c]
        xa, xb, xc = (dg.toy_x_at(x_mag, tx + dtx, dtx, zz) for zz in (za, zb, zc))
        t = (xc - xa) / (zc - za)
        x1e = zb * t + (xa - t * za) * K
        assert np.max(np.abs(x1e - xb)) < 1e-9
