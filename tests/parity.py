"""Comparison rules of BASELINE.json north_star for GPU output vs oracle output (same seeded inputs).

  * hit indices, seed indices, hit counts, per-event offsets, track count: BIT-EXACT;
  * fitted x, y within 1e-3 mm; slopes within 1e-6; q/p within 1e-4 relative;
  * Q within 1e-6 absolute + 1e-4 relative (not named by north_star; same arithmetic).
"""
import numpy as np


def assert_tracks_equal(got, ref, what=""):
    assert got.n_tracks == ref.n_tracks, f"{what}: track count {got.n_tracks} != oracle {ref.n_tracks}"
    assert np.array_equal(got.event_offsets, ref.event_offsets), f"{what}: event offsets differ"
    assert np.array_equal(got.seed_idx, ref.seed_idx), f"{what}: seed indices differ"
    bad = np.nonzero((got.hit_idx != ref.hit_idx).any(1))[0]
    assert bad.size == 0, f"{what}: {bad.size} tracks with different hit lists, first at {bad[:5]}"
    assert np.array_equal(got.n_hits, ref.n_hits), f"{what}: hit counts differ"
    if got.n_tracks == 0:
        return dict(bit_identical=True)
    ds = np.abs(got.state.astype(np.float64) - ref.state.astype(np.float64))
    assert ds[:, 0].max() <= 1e-3 and ds[:, 1].max() <= 1e-3, f"{what}: x/y differ by {ds[:, :2].max(0)}"
    assert ds[:, 2].max() <= 1e-6 and ds[:, 3].max() <= 1e-6, f"{what}: slopes differ by {ds[:, 2:4].max(0)}"
    rq = np.abs(got.state[:, 4].astype(np.float64) / ref.state[:, 4].astype(np.float64) - 1.0)
    assert rq.max() <= 1e-4, f"{what}: q/p differs by {rq.max()} relative"
    dq = np.abs(got.quality.astype(np.float64) - ref.quality.astype(np.float64))
    assert np.all(dq <= 1e-6 + 1e-4 * np.abs(ref.quality)), f"{what}: Q differs by {dq.max()}"
    return dict(bit_identical=bool(np.array_equal(got.state.view(np.uint32), ref.state.view(np.uint32))
                                   and np.array_equal(got.quality.view(np.uint32), ref.quality.view(np.uint32))),
                max_dx=float(ds[:, 0].max()), max_dy=float(ds[:, 1].max()))


def assert_debug_equal(gd, rd, n_window_ok=True):
    """Stage boundaries: windows, kept triplets, extension results, per-candidate Q."""
    assert np.array_equal(gd["win_count"], rd.win_count), "window counts differ"
    m = rd.win_count > 0
    assert np.array_equal(gd["win_first"][m], rd.win_first[m]), "window starts differ"
    assert np.array_equal(gd["n_triplets"], rd.n_triplets), "triplet counts differ"
    assert np.array_equal(gd["trip_hits"], rd.trip_hits), "triplet hits differ"
    assert np.array_equal(gd["trip_set"], rd.trip_set), "triplet layer sets differ"
    assert np.array_equal(gd["trip_chi2"].view(np.uint32), rd.trip_chi2.view(np.uint32)), "triplet chi2 differ"
    assert np.array_equal(gd["cand_hits"], rd.cand_hits), "extension hit lists differ"
    gq, rq = gd["cand_quality"], rd.cand_quality
    assert np.array_equal(gq < 0, rq < 0) and np.array_equal(gq[rq < 0], rq[rq < 0]), "candidate status differs"
    ok = rq >= 0
    assert np.all(np.abs(gq[ok] - rq[ok]) <= 1e-6 + 1e-4 * np.abs(rq[ok])), "candidate Q differs"
