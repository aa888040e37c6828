"""Truth matching on generated batches (evaluation only; no step of the algorithm).

Follows the paper's methodology: a reconstructed track is matched to a particle
if more than 70 % of its hits come from that particle; efficiency is measured with respect to
"reconstructible" particles; the fake (ghost) rate is the unmatched fraction of tracks.
Reconstructible here: >= 9 generated hits with >= 1 u/v hit per station -- the
algorithm's own acceptance rule applied to the truth hits.
"""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np

N_LAYERS = 12


def hit_layers(batch) -> np.ndarray:
    """Layer index of every hit, from the segment table."""
    seg_counts = np.diff(batch.seg_offsets.astype(np.int64))
    seg_layer = (np.arange(seg_counts.shape[0]) % (2 * N_LAYERS)) // 2
    return np.repeat(seg_layer, seg_counts).astype(np.int8)


def reconstructible(batch) -> np.ndarray:
    """Boolean mask over the true-track table."""
    lay = hit_layers(batch)
    sel = batch.hit_track >= 0
    tid, l = batch.hit_track[sel].astype(np.int64), lay[sel].astype(np.int64)
    per_layer = np.zeros((batch.n_tracks, N_LAYERS), dtype=np.int32)
    np.add.at(per_layer, (tid, l), 1)
    has = per_layer > 0
    n = has.sum(1)
    uv_ok = np.ones(batch.n_tracks, dtype=bool)
    for st in range(3):
        uv_ok &= has[:, 4 * st + 1] | has[:, 4 * st + 2]
    return (n >= 9) & uv_ok


def evaluate(batch, hit_idx: np.ndarray, n_hits: np.ndarray) -> SimpleNamespace:
    """Efficiency / ghost rate of a set of output tracks (rows of global hit indices, -1 = none)."""
    n_trk = hit_idx.shape[0]
    rec = reconstructible(batch)
    if n_trk == 0:
        return SimpleNamespace(n_tracks=0, n_reconstructible=int(rec.sum()), efficiency=0.0, ghost_rate=0.0,
                               matched_track=np.zeros(0, np.int64))
    ht = np.where(hit_idx >= 0, batch.hit_track[np.maximum(hit_idx, 0)], -2).astype(np.int64)
    # majority particle of each track
    srt = np.sort(ht, axis=1)
    best = np.full(n_trk, -1, dtype=np.int64)
    best_n = np.zeros(n_trk, dtype=np.int64)
    for c in range(N_LAYERS):
        cand = srt[:, c]
        cnt = (ht == cand[:, None]).sum(1)
        upd = (cand >= 0) & (cnt > best_n)
        best[upd], best_n[upd] = cand[upd], cnt[upd]
    matched = best_n > 0.7 * n_hits
    mt = np.where(matched, best, -1)
    found = np.zeros(batch.n_tracks, dtype=bool)
    found[mt[mt >= 0]] = True
    n_rec = int(rec.sum())
    return SimpleNamespace(
        n_tracks=n_trk, n_reconstructible=n_rec,
        efficiency=float((found & rec).sum()) / max(n_rec, 1),
        ghost_rate=float((~matched).sum()) / n_trk,
        matched_track=mt)
