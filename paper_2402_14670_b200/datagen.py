"""Seeded synthetic-event generator (inputs only; holds none of the method's arithmetic).

This module serves BOTH the CUDA path and the oracle with identical arrays.  It
contains the TOY detector / field model of BASELINE.json ``configs[0]`` (the
*truth* propagation that produces hits) and the five workload recipes, but no
step of the Looking Forward algorithm itself (no windows, no seeding, no fit).

Layout produced (north_star (b)):

* seeds : SoA float32 ``x, y, tx, ty, qop`` at ``z_seed`` + ``seed_offsets`` (uint32, n_events+1)
* hits  : float32 stored coordinate ``s = x + y*tan(alpha)``; event-major, then layer 0..11, then
          zone 0 (y<0) / 1 (y>=0); ascending inside every (event, layer, zone) segment;
          ``seg_offsets`` (uint32, n_events*24+1)
* truth : ``hit_track`` (int32 track id per hit, -1 noise), ``seed_track`` (int32, -1 fake seed),
          and the true-track table (``trk_*``).

Determinism: events are generated in fixed chunks of ``CHUNK_EVENTS``; chunk *k* draws from
``numpy.random.Generator(PCG64(SeedSequence([seed, k])))`` in a fixed order, so the output
depends only on (recipe, n_events, seed) and not on the number of worker threads.

The paper measures on LHCb full simulation, which is not available; these
synthetic events stand in for it with the paper's shapes (12 layers x-u-v-x at +-5 deg,
PAPER.md:36; upper/lower halves; a few hundred hits per layer).
"""
from __future__ import annotations

import math
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional

import numpy as np

N_LAYERS = 12
N_ZONES = 2
N_SEGS = N_LAYERS * N_ZONES
CHUNK_EVENTS = 250

TAN5 = 0.0874886635  # tan(5 deg), the single literal used everywhere

# ----------------------------------------------------------------------------------------------
# TOY detector + field (BASELINE.json configs[0])
# ----------------------------------------------------------------------------------------------
TOY_Z = (7826.0, 7896.0, 7966.0, 8036.0, 8508.0, 8578.0, 8648.0, 8718.0, 9193.0, 9263.0, 9333.0, 9403.0)
TOY_TAN = (0.0, TAN5, -TAN5, 0.0) * 3
TOY_Z_SEED = 770.0
TOY_Z_MAG = 5200.0
TOY_KICK = 1.2          # delta tx = kick * q/p  (p in GeV)
TOY_C2 = 4.0e-7         # x(z) += c2 * dtx * (z - z0)^2 for z beyond z0
TOY_Z0 = 7800.0         # = z_mag + 2600
TOY_X_HALF = 3000.0
TOY_Y_HALF = 2500.0
TOY_Z_REF = 8520.0
X_LAYER_SETS = ((0, 4, 8), (3, 7, 11))  # first / last x layer of each station


def _toy_k(za: float, zb: float, zc: float) -> float:
    """Sagitta factor K_x1 of PAPER.md:215-219 for the TOY field, closed form (C5).

    For x(z) = x_m + tx'(z - z_mag) + c2*dtx*(z - z0)^2 and a track from the origin the chord
    through layers a, c misses layer b by -c2*dtx*(zb-za)*(zc-zb) while the chord's intercept at
    z = 0 is -dtx*(z_mag - c2*(z0^2 - za*zc)); K - 1 is the ratio of the two.
    """
    return 1.0 + TOY_C2 * (zb - za) * (zc - zb) / (TOY_Z_MAG - TOY_C2 * (TOY_Z0 ** 2 - za * zc))


def toy_geometry(polarity: int = 1, kick_sign: float = 1.0) -> Dict[str, object]:
    """Plain-value description of the TOY geometry (fields of ``lf_geometry``).  ``kick_sign = -1`` is the magnet with
    the field reversed (particles bend the other way; generate the events with ``GenConfig.kick_sign = -1``)."""
    z = TOY_Z
    kick = math.copysign(TOY_KICK, kick_sign)
    return {
        "n_layers": N_LAYERS,
        "z": list(z),
        "tan_alpha": list(TOY_TAN),
        "z_seed": TOY_Z_SEED,
        "z_mag": TOY_Z_MAG,
        "kick": kick,
        "z_ref": TOY_Z_REF,
        "d_ratio": 0.0,
        "k_first": _toy_k(z[0], z[4], z[8]),
        "k_last": _toy_k(z[3], z[7], z[11]),
        # Eq. (9) reduced to a constant (C18): slope at z_ref includes the quadratic term
        "qop_poly": [kick * (1.0 + 2.0 * TOY_C2 * (TOY_Z_REF - TOY_Z0)), 0.0, 0.0, 0.0, 0.0],
        # full Eq. (9): coefficients of dSlope^i as 2-D polynomials in the seed slopes; inactive
        # while qop_mode == 0.  `momentum_fit.fit_qop_poly2d` produces them from toy tracks.
        "qop_mode": 0,
        "qop_poly2d": [[0.0] * 10 for _ in range(5)],
        "x_half": TOY_X_HALF,
        "y_half": TOY_Y_HALF,
        "z_state": z[11],
        "polarity": int(polarity),
    }


def default_params() -> Dict[str, object]:
    """Table 3 "Forward" column + Table 4 + the DESIGN.md readings."""
    return {
        "T_triplet": 8.0, "T_x": 2.0, "T_uv_slope": 50.0, "T_uv_min": 0.5,
        "T_ty": 0.02, "T_y": 800.0, "T_Q": 0.5,
        "C_nhits": [5.0, 1.0, 0.8, 0.5],
        "n_window": 32, "n_triplets": 12, "min_hits": 9,
        "xtol_base": 150.0, "xtol_inv_p": 2000.0, "x_asym": 100.0, "uv_half_width": 800.0,
        "p_same_bend": 5.0, "mag_tol_base": 8.0, "mag_tol_inv_p": 60.0, "mag_tol_tx": 20.0,
        "mag_tol_max": 40.0,
        "hit_storage": 0,
        # no-UT tuning; inactive while mode == 0
        "mode": 0, "velo_p_min": 5.0, "velo_pt_min": 1.0,
        "xtol_poly": [4824.3, 426.3, 7071.1, 12080.4, 14077.8, 13909.3, 9315.3, 3209.5],  # Table 5
        "x_overlap": 5.0,
        "seed_arith": 1,  # hit_storage = 1 only: 1 = fp32 per doublet on the decoded fp16 hits (default: the faster one, DESIGN.md
                          # section 7b), 0 = pairs of doublets in __half2 (kept as the comparison)
    }


def no_ut_params() -> Dict[str, object]:
    """Table 3 "Forward no-UT" column + section VI.E: VELO seeds without
    momentum, double-sided windows of Eq. (7)/(8) with Table 5, u/v tolerance 1200 mm, 64 hits per window,
    20 triplets, fixed 10 mm tolerance at the magnet, no same-bend filter (N1..N9)."""
    return dict(default_params(), mode=1, T_triplet=2.0, T_x=0.5, T_uv_slope=15.0, T_ty=0.003,
                n_window=64, n_triplets=20, uv_half_width=1200.0,
                p_same_bend=0.0, mag_tol_base=10.0, mag_tol_inv_p=0.0, mag_tol_tx=0.0, mag_tol_max=10.0)


def toy_dtx(tx, ty, qop, field_ax: float = 0.0, field_ay: float = 0.0):
    """Change of the x slope across the magnet.  BASELINE.json's TOY field: kick * q/p.  With a non-uniform field
    (`field_ax`, `field_ay` != 0; stand-in for LHCb's field map) the kick acts on the normalised slope
    as in Eq. (2) with an integrated field that grows with the entry slopes:
    n(t) = t / sqrt(1 + t^2 + ty^2),  n(tx_out) = n(tx_in) + kick * q/p * (1 + ax tx^2 + ay ty^2)."""
    if field_ax == 0.0 and field_ay == 0.0:
        return TOY_KICK * qop
    n_in = tx / np.sqrt(1.0 + tx * tx + ty * ty)
    n_out = n_in + TOY_KICK * qop * (1.0 + field_ax * tx * tx + field_ay * ty * ty)
    n_out = np.clip(n_out, -0.95, 0.95)
    tx_out = n_out * np.sqrt((1.0 + ty * ty) / (1.0 - n_out * n_out))
    return tx_out - tx


def toy_x_at(x_mag, txp, dtx, z):
    """TOY truth x(z) downstream of the magnet (BASELINE.json configs[0])."""
    return x_mag + txp * (z - TOY_Z_MAG) + TOY_C2 * dtx * (z - TOY_Z0) ** 2


def toy_tx_at(txp, dtx, z):
    """TOY truth dx/dz downstream of the magnet."""
    return txp + 2.0 * TOY_C2 * dtx * (z - TOY_Z0)


# ----------------------------------------------------------------------------------------------
# Workload recipes (BASELINE.json configs[0..4])
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class GenConfig:
    name: str
    n_events: int
    seed: int
    true_fixed: Optional[int] = None    # exactly this many true tracks per event ...
    true_mean: float = 0.0              # ... or Poisson(true_mean)
    fake_mean: float = 0.0              # Poisson(fake_mean) fake seeds per event
    noise_fixed: Optional[int] = None   # exactly this many noise hits per layer ...
    noise_mean: float = 0.0             # ... or Poisson(noise_mean) per layer
    p_min: float = 2.0
    p_max: float = 100.0
    smear: float = 0.10                 # Gaussian q/p smear of the seed
    sigma: float = 0.08                 # hit resolution, mm
    eff: float = 0.98                   # per-layer hit efficiency
    zpv_sigma: float = 60.0             # origin spread along z, mm (C20)
    hit_storage: int = 0                # 0 fp32, 1 fp16 storage for windows + seeding
    field_ax: float = 0.0               # non-uniform field (toy_dtx); 0, 0 = BASELINE.json's TOY kick
    field_ay: float = 0.0
    kick_sign: float = 1.0              # -1: reversed field, delta tx = -kick * q/p (pair with toy_geometry(kick_sign=-1))


CONFIGS: Dict[int, GenConfig] = {
    0: GenConfig("cfg0_tiny", 10, 1000, true_fixed=20, noise_fixed=40),
    1: GenConfig("cfg1_run3", 1000, 1001, true_mean=150.0, fake_mean=30.0, noise_mean=274.0),
    2: GenConfig("cfg2_run3_fp16", 1000, 1001, true_mean=150.0, fake_mean=30.0, noise_mean=274.0,
                 hit_storage=1),
    3: GenConfig("cfg3_throughput", 20000, 1003, true_mean=150.0, fake_mean=30.0, noise_mean=274.0),
    4: GenConfig("cfg4_stress", 5000, 1004, true_mean=300.0, fake_mean=60.0, noise_mean=716.0,
                 p_min=1.5, smear=0.25),
}


@dataclass
class Batch:
    """One generated batch in the layout both implementations consume."""
    n_events: int
    seed_x: np.ndarray
    seed_y: np.ndarray
    seed_tx: np.ndarray
    seed_ty: np.ndarray
    seed_qop: np.ndarray
    seed_offsets: np.ndarray      # uint32 [n_events+1]
    hit_x: np.ndarray             # float32 [n_hits]
    seg_offsets: np.ndarray       # uint32 [n_events*24+1]
    hit_track: np.ndarray         # int32 [n_hits]   truth: track id or -1
    seed_track: np.ndarray        # int32 [n_seeds]  truth: track id or -1
    trk_event: np.ndarray         # int32 [n_tracks]
    trk_x: np.ndarray             # float64 true state at z_seed
    trk_y: np.ndarray
    trk_tx: np.ndarray
    trk_ty: np.ndarray
    trk_qop: np.ndarray
    config: Optional[GenConfig] = None

    @property
    def n_seeds(self) -> int:
        return int(self.seed_x.shape[0])

    @property
    def n_hits(self) -> int:
        return int(self.hit_x.shape[0])

    @property
    def n_tracks(self) -> int:
        return int(self.trk_event.shape[0])

    def input_bytes(self) -> int:
        """Bytes of the algorithm's inputs (seeds, hits, both offset tables)."""
        return int(5 * 4 * self.n_seeds + 4 * self.n_hits
                   + self.seed_offsets.nbytes + self.seg_offsets.nbytes)

    def slice_events(self, e0: int, e1: int) -> "Batch":
        """Events [e0, e1) as an independent batch (offsets rebased; truth ids kept global)."""
        s0, s1 = int(self.seed_offsets[e0]), int(self.seed_offsets[e1])
        h0, h1 = int(self.seg_offsets[e0 * N_SEGS]), int(self.seg_offsets[e1 * N_SEGS])
        tsel = (self.trk_event >= e0) & (self.trk_event < e1)
        return Batch(
            n_events=e1 - e0,
            seed_x=self.seed_x[s0:s1], seed_y=self.seed_y[s0:s1], seed_tx=self.seed_tx[s0:s1],
            seed_ty=self.seed_ty[s0:s1], seed_qop=self.seed_qop[s0:s1],
            seed_offsets=(self.seed_offsets[e0:e1 + 1] - np.uint32(s0)).astype(np.uint32),
            hit_x=self.hit_x[h0:h1],
            seg_offsets=(self.seg_offsets[e0 * N_SEGS:e1 * N_SEGS + 1] - np.uint32(h0)).astype(np.uint32),
            hit_track=self.hit_track[h0:h1], seed_track=self.seed_track[s0:s1],
            trk_event=self.trk_event[tsel] - e0, trk_x=self.trk_x[tsel], trk_y=self.trk_y[tsel],
            trk_tx=self.trk_tx[tsel], trk_ty=self.trk_ty[tsel], trk_qop=self.trk_qop[tsel],
            config=self.config,
        )


# ----------------------------------------------------------------------------------------------
# Generation
# ----------------------------------------------------------------------------------------------
@dataclass
class _Chunk:
    n_events: int
    seeds: np.ndarray        # float32 [5, n_seeds]
    seed_counts: np.ndarray  # int64 [n_events]
    seed_track: np.ndarray   # int64 local track id or -1
    hit_x: np.ndarray
    seg_counts: np.ndarray   # int64 [n_events*24]
    hit_track: np.ndarray    # int64 local track id or -1
    trk: np.ndarray          # float64 [5, n_tracks]
    trk_event: np.ndarray    # int64 local event


def _gen_chunk(cfg: GenConfig, chunk_idx: int, n_ev: int) -> _Chunk:
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed, chunk_idx])))
    z = np.asarray(TOY_Z)
    tana = np.asarray(TOY_TAN)

    # --- multiplicities -----------------------------------------------------------------------
    if cfg.true_fixed is not None:
        n_true = np.full(n_ev, cfg.true_fixed, dtype=np.int64)
    else:
        n_true = rng.poisson(cfg.true_mean, n_ev).astype(np.int64)
    n_fake = rng.poisson(cfg.fake_mean, n_ev).astype(np.int64) if cfg.fake_mean > 0 else np.zeros(n_ev, np.int64)
    if cfg.noise_fixed is not None:
        n_noise = np.full((n_ev, N_LAYERS), cfg.noise_fixed, dtype=np.int64)
    else:
        n_noise = rng.poisson(cfg.noise_mean, (n_ev, N_LAYERS)).astype(np.int64)

    def states(n):
        p = np.exp(rng.uniform(math.log(cfg.p_min), math.log(cfg.p_max), n))
        q = rng.integers(0, 2, n) * 2.0 - 1.0
        tx = rng.uniform(-0.25, 0.25, n)
        ty = rng.uniform(-0.2, 0.2, n)
        zpv = rng.normal(0.0, cfg.zpv_sigma, n)
        x = tx * (TOY_Z_SEED - zpv)
        y = ty * (TOY_Z_SEED - zpv)
        return x, y, tx, ty, q / p

    # --- true tracks and their hits -----------------------------------------------------------
    nt = int(n_true.sum())
    trk_event = np.repeat(np.arange(n_ev, dtype=np.int64), n_true)
    x, y, tx, ty, qop = states(nt)
    x_mag = x + tx * (TOY_Z_MAG - TOY_Z_SEED)
    dtx = cfg.kick_sign * toy_dtx(tx, ty, qop, cfg.field_ax, cfg.field_ay)
    txp = tx + dtx
    xt = toy_x_at(x_mag[:, None], txp[:, None], dtx[:, None], z[None, :])
    yt = y[:, None] + ty[:, None] * (z[None, :] - TOY_Z_SEED)
    meas = xt + yt * tana[None, :] + cfg.sigma * rng.normal(0.0, 1.0, (nt, N_LAYERS))
    keep = (np.abs(xt) < TOY_X_HALF) & (np.abs(yt) < TOY_Y_HALF) & (rng.uniform(0.0, 1.0, (nt, N_LAYERS)) < cfg.eff)
    ti, li = np.nonzero(keep)
    th_x = meas[ti, li]
    th_zone = (yt[ti, li] >= 0.0).astype(np.int64)
    th_seg = trk_event[ti] * N_SEGS + li * N_ZONES + th_zone

    # --- noise hits ---------------------------------------------------------------------------
    nn = int(n_noise.sum())
    flat = n_noise.reshape(-1)
    nz_el = np.repeat(np.arange(n_ev * N_LAYERS, dtype=np.int64), flat)  # event*12 + layer
    nz_x = rng.uniform(-TOY_X_HALF, TOY_X_HALF, nn)
    nz_zone = rng.integers(0, 2, nn).astype(np.int64)
    nz_seg = nz_el * N_ZONES + nz_zone

    hx = np.concatenate([th_x, nz_x]).astype(np.float32)
    hseg = np.concatenate([th_seg, nz_seg])
    htrk = np.concatenate([ti.astype(np.int64), np.full(nn, -1, dtype=np.int64)])
    order = np.lexsort((hx, hseg))
    hx, hseg, htrk = hx[order], hseg[order], htrk[order]
    seg_counts = np.bincount(hseg, minlength=n_ev * N_SEGS).astype(np.int64)

    # --- seeds: smeared true states + fake states, shuffled per event -------------------------
    fac = np.maximum(0.25, 1.0 + cfg.smear * rng.normal(0.0, 1.0, nt))
    nf = int(n_fake.sum())
    fx, fy, ftx, fty, fqop = states(nf)
    f_event = np.repeat(np.arange(n_ev, dtype=np.int64), n_fake)
    s_all = np.stack([np.concatenate([x, fx]), np.concatenate([y, fy]), np.concatenate([tx, ftx]),
                      np.concatenate([ty, fty]), np.concatenate([qop * fac, fqop])])
    s_event = np.concatenate([trk_event, f_event])
    s_trk = np.concatenate([np.arange(nt, dtype=np.int64), np.full(nf, -1, dtype=np.int64)])
    key = rng.uniform(0.0, 1.0, nt + nf)
    sorder = np.lexsort((key, s_event))
    return _Chunk(
        n_events=n_ev,
        seeds=s_all[:, sorder].astype(np.float32),
        seed_counts=(n_true + n_fake),
        seed_track=s_trk[sorder],
        hit_x=hx, seg_counts=seg_counts, hit_track=htrk,
        trk=np.stack([x, y, tx, ty, qop]), trk_event=trk_event,
    )


def generate(cfg: GenConfig, n_events: Optional[int] = None, workers: Optional[int] = None) -> Batch:
    """Generate ``n_events`` (default ``cfg.n_events``) events of recipe ``cfg``."""
    n_events = cfg.n_events if n_events is None else int(n_events)
    sizes: List[int] = []
    left = n_events
    while left > 0:
        sizes.append(min(CHUNK_EVENTS, left))
        left -= sizes[-1]
    workers = workers or min(len(sizes), os.cpu_count() or 1) or 1
    if len(sizes) <= 1 or workers <= 1:
        chunks = [_gen_chunk(cfg, k, n) for k, n in enumerate(sizes)]
    else:
        with ThreadPoolExecutor(max_workers=workers) as pool:
            chunks = list(pool.map(lambda a: _gen_chunk(cfg, a[0], a[1]), enumerate(sizes)))

    def cat(arrs, dtype):
        return np.concatenate(arrs).astype(dtype, copy=False) if arrs else np.zeros(0, dtype)

    trk_base = np.cumsum([0] + [c.trk.shape[1] for c in chunks])
    ev_base = np.cumsum([0] + [c.n_events for c in chunks])
    seeds = np.concatenate([c.seeds for c in chunks], axis=1) if chunks else np.zeros((5, 0), np.float32)
    seed_counts = cat([c.seed_counts for c in chunks], np.int64)
    seg_counts = cat([c.seg_counts for c in chunks], np.int64)
    seed_offsets = np.zeros(n_events + 1, dtype=np.uint32)
    seed_offsets[1:] = np.cumsum(seed_counts)
    seg_offsets = np.zeros(n_events * N_SEGS + 1, dtype=np.uint32)
    seg_offsets[1:] = np.cumsum(seg_counts)
    trk = np.concatenate([c.trk for c in chunks], axis=1) if chunks else np.zeros((5, 0))
    return Batch(
        n_events=n_events,
        seed_x=np.ascontiguousarray(seeds[0]), seed_y=np.ascontiguousarray(seeds[1]),
        seed_tx=np.ascontiguousarray(seeds[2]), seed_ty=np.ascontiguousarray(seeds[3]),
        seed_qop=np.ascontiguousarray(seeds[4]),
        seed_offsets=seed_offsets,
        hit_x=cat([c.hit_x for c in chunks], np.float32),
        seg_offsets=seg_offsets,
        hit_track=cat([np.where(c.hit_track >= 0, c.hit_track + trk_base[k], -1) for k, c in enumerate(chunks)], np.int32),
        seed_track=cat([np.where(c.seed_track >= 0, c.seed_track + trk_base[k], -1) for k, c in enumerate(chunks)], np.int32),
        trk_event=cat([c.trk_event + ev_base[k] for k, c in enumerate(chunks)], np.int32),
        trk_x=trk[0].copy(), trk_y=trk[1].copy(), trk_tx=trk[2].copy(), trk_ty=trk[3].copy(), trk_qop=trk[4].copy(),
        config=cfg,
    )


def generate_config(config_id: int, n_events: Optional[int] = None, workers: Optional[int] = None) -> Batch:
    return generate(CONFIGS[config_id], n_events=n_events, workers=workers)


def single_track_config(n_events: int, seed: int, sigma: float = 0.0, smear: float = 0.0,
                        p_min: float = 2.0, p_max: float = 100.0) -> GenConfig:
    """Noise-free, fully efficient, one true track per event (truth pins; SURVEY §8(c) pin 2)."""
    return GenConfig("single_track", n_events, seed, true_fixed=1, noise_fixed=0, sigma=sigma,
                     eff=2.0, smear=smear, p_min=p_min, p_max=p_max)


def with_overrides(cfg: GenConfig, **kw) -> GenConfig:
    return replace(cfg, **kw)
