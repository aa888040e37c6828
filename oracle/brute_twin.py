"""Brute-force twin of the oracle (TEST INFRASTRUCTURE ONLY; pin 1 of DESIGN.md "Pins").

A second, independent statement of the algorithm written from the *definitions*, in float64,
for tiny events only (pure-Python loops):

* window membership by testing every hit of the segment (no sortedness, no binary search);
  the n_window cap by ranking the members and keeping ranks within n_window/2 of the centre's rank;
* every (h0, h2) pair of the two windows; closest hit by a linear ``min``; top-n by a full sort;
* the triplet parabola by ``numpy.linalg.solve`` on the 3x3 system in millimetres;
* the x fit and the y fit by ``numpy.linalg.lstsq`` directly on the measurements
  (m_i = s_i - y_i tan(alpha_i) against [1, dz, dz^2 (1 + dRatio dz)]; y_i = (s_i - x_fit)/tan(alpha_i)
  against [1, dz]) -- not the residual / cofactor form the oracle uses.

It is compared with the **fp64 build** of the oracle (same decisions up to 1e-9-level ties), which in
turn is compared with the fp32 reference build.  Citations as in lf_oracle.cpp.
"""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np

NL = 12
SETS = ((0, 4, 8), (3, 7, 11))


def _is_uv(l: int) -> bool:
    return (l & 3) in (1, 2)


def run(G: dict, P: dict, b) -> SimpleNamespace:
    z = np.asarray(G["z"], dtype=np.float64)
    # the oracle receives float32 geometry; mirror the *inputs*, not the arithmetic
    z = np.asarray(np.float32(z), dtype=np.float64)
    tana = np.asarray(np.float32(np.asarray(G["tan_alpha"])), dtype=np.float64)
    f = lambda v: float(np.float32(v))
    z_seed, z_mag, kick, z_ref, d_ratio = f(G["z_seed"]), f(G["z_mag"]), f(G["kick"]), f(G["z_ref"]), f(G["d_ratio"])
    K = (f(G["k_first"]), f(G["k_last"]))
    poly = [f(c) for c in G["qop_poly"]]
    qop_mode = int(G.get("qop_mode", 0))
    poly2d = [[f(c) for c in row] for row in G.get("qop_poly2d", [[0.0] * 10] * 5)]
    # Eq. (9): exponents (k, m) of tx^k ty^m allowed by the field symmetries, k + m <= 6
    even_terms = [(k, m) for d in (0, 2, 4, 6) for k in range(d, -1, -2) for m in [d - k]]
    odd_terms = [(k, m) for d in (1, 3, 5) for k in range(d, 0, -2) for m in [d - k]]
    z_state = f(G["z_state"])
    pol = int(G["polarity"])
    hx = np.asarray(b.hit_x, dtype=np.float64)
    seg = np.asarray(b.seg_offsets, dtype=np.int64)
    so = np.asarray(b.seed_offsets, dtype=np.int64)
    n_window, n_trip, min_hits = int(P["n_window"]), int(P["n_triplets"]), int(P["min_hits"])
    pf = {k: (f(v) if not isinstance(v, (list, tuple)) else [f(t) for t in v]) for k, v in P.items()
          if k not in ("n_window", "n_triplets", "min_hits", "hit_storage", "mode")}
    mode = int(P.get("mode", 0))
    n_sides = 2 if mode == 1 else 1  # no-UT: LEFT and RIGHT windows of Eq. (8), followed separately

    def basis(zz):
        dz = zz - z_ref
        return np.array([1.0, dz, dz * dz * (1.0 + d_ratio * dz)])

    def dbasis(zz):
        dz = zz - z_ref
        return np.array([0.0, 1.0, 2.0 * dz + 3.0 * d_ratio * dz * dz])

    tracks = []
    win_first = np.zeros((b.seed_x.shape[0] * n_sides, NL), np.int64)
    win_count = np.zeros((b.seed_x.shape[0] * n_sides, NL), np.int64)
    all_trips = []
    ev_off = [0]
    for ev in range(b.n_events):
        for si in range(so[ev], so[ev + 1]):
            x, y, tx, ty = float(b.seed_x[si]), float(b.seed_y[si]), float(b.seed_tx[si]), float(b.seed_ty[si])
            qop = float(b.seed_qop[si]) if mode == 0 else 0.0
            x_mag = x + tx * (z_mag - z_seed)
            zone = 1 if ty >= 0 else 0
            yl = y + ty * (z - z_seed)
            best = None
            for side in range(n_sides):
              row = si * n_sides + side
              if mode == 0:
                aq = max(abs(qop), 1e-6)
                p = 1.0 / aq
                txp = tx + kick * qop
                x_tol = pf["xtol_base"] + pf["xtol_inv_p"] / p
                q = 1 if qop > 0 else -1
                a_left = pf["x_asym"] if q * pol > 0 else 0.0
                a_right = pf["x_asym"] if q * pol < 0 else 0.0
              else:
                # assumed momentum = the tighter of p_min and pT_min / sin(theta)
                slope2 = tx * tx + ty * ty
                p = pf["velo_p_min"]
                if slope2 > 0.0:
                    p = max(p, pf["velo_pt_min"] * np.sqrt(1.0 + slope2) / np.sqrt(slope2))
                else:
                    p = np.inf
                ip = 1.0 / p
                c = pf["xtol_poly"]
                # Eq. (7), term by term as printed
                x_tol = ip * (c[0] + c[1] * tx + c[2] * tx ** 2 + ty ** 2 * (c[3] + c[4] * tx + c[5] * tx ** 2)
                              + ip * (c[6] * tx + c[7] * ip))
              windows = []
              for l in range(NL):
                if mode == 0:
                    xc = x_mag + txp * (z[l] - z_mag)
                    if _is_uv(l):
                        ctr = xc + yl[l] * tana[l]
                        lo, hi = ctr - pf["uv_half_width"], ctr + pf["uv_half_width"]
                    else:
                        lo, hi = xc - x_tol - a_left, xc + x_tol + a_right
                else:
                    # Eq. (8) about the straight-line extrapolation
                    ctr = x + tx * (z[l] - z_seed) + (yl[l] * tana[l] if _is_uv(l) else 0.0)
                    tol = pf["uv_half_width"] if _is_uv(l) else x_tol
                    lo, hi = ((ctr - tol, ctr + pf["x_overlap"]) if side == 0 else (ctr - pf["x_overlap"], ctr + tol))
                s0, s1 = seg[ev * 24 + l * 2 + zone], seg[ev * 24 + l * 2 + zone + 1]
                members = [i for i in range(s0, s1) if lo <= hx[i] <= hi]
                members.sort(key=lambda i: (hx[i], i))
                if len(members) > n_window:
                    mid = 0.5 * (lo + hi)
                    c_rank = sum(1 for i in members if hx[i] < mid)
                    members = [i for r, i in enumerate(members) if c_rank - n_window // 2 <= r < c_rank + n_window // 2]
                windows.append(members)
                win_count[row, l] = len(members)
                win_first[row, l] = members[0] if members else -1
              # ---- seeding
              trips = []
              for s, (la, lb, lc) in enumerate(SETS):
                  for i0 in windows[la]:
                      for i2 in windows[lc]:
                          t = (hx[i2] - hx[i0]) / (z[lc] - z[la])
                          if mode == 0 and p < pf["p_same_bend"] and not ((t - tx) * (kick * qop) > 0):
                              continue
                          tol = min(pf["mag_tol_max"], pf["mag_tol_base"] + pf["mag_tol_inv_p"] / p + pf["mag_tol_tx"] * abs(t))
                          if not abs(hx[i0] + t * (z_mag - z[la]) - x_mag) < tol:
                              continue
                          if not windows[lb]:
                              continue
                          x1e = z[lb] * t + (hx[i0] - t * z[la]) * K[s]
                          i1 = min(windows[lb], key=lambda i: (abs(hx[i] - x1e), i))
                          chi2 = (hx[i1] - x1e) ** 2
                          if chi2 < pf["T_triplet"]:
                              trips.append((chi2, s, i0, i2, i1))
              trips.sort()
              trips = trips[:n_trip]
              all_trips.append(trips)
              # ---- extension + fit
              T_uv = max(pf["T_uv_min"], pf["T_uv_slope"] * (abs(tx) + abs(ty)))
              for (chi2_t, s, i0, i2, i1) in trips:
                  la, lb, lc = SETS[s]
                  A3 = np.array([basis(z[la]), basis(z[lb]), basis(z[lc])])
                  par0 = np.linalg.solve(A3, np.array([hx[i0], hx[i1], hx[i2]]))
                  hit = [-1] * NL
                  hit[la], hit[lb], hit[lc] = i0, i1, i2
                  for l in range(NL):
                      if l in (la, lb, lc) or not windows[l]:
                          continue
                      pred = float(basis(z[l]) @ par0) + (yl[l] * tana[l] if _is_uv(l) else 0.0)
                      k = min(windows[l], key=lambda i: (abs(hx[i] - pred), i))
                      if (hx[k] - pred) ** 2 < (T_uv if _is_uv(l) else pf["T_x"]):
                          hit[l] = k
                  layers = [l for l in range(NL) if hit[l] >= 0]
                  uv = [l for l in layers if _is_uv(l)]
                  n, n_uv = len(layers), len(uv)
                  if n < min_hits or any(not any((l >> 2) == st for l in uv) for st in range(3)):
                      continue
                  A = np.array([basis(z[l]) for l in layers])
                  m = np.array([hx[hit[l]] - yl[l] * tana[l] for l in layers])
                  par, *_ = np.linalg.lstsq(A, m, rcond=None)
                  res = m - A @ par
                  Qx = sum(res[j] ** 2 / (T_uv if _is_uv(l) else pf["T_x"]) for j, l in enumerate(layers))
                  Ay = np.array([[1.0, z[l] - z_ref] for l in uv])
                  yi = np.array([(hx[hit[l]] - float(basis(z[l]) @ par)) / tana[l] for l in uv])
                  ypar, *_ = np.linalg.lstsq(Ay, yi, rcond=None)
                  # seed line in the same parameterisation: y(z) = y + ty (z - z_seed)
                  ty_fit = ypar[1]
                  if not abs(ty_fit - ty) < pf["T_ty"]:
                      continue
                  Qy = float(np.sum((yi - Ay @ ypar) ** 2)) / pf["T_y"]
                  Q = (Qx / (n - 3) + Qy / (n_uv - 2)) * pf["C_nhits"][min(3, max(0, n - 9))]
                  if not Q < pf["T_Q"]:
                      continue
                  if best is None or Q < best[0]:
                      dslope = par[1] - tx
                      if qop_mode == 0:
                          coef = poly
                      else:
                          coef = [sum(a * tx ** k * ty ** m for a, (k, m) in zip(poly2d[i], even_terms if i % 2 == 0 else odd_terms))
                                  for i in range(5)]
                      F = sum(c * dslope ** k for k, c in enumerate(coef))
                      state = [float(basis(z_state) @ par), ypar[0] + ypar[1] * (z_state - z_ref),
                               float(dbasis(z_state) @ par), ty_fit, dslope / F]
                      best = (Q, hit, n, state)
            if best is not None:
                tracks.append((si, best[1], best[2], best[3], best[0]))
        ev_off.append(len(tracks))
    n = len(tracks)
    return SimpleNamespace(
        n_tracks=n,
        seed_idx=np.array([t[0] for t in tracks], np.int32),
        hit_idx=np.array([t[1] for t in tracks], np.int32).reshape(n, NL),
        n_hits=np.array([t[2] for t in tracks], np.int32),
        state=np.array([t[3] for t in tracks], np.float64).reshape(n, 5),
        quality=np.array([t[4] for t in tracks], np.float64),
        event_offsets=np.array(ev_off, np.uint32),
        win_first=win_first, win_count=win_count, triplets=all_trips)
