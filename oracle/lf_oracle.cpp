/*
 * lf_oracle.cpp -- CPU ORACLE of the Looking Forward hot path (arxiv 2402.14670).
 *
 * TEST INFRASTRUCTURE ONLY (see lf_oracle.h).  Plain single-threaded C++17, no blocking, no
 * fusion, no early exits beyond what the paper's algorithm states.  The method is a heuristic
 * search, so the oracle follows the algorithm step by step in the paper's order:
 *
 *   O1 extrapolate      PAPER.md:167-179  (pT-kick from the magnet centre)
 *   O2 search windows   PAPER.md:165, 181-204 (zone from t_y, Eq. 3, +-800 mm u/v, n_window cap)
 *   O3 triplet seeding
 *   O4 x extension      PAPER.md:227-232 (Eq. 4)
 *   O5 u/v extension
 *   O6 fit + quality    PAPER.md:238-279 (Eq. 5, 6, Table 4)
 *   O7 momentum, state  PAPER.md:327-338 (Eq. 9), 388
 *   no-UT tuning        PAPER.md:285-325 (Eq. 7, 8, Table 5): params.mode == 1 replaces O1/O2 by a
 *                       straight-line extrapolation with double-sided windows and follows each window
 *                       side (charge assumption) separately through O3..O6 (N1..N9)
 *
 * Arithmetic: every floating-point operation is done in `Real` (float in the reference build,
 * double in the pin build) in exactly the order written below, one rounding per operation
 * (build with -ffp-contract=off, no fast-math).  DESIGN.md "Canonical arithmetic" lists the
 * same expressions; the CUDA path restates them independently.
 */
#include "lf_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

#ifndef LF_ORACLE_REAL
#define LF_ORACLE_REAL float
#endif
typedef LF_ORACLE_REAL Real;

namespace {

const int NL = LFO_N_LAYERS;
const int NSEG = 2 * NL;
/* x-layer sets used for seeding: first / last x layer of each T-station. */
const int SETS[2][3] = {{0, 4, 8}, {3, 7, 11}};

inline Real RC(double v) { return static_cast<Real>(v); }
inline Real rabs(Real v) { return v < 0 ? -v : v; }
inline bool is_uv(int l) { return (l & 3) == 1 || (l & 3) == 2; } /* x-u-v-x */

/* Constants derived from the geometry, each computed once in Real, in this order. */
struct Geo {
  Real z[NL], tana[NL], inv_tan[NL];
  Real dzs[NL];  /* z_l - z_seed */
  Real dzm[NL];  /* z_l - z_mag  */
  Real d[NL];    /* (z_l - z_ref) in metres: Eq. (4) dz, scaled for fp32 conditioning (C14) */
  Real w[NL];    /* d^2 (1 + dRatio d): the curvature basis function of Eq. (1)/(4) */
  Real z_seed, z_mag, kick, dr, K[2], poly[5];
  Real mag_dz_seed;                     /* z_mag - z_seed */
  Real inv_dz_ac[2], zmag_a[2];         /* per layer set: 1/(z_c - z_a), z_mag - z_a */
  Real D10[2], D20[2], W10[2], W20[2], inv_det[2], inv_D10[2]; /* 3-point solve (C11) */
  Real dz_state, ds, ws, dws;           /* output state plane (C19) */
  int polarity;
  int qop_mode;
  Real poly2d[5][10];
};

Geo make_geo(const lfo_geometry& G) {
  Geo g;
  g.z_seed = G.z_seed; g.z_mag = G.z_mag; g.kick = G.kick;
  g.dr = Real(G.d_ratio) * RC(1000.0);   /* dRatio per metre */
  g.K[0] = G.k_first; g.K[1] = G.k_last;
  for (int i = 0; i < 5; ++i) g.poly[i] = G.qop_poly[i];
  g.polarity = G.polarity;
  g.qop_mode = G.qop_mode;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 10; ++j) g.poly2d[i][j] = G.qop_poly2d[i][j];
  g.mag_dz_seed = g.z_mag - g.z_seed;
  for (int l = 0; l < NL; ++l) {
    g.z[l] = G.z[l];
    g.tana[l] = G.tan_alpha[l];
    g.inv_tan[l] = is_uv(l) ? RC(1.0) / g.tana[l] : RC(0.0);
    g.dzs[l] = g.z[l] - g.z_seed;
    g.dzm[l] = g.z[l] - g.z_mag;
    g.d[l] = (g.z[l] - Real(G.z_ref)) * RC(0.001);
    g.w[l] = (g.d[l] * g.d[l]) * (RC(1.0) + g.dr * g.d[l]);
  }
  for (int s = 0; s < 2; ++s) {
    const int a = SETS[s][0], b = SETS[s][1], c = SETS[s][2];
    g.inv_dz_ac[s] = RC(1.0) / (g.z[c] - g.z[a]);
    g.zmag_a[s] = g.z_mag - g.z[a];
    g.D10[s] = g.d[b] - g.d[a];
    g.D20[s] = g.d[c] - g.d[a];
    g.W10[s] = g.w[b] - g.w[a];
    g.W20[s] = g.w[c] - g.w[a];
    g.inv_det[s] = RC(1.0) / (g.W20[s] * g.D10[s] - g.W10[s] * g.D20[s]);
    g.inv_D10[s] = RC(1.0) / g.D10[s];
  }
  g.dz_state = Real(G.z_state) - g.z_seed;
  g.ds = (Real(G.z_state) - Real(G.z_ref)) * RC(0.001);
  g.ws = (g.ds * g.ds) * (RC(1.0) + g.dr * g.ds);
  g.dws = RC(2.0) * g.ds + (RC(3.0) * g.dr) * (g.ds * g.ds);  /* dw/dd at the state plane */
  return g;
}

struct Window { int first; int count; };           /* global hit indices [first, first+count) */
struct Triplet { Real chi2; int set, i0, i1, i2; }; /* global hit indices */

/* C9 order: (chi2, set, i0, i2) ascending. */
bool triplet_before(const Triplet& a, const Triplet& b) {
  if (a.chi2 != b.chi2) return a.chi2 < b.chi2;
  if (a.set != b.set) return a.set < b.set;
  if (a.i0 != b.i0) return a.i0 < b.i0;
  return a.i2 < b.i2;
}

/* First i in [b, e) with x[i] >= v / with x[i] > v. */
int lower_idx(const float* x, int b, int e, Real v) {
  int i = b;
  while (i < e && Real(x[i]) < v) ++i;
  return i;
}
int upper_idx(const float* x, int b, int e, Real v) {
  int i = b;
  while (i < e && !(v < Real(x[i]))) ++i;
  return i;
}

/* Hit of the window whose x is closest to `pred`; ties -> lower index (C15).  -1 if empty. */
int closest_idx(const float* x, const Window& wdw, Real pred) {
  int best = -1;
  Real best_d = 0;
  for (int i = wdw.first; i < wdw.first + wdw.count; ++i) {
    const Real dist = rabs(Real(x[i]) - pred);
    if (best < 0 || dist < best_d) { best = i; best_d = dist; }
  }
  return best;
}

struct SeedState {
  Real x, y, tx, ty, qop;
  Real aq, p, x_mag, txp;  /* mode 1: aq = 1/p of the assumed minimum momentum, qop and txp unused */
  Real yl[NL], yt[NL];  /* y at each layer; y*tan_alpha */
  int zone;
  Window win[NL];
};

/* O1 + O2. */
void extrapolate_and_windows(const Geo& g, const lfo_params& P, const float* hx, const uint32_t* seg,
                             SeedState& s) {
  /* O1: pT-kick extrapolation from the magnet centre. */
  s.aq = std::max(rabs(s.qop), RC(1e-6));
  s.p = RC(1.0) / s.aq;
  s.x_mag = s.x + s.tx * g.mag_dz_seed;
  s.txp = s.tx + g.kick * s.qop;
  /* t_y decides the half (C3). */
  s.zone = (s.ty >= 0) ? 1 : 0;
  /* x_tol = 150 mm + 2000 GeV / p (C1), Eq. (3) asymmetry by charge x polarity. */
  const Real x_tol = Real(P.xtol_base) + Real(P.xtol_inv_p) * s.aq;
  const bool q_pos = s.qop > 0;
  const bool pol_pos = g.polarity > 0;
  const Real a_left = (q_pos == pol_pos) ? Real(P.x_asym) : RC(0.0);
  const Real a_right = (q_pos != pol_pos) ? Real(P.x_asym) : RC(0.0);
  for (int l = 0; l < NL; ++l) {
    const Real xc = s.x_mag + s.txp * g.dzm[l];
    s.yl[l] = s.y + s.ty * g.dzs[l];
    s.yt[l] = is_uv(l) ? s.yl[l] * g.tana[l] : RC(0.0);
    Real lo, hi;
    if (!is_uv(l)) {
      lo = (xc - x_tol) - a_left;
      hi = (xc + x_tol) + a_right;
    } else { /* straight line corrected by the stereo angle, +-800 mm */
      const Real ctr = xc + s.yt[l];
      lo = ctr - Real(P.uv_half_width);
      hi = ctr + Real(P.uv_half_width);
    }
    const int sb = int(seg[l * 2 + s.zone]), se = int(seg[l * 2 + s.zone + 1]);
    int first = lower_idx(hx, sb, se, lo);
    int last = upper_idx(hx, sb, se, hi);
    if (last < first) last = first;
    /* more than n_window hits -> keep those symmetric about the window centre (C4). */
    if (last - first > P.n_window) {
      const Real mid = (lo + hi) * RC(0.5);
      const int c = lower_idx(hx, first, last, mid);
      const int half = P.n_window / 2;
      const int f2 = std::max(first, c - half);
      const int l2 = std::min(last, c + half);
      first = f2; last = l2;
    }
    s.win[l].first = first;
    s.win[l].count = last - first;
  }
}

/* no-UT O1 + O2 for one window side (0 = LEFT, 1 = RIGHT of Eq. 8). */
void velo_windows(const Geo& g, const lfo_params& P, const float* hx, const uint32_t* seg, int side,
                  SeedState& s) {
  /* the momentum is set to the tighter (larger) of p_min and pT_min / sin(theta);
   * as 1/p: min(1/p_min, sin(theta)/pT_min), sin^2(theta) = (tx^2+ty^2)/(1+tx^2+ty^2)  (N2). */
  const Real s2 = s.tx * s.tx + s.ty * s.ty;
  const Real sin_theta = std::sqrt(s2 / (RC(1.0) + s2));
  const Real inv_p = std::min(RC(1.0) / Real(P.velo_p_min), sin_theta * (RC(1.0) / Real(P.velo_pt_min)));
  s.aq = inv_p;
  s.p = RC(1.0) / std::max(inv_p, RC(1e-6));
  s.x_mag = s.x + s.tx * g.mag_dz_seed;
  s.txp = s.tx;
  s.zone = (s.ty >= 0) ? 1 : 0; /* t_y still chooses the half */
  /* Eq. (7) with Table 5. */
  Real c[8];
  for (int i = 0; i < 8; ++i) c[i] = Real(P.xtol_poly[i]);
  const Real x_tol = inv_p * (((c[0] + s.tx * (c[1] + c[2] * s.tx)) +
                               (s.ty * s.ty) * (c[3] + s.tx * (c[4] + c[5] * s.tx))) +
                              inv_p * (c[6] * s.tx + c[7] * inv_p));
  for (int l = 0; l < NL; ++l) {
    /* straight-line extrapolation of the VELO track to the layer */
    const Real xe = s.x + s.tx * g.dzs[l];
    s.yl[l] = s.y + s.ty * g.dzs[l];
    s.yt[l] = is_uv(l) ? s.yl[l] * g.tana[l] : RC(0.0);
    const Real ctr = is_uv(l) ? xe + s.yt[l] : xe;                 /* PAPER.md:321 (as PAPER.md:202) */
    const Real tol = is_uv(l) ? Real(P.uv_half_width) : x_tol;     /* 1200 mm on u/v */
    /* Eq. (8) */
    const Real lo = (side == 0) ? ctr - tol : ctr - Real(P.x_overlap);
    const Real hi = (side == 0) ? ctr + Real(P.x_overlap) : ctr + tol;
    const int sb = int(seg[l * 2 + s.zone]), se = int(seg[l * 2 + s.zone + 1]);
    int first = lower_idx(hx, sb, se, lo);
    int last = upper_idx(hx, sb, se, hi);
    if (last < first) last = first;
    /* at most n_window hits, symmetric about the centre of each window (C4) */
    if (last - first > P.n_window) {
      const Real mid = (lo + hi) * RC(0.5);
      const int cidx = lower_idx(hx, first, last, mid);
      const int half = P.n_window / 2;
      const int f2 = std::max(first, cidx - half);
      const int l2 = std::min(last, cidx + half);
      first = f2; last = l2;
    }
    s.win[l].first = first;
    s.win[l].count = last - first;
  }
}

/* O3: all doublets of both layer sets, two filters, h1 lookup, top n by chi2. */
void triplet_seeding(const Geo& g, const lfo_params& P, const float* hx, const SeedState& s,
                     std::vector<Triplet>& out) {
  out.clear();
  for (int set = 0; set < 2; ++set) {
    const int la = SETS[set][0], lb = SETS[set][1], lc = SETS[set][2];
    const Window &wa = s.win[la], &wb = s.win[lb], &wc = s.win[lc];
    for (int i0 = wa.first; i0 < wa.first + wa.count; ++i0) {
      for (int i2 = wc.first; i2 < wc.first + wc.count; ++i2) {
        const Real x0 = hx[i0], x2 = hx[i2];
        const Real t = (x2 - x0) * g.inv_dz_ac[set];
        /* filter 1 (C7): below 5 GeV the doublet's slope change t - tx must have the sign of the
         * expected kick, delta tx = kick * q/p (Eq. 2) */
        /* (no-UT: the VELO track has no momentum or charge, so the filter does not exist) */
        if (P.mode == 0 && s.p < Real(P.p_same_bend) && !((t - s.tx) * (g.kick * s.qop) > 0)) continue;
        /* filter 2 (C6): opening at the magnet centre */
        const Real x_at_mag = x0 + t * g.zmag_a[set];
        const Real tol = std::min(Real(P.mag_tol_max),
                                  (Real(P.mag_tol_base) + Real(P.mag_tol_inv_p) * s.aq) + Real(P.mag_tol_tx) * rabs(t));
        if (!(rabs(x_at_mag - s.x_mag) < tol)) continue;
        /* x1_expected = z1*t + (x0 - t*z0)*K */
        const Real x1e = g.z[lb] * t + (x0 - t * g.z[la]) * g.K[set];
        const int i1 = closest_idx(hx, wb, x1e);
        if (i1 < 0) continue;
        const Real dx = Real(hx[i1]) - x1e;
        const Real chi2 = dx * dx;
        if (!(chi2 < Real(P.T_triplet))) continue;
        out.push_back(Triplet{chi2, set, i0, i1, i2});
      }
    }
  }
  /* keep the n_triplets smallest chi2 per input track (C9: over both sets). */
  std::sort(out.begin(), out.end(), triplet_before);
  if (int(out.size()) > P.n_triplets) out.resize(P.n_triplets);
}

/* Coefficients c_0..c_4 of Eq. (9) for a seed with slopes (tx, ty): constants, or 2-D
 * polynomials in the slopes with the terms the field symmetries allow (term order: lf_oracle.h). */
void eq9_coefficients(const Geo& g, Real tx, Real ty, Real c[5]) {
  if (g.qop_mode == 0) {
    for (int i = 0; i < 5; ++i) c[i] = g.poly[i];
    return;
  }
  const Real u = tx * tx, v = ty * ty;
  const Real uu = u * u, uv = u * v, vv = v * v;
  const Real mono[10] = {RC(1.0), u, v, uu, uv, vv, uu * u, uu * v, u * vv, vv * v};
  for (int i = 0; i < 5; ++i) {
    const int n_terms = (i % 2 == 0) ? 10 : 6;
    Real acc = g.poly2d[i][0];
    for (int j = 1; j < n_terms; ++j) acc = acc + g.poly2d[i][j] * mono[j];
    c[i] = (i % 2 == 0) ? acc : tx * acc;   /* odd i: tx^(2a+1) ty^(2b) = tx * (tx^2)^a (ty^2)^b */
  }
}

struct Candidate {
  int hit[NL];       /* global hit index per layer or -1 */
  int n, n_uv;
  Real a0, t0, c0;   /* triplet parabola in (d, w) */
  bool enough;       /* hit-count rule */
  bool ty_ok;
  Real Q;
  Real a, t, c, dy0, dtym; /* fitted model */
};

/* O4 + O5: extend the triplet with the parabola through its three hits. */
void extend(const Geo& g, const lfo_params& P, const float* hx, const SeedState& s, const Triplet& tr,
            Candidate& cd) {
  const int set = tr.set;
  const int la = SETS[set][0], lb = SETS[set][1], lc = SETS[set][2];
  for (int l = 0; l < NL; ++l) cd.hit[l] = -1;
  cd.hit[la] = tr.i0; cd.hit[lb] = tr.i1; cd.hit[lc] = tr.i2;
  /* Eq. (4) parameters from the three triplet hits: exact 3-point solve (C11). */
  const Real x0 = hx[tr.i0], x1 = hx[tr.i1], x2 = hx[tr.i2];
  const Real X10 = x1 - x0, X20 = x2 - x0;
  cd.c0 = (X20 * g.D10[set] - X10 * g.D20[set]) * g.inv_det[set];
  cd.t0 = (X10 - cd.c0 * g.W10[set]) * g.inv_D10[set];
  cd.a0 = (x0 - cd.t0 * g.d[la]) - cd.c0 * g.w[la];
  /* u/v tolerance grows with the seed slopes (Table 3; C12). */
  const Real T_uv = std::max(Real(P.T_uv_min), Real(P.T_uv_slope) * (rabs(s.tx) + rabs(s.ty)));
  for (int l = 0; l < NL; ++l) {
    if (l == la || l == lb || l == lc) continue;
    const bool uv = is_uv(l);
    Real pred = (cd.a0 + cd.t0 * g.d[l]) + cd.c0 * g.w[l];
    if (uv) pred = pred + s.yt[l];
    const int k = closest_idx(hx, s.win[l], pred);
    if (k < 0) continue;
    const Real dx = Real(hx[k]) - pred;
    const Real chi2 = dx * dx;
    if (chi2 < (uv ? T_uv : Real(P.T_x))) cd.hit[l] = k;
  }
  cd.n = 0; cd.n_uv = 0;
  bool station_uv[3] = {false, false, false};
  for (int l = 0; l < NL; ++l) {
    if (cd.hit[l] < 0) continue;
    ++cd.n;
    if (is_uv(l)) { ++cd.n_uv; station_uv[l >> 2] = true; }
  }
  /* at least 9 hits, at least one u or v hit per T-station. */
  cd.enough = cd.n >= P.min_hits && station_uv[0] && station_uv[1] && station_uv[2];
}

/* O6: x fit over all hits, y line over u/v hits, quality factor Q. */
void fit_quality(const Geo& g, const lfo_params& P, const float* hx, const SeedState& s, Candidate& cd) {
  const Real T_uv = std::max(Real(P.T_uv_min), Real(P.T_uv_slope) * (rabs(s.tx) + rabs(s.ty)));
  const Real inv_Tx = RC(1.0) / Real(P.T_x);
  const Real inv_Tuv = RC(1.0) / T_uv;
  const Real inv_Ty = RC(1.0) / Real(P.T_y);
  /* Unweighted least squares of (a, t, c) to m_i = s_i - y_i tan(alpha_i) (C13).  The fit is done
   * on the residuals r_i to the triplet parabola (same minimiser; keeps fp32 well conditioned). */
  Real r[NL];
  Real S1 = 0, Sd = 0, Sw = 0, Sdd = 0, Sdw = 0, Sww = 0, Sr = 0, Sdr = 0, Swr = 0;
  for (int l = 0; l < NL; ++l) {
    if (cd.hit[l] < 0) continue;
    const Real m = Real(hx[cd.hit[l]]) - s.yt[l];
    r[l] = m - ((cd.a0 + cd.t0 * g.d[l]) + cd.c0 * g.w[l]);
    S1 = S1 + RC(1.0);
    Sd = Sd + g.d[l];
    Sw = Sw + g.w[l];
    Sdd = Sdd + g.d[l] * g.d[l];
    Sdw = Sdw + g.d[l] * g.w[l];
    Sww = Sww + g.w[l] * g.w[l];
    Sr = Sr + r[l];
    Sdr = Sdr + g.d[l] * r[l];
    Swr = Swr + g.w[l] * r[l];
  }
  /* 3x3 normal equations by cofactors. */
  const Real C00 = Sdd * Sww - Sdw * Sdw;
  const Real C01 = Sdw * Sw - Sd * Sww;
  const Real C02 = Sd * Sdw - Sdd * Sw;
  const Real C11 = S1 * Sww - Sw * Sw;
  const Real C12 = Sd * Sw - S1 * Sdw;
  const Real C22 = S1 * Sdd - Sd * Sd;
  const Real det = (S1 * C00 + Sd * C01) + Sw * C02;
  const Real inv = RC(1.0) / det;
  const Real da = ((C00 * Sr + C01 * Sdr) + C02 * Swr) * inv;
  const Real dt = ((C01 * Sr + C11 * Sdr) + C12 * Swr) * inv;
  const Real dc = ((C02 * Sr + C12 * Sdr) + C22 * Swr) * inv;
  /* chi2 per hit from the fit residuals; Q_x of Eq. (5); y_i of the u/v hits as a residual to the
   * seed's straight line: (s_i - x_fit(z_i))/tan(alpha_i) - y_i = e_i / tan(alpha_i). */
  Real rho[NL];
  Real Qx = 0;
  Real U1 = 0, Ud = 0, Udd = 0, Ur = 0, Udr = 0;
  for (int l = 0; l < NL; ++l) {
    if (cd.hit[l] < 0) continue;
    const Real e = r[l] - ((da + dt * g.d[l]) + dc * g.w[l]);
    const Real chi2 = e * e;
    if (is_uv(l)) {
      Qx = Qx + chi2 * inv_Tuv;
      rho[l] = e * g.inv_tan[l];
      U1 = U1 + RC(1.0);
      Ud = Ud + g.d[l];
      Udd = Udd + g.d[l] * g.d[l];
      Ur = Ur + rho[l];
      Udr = Udr + g.d[l] * rho[l];
    } else {
      Qx = Qx + chi2 * inv_Tx;
    }
  }
  /* linear least-squares fit in y on the u/v hits. */
  const Real det2 = U1 * Udd - Ud * Ud;
  const Real inv2 = RC(1.0) / det2;
  const Real dy0 = (Udd * Ur - Ud * Udr) * inv2;
  const Real dtym = (U1 * Udr - Ud * Ur) * inv2;   /* per metre */
  const Real dty = dtym * RC(0.001);
  /* |t_y(fit) - t_y(seed)| < T_ty */
  cd.ty_ok = rabs(dty) < Real(P.T_ty);
  Real Qy = 0;
  for (int l = 0; l < NL; ++l) {
    if (cd.hit[l] < 0 || !is_uv(l)) continue;
    const Real ey = rho[l] - (dy0 + dtym * g.d[l]);
    Qy = Qy + (ey * ey) * inv_Ty;
  }
  /* Eq. (6) with nDoF_x = n - 3, nDoF_y = n_uv - 2, C(n) of Table 4. */
  const int ci = std::min(3, std::max(0, cd.n - 9));
  cd.Q = (Qx / Real(cd.n - 3) + Qy / Real(cd.n_uv - 2)) * Real(P.C_nhits[ci]);
  cd.a = cd.a0 + da; cd.t = cd.t0 + dt; cd.c = cd.c0 + dc;
  cd.dy0 = dy0; cd.dtym = dtym;
}

} // namespace

extern "C" int lf_oracle_real_bytes(void) { return int(sizeof(Real)); }

extern "C" int lf_oracle_run(const lfo_geometry* G, const lfo_params* P, const lfo_seeds* seeds,
                             const lfo_hits* hits, size_t n_events, lfo_tracks* out, lfo_debug* dbg) {
  if (!G || !P || !seeds || !hits || !out) return 1;
  if (G->n_layers != NL || P->n_window < 2 || P->n_triplets < 1) return 1;
  if (P->mode != 0 && P->mode != 1) return 1;
  if (G->qop_mode != 0 && G->qop_mode != 1) return 1;
  if (P->mode == 0 && !seeds->qop) return 1;
  const int n_sides = (P->mode == 1) ? 2 : 1;
  if (!out->event_offsets || !out->n_tracks) return 1;
  const Geo g = make_geo(*G);
  const float* hx = hits->x;
  const int NT = P->n_triplets;
  std::vector<Triplet> trips;
  size_t n_out = 0;
  out->event_offsets[0] = 0;
  for (size_t ev = 0; ev < n_events; ++ev) {
    const uint32_t* seg = hits->seg_offsets + ev * NSEG;
    for (uint32_t si = seeds->event_offsets[ev]; si < seeds->event_offsets[ev + 1]; ++si) {
      SeedState s;
      s.x = seeds->x[si]; s.y = seeds->y[si]; s.tx = seeds->tx[si]; s.ty = seeds->ty[si];
      s.qop = (P->mode == 0) ? Real(seeds->qop[si]) : RC(0.0);
      /* accept Q < T_Q, keep the lowest Q (C15, C16).  no-UT: each window side (charge
       * assumption) is followed on its own; the lowest Q over both sides is kept (N8). */
      bool have_best = false;
      Candidate best;
      for (int side = 0; side < n_sides; ++side) {
        if (P->mode == 0) extrapolate_and_windows(g, *P, hx, seg, s);
        else velo_windows(g, *P, hx, seg, side, s);
        triplet_seeding(g, *P, hx, s, trips);
        const size_t row = size_t(si) * n_sides + side;
        if (dbg) {
          for (int l = 0; l < NL; ++l) {
            if (dbg->win_first) dbg->win_first[row * NL + l] = s.win[l].first;
            if (dbg->win_count) dbg->win_count[row * NL + l] = s.win[l].count;
          }
          if (dbg->n_triplets) dbg->n_triplets[row] = int(trips.size());
          for (int k = 0; k < NT; ++k) {
            const bool have = k < int(trips.size());
            const size_t o = row * NT + k;
            if (dbg->trip_hits) {
              dbg->trip_hits[o * 3 + 0] = have ? trips[k].i0 : -1;
              dbg->trip_hits[o * 3 + 1] = have ? trips[k].i1 : -1;
              dbg->trip_hits[o * 3 + 2] = have ? trips[k].i2 : -1;
            }
            if (dbg->trip_set) dbg->trip_set[o] = have ? trips[k].set : -1;
            if (dbg->trip_chi2) dbg->trip_chi2[o] = have ? float(trips[k].chi2) : -1.0f;
            if (dbg->cand_quality) dbg->cand_quality[o] = -1.0f;
            if (dbg->cand_hits) for (int l = 0; l < NL; ++l) dbg->cand_hits[o * NL + l] = -1;
          }
        }
        /* O4..O6 for each kept triplet */
        for (int k = 0; k < int(trips.size()); ++k) {
          Candidate cd;
          extend(g, *P, hx, s, trips[k], cd);
          const size_t o = row * NT + k;
          if (dbg && dbg->cand_hits) for (int l = 0; l < NL; ++l) dbg->cand_hits[o * NL + l] = cd.hit[l];
          if (!cd.enough) continue;
          fit_quality(g, *P, hx, s, cd);
          if (dbg && dbg->cand_quality) dbg->cand_quality[o] = cd.ty_ok ? float(cd.Q) : -2.0f;
          if (!cd.ty_ok) continue;
          if (!(cd.Q < Real(P->T_Q))) continue;
          if (!have_best || cd.Q < best.Q) { best = cd; have_best = true; }
        }
      }
      if (!have_best) continue;
      if (n_out >= out->capacity) return 3;
      /* O7: q/p from the slope change, state at z_state. */
      const Real t_ref = best.t * RC(0.001);
      const Real dslope = t_ref - s.tx;
      Real cq[5];
      eq9_coefficients(g, s.tx, s.ty, cq);
      const Real F = cq[0] + dslope * (cq[1] + dslope * (cq[2] + dslope * (cq[3] + dslope * cq[4])));
      const Real qop_out = dslope / F;
      const Real x_out = (best.a + best.t * g.ds) + best.c * g.ws;
      const Real tx_out = (best.t + best.c * g.dws) * RC(0.001);
      const Real y_out = (s.y + s.ty * g.dz_state) + (best.dy0 + best.dtym * g.ds);
      const Real ty_out = s.ty + best.dtym * RC(0.001);
      for (int l = 0; l < NL; ++l) out->hit_idx[n_out * NL + l] = best.hit[l];
      out->seed_idx[n_out] = int32_t(si);
      out->n_hits[n_out] = best.n;
      out->state[n_out * 5 + 0] = float(x_out);
      out->state[n_out * 5 + 1] = float(y_out);
      out->state[n_out * 5 + 2] = float(tx_out);
      out->state[n_out * 5 + 3] = float(ty_out);
      out->state[n_out * 5 + 4] = float(qop_out);
      out->quality[n_out] = float(best.Q);
      ++n_out;
    }
    out->event_offsets[ev + 1] = uint32_t(n_out);
  }
  *out->n_tracks = uint32_t(n_out);
  return 0;
}
