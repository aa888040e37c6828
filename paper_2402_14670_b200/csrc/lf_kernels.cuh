/*
 * lf_kernels.cuh -- sm_100a device code of the Looking Forward hot path (include/lf.h, a1..a7).
 *
 * Execution model:
 *   lf_track_kernel    persistent CTAs take events from an atomic ticket.  The event's 24 x-sorted
 *                      hit segments are contiguous in HBM, so one 1-D bulk async copy (TMA,
 *                      cp.async.bulk + mbarrier) stages the whole event into shared memory; the
 *                      CTA's warps then take seeds from a shared counter, ONE WARP PER SEED:
 *                        a1/a2  lanes 0..23 = (layer, edge): 24 binary searches in parallel;
 *                        a3     lanes = h2 hits of the window, loop over h0; ballot-compacted
 *                               survivors are finished lane-per-doublet (binary-search closest h1);
 *                               top-n by rank selection on 64-bit (chi2, set, h0, h2) keys;
 *                        a4/a5  lanes = (triplet, layer) pairs, binary-search closest hit;
 *                        a6     lanes = candidates, sequential-order fp32 fit (the oracle's
 *                               summation order), warp min-reduce on (Q, order) keys.
 *                      At the end of an event the CTA ranks its found tracks in seed order.
 *   lf_scan_kernel     exclusive scan of the per-event track counts -> event_offsets, n_tracks.
 *   lf_compact_kernel  stream compaction: per-seed records -> dense SoA outputs in (event, seed)
 *                      order, one thread per (seed, word), coalesced.
 *
 * Arithmetic contract: fp32, one rounding per operation, in the order DESIGN.md "Canonical
 * arithmetic" lists (compile with -fmad=false, no fast-math; '/' is IEEE division).  This file is
 * written from PAPER.md + DESIGN.md and shares nothing with oracle/.
 */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lf {

constexpr int NL = 12;
constexpr int NSEG = 24;
constexpr int WARPS_PER_CTA = 8;
constexpr int CTA_THREADS = WARPS_PER_CTA * 32;
constexpr int REC_WORDS = 20;  /* 12 hit idx, seed, n_hits, 5 state, Q */
constexpr int TRIP_BUF = 64;   /* per-warp triplet key buffer */
constexpr int MAX_NT = 16;     /* == LF_MAX_TRIPLETS */
constexpr unsigned FULL = 0xffffffffu;
constexpr unsigned NO_HIT = 0xFFu;

/* Geometry-derived constants and tunables, computed once on the host in fp32 (lf_api.cu). */
struct Consts {
  float z[NL], tana[NL], inv_tan[NL], dzs[NL], dzm[NL], d[NL], w[NL];
  float z_seed, z_mag, kick, dr, K[2], poly[5], mag_dz_seed;
  float inv_dz_ac[2], zmag_a[2], D10[2], D20[2], W10[2], W20[2], inv_det[2], inv_D10[2];
  float dz_state, ds, ws, dws;
  int polarity;
  float T_triplet, T_x, T_uv_slope, T_uv_min, T_ty, inv_Tx, inv_Ty, T_Q, C_nhits[4];
  int n_window, n_triplets, min_hits;
  float xtol_base, xtol_inv_p, x_asym, uv_half_width;
  float p_same_bend, mag_tol_base, mag_tol_inv_p, mag_tol_tx, mag_tol_max;
};

struct DebugOut {
  int32_t *win_first, *win_count, *n_triplets, *trip_hits, *trip_set;
  float* trip_chi2;
  int32_t* cand_hits;
  float* cand_quality;
};

struct TrackArgs {
  const float *sx, *sy, *stx, *sty, *sqop;
  const uint32_t* seed_off;
  const float* hx;
  const uint32_t* seg_off;
  uint32_t n_events;
  int32_t* ws_rec;     /* n_seeds * REC_WORDS */
  int32_t* ws_nh;      /* n_seeds: n_hits of the seed's track, 0 = none */
  int32_t* ws_rank;    /* n_seeds: rank among the event's tracks, -1 = none */
  int32_t* ws_event;   /* n_seeds: event of the seed */
  uint32_t* ev_count;  /* n_events */
  uint32_t* ticket;    /* 1 */
  int stage_cap;       /* floats of shared memory available for one event's hits */
  DebugOut dbg;
};

struct __align__(16) WarpScratch {
  unsigned long long trip[TRIP_BUF];
  uint16_t dq[64];
  uint8_t ext[MAX_NT][16];
  int32_t rec[REC_WORDS];
  int32_t pad[12];
};

struct __align__(16) CtaShared {
  unsigned long long mbar;
  int seg[NSEG + 3];
  int ev, next_seed;
  int warp_tot[WARPS_PER_CTA];
  float g_tana[NL], g_dzs[NL], g_dzm[NL], g_d[NL], g_w[NL];
  WarpScratch ws[WARPS_PER_CTA];
};

/* ---------------------------------------------------------------- PTX helpers (TMA 1-D bulk copy) */
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  uint32_t done = 0;
  const uint32_t a = smem_u32(bar);
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(a), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ bool is_uv(int l) { return ((l & 3) == 1) || ((l & 3) == 2); }

/* The one dynamic shared-memory array of the track kernel: CtaShared, then the staged hits. */
extern __shared__ __align__(16) unsigned char lf_smem[];
constexpr size_t FIXED_SMEM = (sizeof(CtaShared) + 15) & ~size_t(15);
__device__ __forceinline__ float* stage_buf() { return reinterpret_cast<float*>(lf_smem + FIXED_SMEM); }

/* View of the current event's hits, indexed event-relative.  Staged: shared memory (LDS);
 * fallback for events larger than the stage buffer: read-only global loads. */
template <bool STAGED>
struct HitView;
template <>
struct HitView<true> {
  int off; /* skew of the event inside the stage buffer */
  __device__ __forceinline__ float operator[](int i) const { return stage_buf()[off + i]; }
};
template <>
struct HitView<false> {
  const float* p;
  __device__ __forceinline__ float operator[](int i) const { return __ldg(p + i); }
};

/* Closest hit to `pred` in the x-sorted window [f, f+n): binary search for the first x >= pred, then
 * compare the two neighbours; ties -> lower index, including runs of equal distance on the low side
 * (equals a linear argmin with strict '<').  Returns the event-relative index, or -1 if n == 0. */
template <class HV>
__device__ __forceinline__ int closest_hit(const HV& hx, int f, int n, float pred) {
  if (n <= 0) return -1;
  int pos = f, cnt = n;
  while (cnt > 0) {
    const int half = cnt >> 1;
    const int mid = pos + half;
    if (hx[mid] < pred) { pos = mid + 1; cnt -= half + 1; } else { cnt = half; }
  }
  int k;
  if (pos == f) {
    k = f;
  } else {
    k = pos - 1;
    float dk = pred - hx[k];
    if (pos < f + n) {
      const float dh = hx[pos] - pred;
      if (!(dk <= dh)) return pos;
    }
    while (k > f && (pred - hx[k - 1]) == dk) --k;
  }
  return k;
}

/* Rank selection on the warp's triplet keys: keeps the `keep` smallest of `n` (<= TRIP_BUF) unique
 * 64-bit keys and leaves them SORTED ascending in W.trip[0..min(n,keep)).  PAPER.md:221. */
__device__ __forceinline__ int select_smallest(WarpScratch& W, int n, int keep, int lane) {
  const unsigned long long k0 = (lane < n) ? W.trip[lane] : ~0ull;
  const unsigned long long k1 = (lane + 32 < n) ? W.trip[lane + 32] : ~0ull;
  int r0 = 0, r1 = 0;
  for (int j = 0; j < n; ++j) {
    const unsigned long long kj = W.trip[j];
    r0 += (kj < k0) ? 1 : 0;
    r1 += (kj < k1) ? 1 : 0;
  }
  __syncwarp();
  if (lane < n && r0 < keep) W.trip[r0] = k0;
  if (lane + 32 < n && r1 < keep) W.trip[r1] = k1;
  __syncwarp();
  return n < keep ? n : keep;
}

/* Finishes the queued doublets, one per lane: x1_expected, closest h1, chi2 cut. */
template <class HV>
__device__ __forceinline__ void finish_doublets(const Consts& C, const HV& hx, WarpScratch& W,
                                                int qcount, int& tcount, int wf, int wn, int lane) {
  for (int base = 0; base < qcount; base += 32) {
    const int e = base + lane;
    const bool act = e < qcount;
    const unsigned code = act ? W.dq[e] : 0u;
    const int set = (code >> 10) & 1, i0 = (code >> 5) & 31, i2 = code & 31;
    const int la = set ? 3 : 0;
    const int fa = __shfl_sync(FULL, wf, la);
    const int fb = __shfl_sync(FULL, wf, la + 4);
    const int nb = __shfl_sync(FULL, wn, la + 4);
    const int fc = __shfl_sync(FULL, wf, la + 8);
    bool pass = false;
    unsigned long long key = 0;
    if (act) {
      const float x0 = hx[fa + i0], x2 = hx[fc + i2];
      const float t = (x2 - x0) * (set ? C.inv_dz_ac[1] : C.inv_dz_ac[0]);
      const float zb = set ? C.z[7] : C.z[4], za = set ? C.z[3] : C.z[0];
      const float x1e = zb * t + (x0 - t * za) * (set ? C.K[1] : C.K[0]);
      const int k = closest_hit(hx, fb, nb, x1e);
      if (k >= 0) {
        const float dx = hx[k] - x1e;
        const float chi2 = dx * dx;
        if (chi2 < C.T_triplet) {
          pass = true;
          key = ((unsigned long long)__float_as_uint(chi2) << 32) |
                (unsigned)((set << 15) | (i0 << 10) | (i2 << 5) | (k - fb));
        }
      }
    }
    const unsigned m = __ballot_sync(FULL, pass);
    if (m) {
      if (tcount > 32) tcount = select_smallest(W, tcount, C.n_triplets, lane);
      if (pass) W.trip[tcount + __popc(m & ((1u << lane) - 1u))] = key;
      tcount += __popc(m);
      __syncwarp();
    }
  }
}

/* One warp follows one seed through a1..a6 and leaves its record in the per-seed workspace. */
template <bool DEBUG, class HV>
__device__ __forceinline__ void process_seed(const Consts& C, const TrackArgs& A, const CtaShared& S,
                                             const HV& hx, uint32_t h0, uint32_t seed,
                                             WarpScratch& W, int lane) {
  /* ---- a1: pT-kick extrapolation */
  const float x = A.sx[seed], y = A.sy[seed], tx = A.stx[seed], ty = A.sty[seed], qop = A.sqop[seed];
  const float aq = fmaxf(fabsf(qop), 1e-6f);
  const float p = 1.0f / aq;
  const float x_mag = x + tx * C.mag_dz_seed;
  const float txp = tx + C.kick * qop;
  const int zone = (ty >= 0.0f) ? 1 : 0;
  /* ---- a2: windows.  lanes 0..11: lower edge of layer `lane`; lanes 12..23: upper edge */
  const float x_tol = C.xtol_base + C.xtol_inv_p * aq;
  const bool q_pos = qop > 0.0f, pol_pos = C.polarity > 0;
  const float a_left = (q_pos == pol_pos) ? C.x_asym : 0.0f; /* Eq. (3) */
  const float a_right = (q_pos != pol_pos) ? C.x_asym : 0.0f;
  const int wl = lane < 12 ? lane : (lane < 24 ? lane - 12 : 0);
  const bool wuv = is_uv(wl);
  const float d_reg = S.g_d[wl], w_reg = S.g_w[wl];
  const float xc = x_mag + txp * S.g_dzm[wl];
  const float yl = y + ty * S.g_dzs[wl];
  const float yt = wuv ? yl * S.g_tana[wl] : 0.0f;
  float lo, hi;
  if (!wuv) {
    lo = (xc - x_tol) - a_left;
    hi = (xc + x_tol) + a_right;
  } else {
    const float ctr = xc + yt;
    lo = ctr - C.uv_half_width;
    hi = ctr + C.uv_half_width;
  }
  const int sb = S.seg[wl * 2 + zone], se = S.seg[wl * 2 + zone + 1];
  /* lower edge: first x >= lo; upper edge: first x > hi */
  const bool upper = lane >= 12;
  const float v = upper ? hi : lo;
  int pos = sb, cnt = (lane < 24) ? (se - sb) : 0;
  while (__any_sync(FULL, cnt > 0)) {
    if (cnt > 0) {
      const int half = cnt >> 1;
      const int mid = pos + half;
      const float xm = hx[mid];
      const bool right = upper ? (xm <= v) : (xm < v);
      if (right) { pos = mid + 1; cnt -= half + 1; } else { cnt = half; }
    }
  }
  int first = __shfl_sync(FULL, pos, wl);
  int last = __shfl_sync(FULL, pos, wl + 12);
  if (last < first) last = first;
  /* cap to n_window hits, index-symmetric about the geometric centre */
  const bool capped = (lane < 12) && (last - first > C.n_window);
  {
    const float midv = (lo + hi) * 0.5f;
    int cpos = first, ccnt = capped ? (last - first) : 0;
    while (__any_sync(FULL, ccnt > 0)) {
      if (ccnt > 0) {
        const int half = ccnt >> 1;
        const int mid = cpos + half;
        if (hx[mid] < midv) { cpos = mid + 1; ccnt -= half + 1; } else { ccnt = half; }
      }
    }
    if (capped) {
      const int halfw = C.n_window / 2;
      const int f2 = max(first, cpos - halfw);
      const int l2 = min(last, cpos + halfw);
      first = f2;
      last = l2;
    }
  }
  const int wf = first;        /* event-relative index of the window's first hit (lanes 0..11) */
  const int wn = last - first; /* hits in the window */
  if (DEBUG && lane < 12) {
    if (A.dbg.win_first) A.dbg.win_first[(size_t)seed * NL + lane] = (int32_t)(h0 + wf);
    if (A.dbg.win_count) A.dbg.win_count[(size_t)seed * NL + lane] = wn;
  }

  /* ---- a3: triplet seeding */
  int qcount = 0, tcount = 0;
  const unsigned lt_mask = (1u << lane) - 1u;
  const bool low_p = p < C.p_same_bend;
  const float tol0 = C.mag_tol_base + C.mag_tol_inv_p * aq;
#pragma unroll
  for (int set = 0; set < 2; ++set) {
    const int la = set ? 3 : 0;
    const int fa = __shfl_sync(FULL, wf, la), na = __shfl_sync(FULL, wn, la);
    const int nb = __shfl_sync(FULL, wn, la + 4);
    const int fc = __shfl_sync(FULL, wf, la + 8), nc = __shfl_sync(FULL, wn, la + 8);
    if (na > 0 && nb > 0 && nc > 0) {
      const float x2 = (lane < nc) ? hx[fc + lane] : 0.0f;
      const float xa = (lane < na) ? hx[fa + lane] : 0.0f;
      const float inv_dz = C.inv_dz_ac[set], zmag_a = C.zmag_a[set];
      for (int i0 = 0; i0 < na; ++i0) {
        const float x0 = __shfl_sync(FULL, xa, i0);
        const float t = (x2 - x0) * inv_dz;
        bool ok = lane < nc;
        /* filter 1: same bending direction below p_same_bend */
        if (low_p) ok = ok && ((t - tx) * qop > 0.0f);
        /* filter 2: opening at the magnet centre */
        const float x_at_mag = x0 + t * zmag_a;
        const float tol = fminf(C.mag_tol_max, tol0 + C.mag_tol_tx * fabsf(t));
        ok = ok && (fabsf(x_at_mag - x_mag) < tol);
        const unsigned m = __ballot_sync(FULL, ok);
        if (m) {
          if (ok) W.dq[qcount + __popc(m & lt_mask)] = (uint16_t)((set << 10) | (i0 << 5) | lane);
          qcount += __popc(m);
          if (qcount > 32) {
            __syncwarp();
            finish_doublets(C, hx, W, qcount, tcount, wf, wn, lane);
            qcount = 0;
          }
        }
      }
    }
  }
  __syncwarp();
  if (qcount > 0) finish_doublets(C, hx, W, qcount, tcount, wf, wn, lane);
  if (tcount > 0) tcount = select_smallest(W, tcount, C.n_triplets, lane); /* sorted in (chi2,set,h0,h2) order */
  const int ntr = tcount;
  const int NT = C.n_triplets;

  if (DEBUG) {
    /* triplet table; hit indices need the window bases held by lanes 0..11, so every lane shuffles */
    const bool have = lane < ntr;
    const unsigned long long key = have ? W.trip[lane] : 0ull;
    const unsigned low = (unsigned)key;
    const int set = (low >> 15) & 1, la = set ? 3 : 0;
    const int fa = __shfl_sync(FULL, wf, la), fb = __shfl_sync(FULL, wf, la + 4), fc = __shfl_sync(FULL, wf, la + 8);
    if (lane == 0 && A.dbg.n_triplets) A.dbg.n_triplets[seed] = ntr;
    if (lane < NT) {
      const size_t o = (size_t)seed * NT + lane;
      if (A.dbg.trip_set) A.dbg.trip_set[o] = have ? set : -1;
      if (A.dbg.trip_chi2) A.dbg.trip_chi2[o] = have ? __uint_as_float((unsigned)(key >> 32)) : -1.0f;
      if (A.dbg.trip_hits) {
        A.dbg.trip_hits[o * 3 + 0] = have ? (int32_t)(h0 + fa + ((low >> 10) & 31)) : -1;
        A.dbg.trip_hits[o * 3 + 1] = have ? (int32_t)(h0 + fb + (low & 31)) : -1;
        A.dbg.trip_hits[o * 3 + 2] = have ? (int32_t)(h0 + fc + ((low >> 5) & 31)) : -1;
      }
      if (A.dbg.cand_quality) A.dbg.cand_quality[o] = -1.0f;
      if (A.dbg.cand_hits)
        for (int l = 0; l < NL; ++l) A.dbg.cand_hits[o * NL + l] = -1;
    }
  }

  if (ntr == 0) {
    if (lane == 0) A.ws_nh[seed] = 0;
    return;
  }

  /* ---- a4/a5: extension, lanes = (triplet, other layer) */
  const float T_uv = fmaxf(C.T_uv_min, C.T_uv_slope * (fabsf(tx) + fabsf(ty)));
  for (int base = 0; base < ntr * 9; base += 32) {
    const int tau = base + lane;
    const bool act = tau < ntr * 9;
    const int trip = act ? tau / 9 : 0;
    const int li = act ? tau - trip * 9 : 0;
    const unsigned low = (unsigned)W.trip[trip];
    const int set = (low >> 15) & 1, i0 = (low >> 10) & 31, i2 = (low >> 5) & 31, i1 = low & 31;
    const int la = set ? 3 : 0;
    const int l = li + li / 3 + (1 - set); /* the 9 layers outside the set, ascending */
    const int fa = __shfl_sync(FULL, wf, la), fb = __shfl_sync(FULL, wf, la + 4), fc = __shfl_sync(FULL, wf, la + 8);
    const int fl = __shfl_sync(FULL, wf, l), nl = __shfl_sync(FULL, wn, l);
    const float yt_l = __shfl_sync(FULL, yt, l);
    const float d_l = __shfl_sync(FULL, d_reg, l), w_l = __shfl_sync(FULL, w_reg, l);
    if (act) {
      /* Eq. (4) parameters: exact parabola through the three triplet hits */
      const float x0 = hx[fa + i0], x1 = hx[fb + i1], x2 = hx[fc + i2];
      const float X10 = x1 - x0, X20 = x2 - x0;
      const float D10 = set ? C.D10[1] : C.D10[0], D20 = set ? C.D20[1] : C.D20[0];
      const float W10 = set ? C.W10[1] : C.W10[0];
      const float c0 = (X20 * D10 - X10 * D20) * (set ? C.inv_det[1] : C.inv_det[0]);
      const float t0 = (X10 - c0 * W10) * (set ? C.inv_D10[1] : C.inv_D10[0]);
      const float a0 = (x0 - t0 * (set ? C.d[3] : C.d[0])) - c0 * (set ? C.w[3] : C.w[0]);
      const bool uv = is_uv(l);
      float pred = (a0 + t0 * d_l) + c0 * w_l;
      if (uv) pred = pred + yt_l;
      const int k = closest_hit(hx, fl, nl, pred);
      unsigned code = NO_HIT;
      if (k >= 0) {
        const float dx = hx[k] - pred;
        const float chi2 = dx * dx;
        if (chi2 < (uv ? T_uv : C.T_x)) code = (unsigned)(k - fl);
      }
      W.ext[trip][l] = (uint8_t)code;
      if (li == 0) {
        W.ext[trip][la] = (uint8_t)i0;
        W.ext[trip][la + 4] = (uint8_t)i1;
        W.ext[trip][la + 8] = (uint8_t)i2;
      }
    }
  }
  __syncwarp();

  /* ---- a6: lanes = candidates.  Hit-count rule, fit, Q */
  const bool cand = lane < ntr;
  const int row = cand ? lane : 0;
  const uint32_t* rowp = reinterpret_cast<const uint32_t*>(&W.ext[row][0]);
  const uint32_t cw0 = rowp[0], cw1 = rowp[1], cw2 = rowp[2];
  int n = 0, n_uv = 0;
  bool st_uv[3] = {false, false, false};
#pragma unroll
  for (int l = 0; l < NL; ++l) {
    const uint32_t wsel = (l < 4) ? cw0 : (l < 8 ? cw1 : cw2);
    const bool present = ((wsel >> (8 * (l & 3))) & 0xFFu) != NO_HIT;
    if (present) {
      ++n;
      if (is_uv(l)) { ++n_uv; st_uv[l >> 2] = true; }
    }
  }
  const bool enough = cand && (n >= C.min_hits) && st_uv[0] && st_uv[1] && st_uv[2];

  if (DEBUG && A.dbg.cand_hits) {
#pragma unroll
    for (int l = 0; l < NL; ++l) {
      const uint32_t wsel = (l < 4) ? cw0 : (l < 8 ? cw1 : cw2);
      const unsigned code = (wsel >> (8 * (l & 3))) & 0xFFu;
      const int f_l = __shfl_sync(FULL, wf, l);
      if (cand) A.dbg.cand_hits[((size_t)seed * NT + lane) * NL + l] = (code != NO_HIT) ? (int32_t)(h0 + f_l + code) : -1;
    }
  }

  if (!__any_sync(FULL, enough)) {
    if (lane == 0) A.ws_nh[seed] = 0;
    return;
  }

  /* triplet parabola again, now for the candidate this lane owns */
  const unsigned low = (unsigned)W.trip[row];
  const int set = (low >> 15) & 1, la = set ? 3 : 0;
  float a0, t0, c0;
  {
    const int fa = __shfl_sync(FULL, wf, la), fb = __shfl_sync(FULL, wf, la + 4), fc = __shfl_sync(FULL, wf, la + 8);
    const float x0 = hx[fa + ((low >> 10) & 31)], x1 = hx[fb + (low & 31)], x2 = hx[fc + ((low >> 5) & 31)];
    const float X10 = x1 - x0, X20 = x2 - x0;
    const float D10 = set ? C.D10[1] : C.D10[0], D20 = set ? C.D20[1] : C.D20[0];
    const float W10 = set ? C.W10[1] : C.W10[0];
    c0 = (X20 * D10 - X10 * D20) * (set ? C.inv_det[1] : C.inv_det[0]);
    t0 = (X10 - c0 * W10) * (set ? C.inv_D10[1] : C.inv_D10[0]);
    a0 = (x0 - t0 * (set ? C.d[3] : C.d[0])) - c0 * (set ? C.w[3] : C.w[0]);
  }
  const float inv_Tuv = 1.0f / T_uv;
  /* x fit on the residuals to the triplet parabola: sums in ascending layer order */
  float r[NL];
  float S1 = 0.f, Sd = 0.f, Sw = 0.f, Sdd = 0.f, Sdw = 0.f, Sww = 0.f, Sr = 0.f, Sdr = 0.f, Swr = 0.f;
#pragma unroll
  for (int l = 0; l < NL; ++l) {
    const uint32_t wsel = (l < 4) ? cw0 : (l < 8 ? cw1 : cw2);
    const unsigned code = (wsel >> (8 * (l & 3))) & 0xFFu;
    const bool present = code != NO_HIT;
    const int f_l = __shfl_sync(FULL, wf, l);
    const float yt_l = __shfl_sync(FULL, yt, l);
    const float s_i = hx[present ? (f_l + (int)code) : 0];
    const float dl = C.d[l], wl_ = C.w[l];
    const float m = s_i - yt_l;
    r[l] = m - ((a0 + t0 * dl) + c0 * wl_);
    if (present) {
      S1 = S1 + 1.0f;
      Sd = Sd + dl;
      Sw = Sw + wl_;
      Sdd = Sdd + dl * dl;
      Sdw = Sdw + dl * wl_;
      Sww = Sww + wl_ * wl_;
      Sr = Sr + r[l];
      Sdr = Sdr + dl * r[l];
      Swr = Swr + wl_ * r[l];
    }
  }
  const float C00 = Sdd * Sww - Sdw * Sdw;
  const float C01 = Sdw * Sw - Sd * Sww;
  const float C02 = Sd * Sdw - Sdd * Sw;
  const float C11 = S1 * Sww - Sw * Sw;
  const float C12 = Sd * Sw - S1 * Sdw;
  const float C22 = S1 * Sdd - Sd * Sd;
  const float det = (S1 * C00 + Sd * C01) + Sw * C02;
  const float inv = 1.0f / det;
  const float da = ((C00 * Sr + C01 * Sdr) + C02 * Swr) * inv;
  const float dt = ((C01 * Sr + C11 * Sdr) + C12 * Swr) * inv;
  const float dc = ((C02 * Sr + C12 * Sdr) + C22 * Swr) * inv;
  float rho[NL];
  float Qx = 0.f, U1 = 0.f, Ud = 0.f, Udd = 0.f, Ur = 0.f, Udr = 0.f;
#pragma unroll
  for (int l = 0; l < NL; ++l) {
    const uint32_t wsel = (l < 4) ? cw0 : (l < 8 ? cw1 : cw2);
    const bool present = ((wsel >> (8 * (l & 3))) & 0xFFu) != NO_HIT;
    const float dl = C.d[l], wl_ = C.w[l];
    const float e = r[l] - ((da + dt * dl) + dc * wl_);
    const float chi2 = e * e;
    if (is_uv(l)) {
      rho[l] = e * C.inv_tan[l];
      if (present) {
        Qx = Qx + chi2 * inv_Tuv;
        U1 = U1 + 1.0f;
        Ud = Ud + dl;
        Udd = Udd + dl * dl;
        Ur = Ur + rho[l];
        Udr = Udr + dl * rho[l];
      }
    } else {
      rho[l] = 0.f;
      if (present) Qx = Qx + chi2 * C.inv_Tx;
    }
  }
  const float det2 = U1 * Udd - Ud * Ud;
  const float inv2 = 1.0f / det2;
  const float dy0 = (Udd * Ur - Ud * Udr) * inv2;
  const float dtym = (U1 * Udr - Ud * Ur) * inv2;
  const float dty = dtym * 0.001f;
  const bool ty_ok = fabsf(dty) < C.T_ty;
  float Qy = 0.f;
#pragma unroll
  for (int l = 0; l < NL; ++l) {
    if (!is_uv(l)) continue;
    const uint32_t wsel = (l < 4) ? cw0 : (l < 8 ? cw1 : cw2);
    const bool present = ((wsel >> (8 * (l & 3))) & 0xFFu) != NO_HIT;
    const float ey = rho[l] - (dy0 + dtym * C.d[l]);
    if (present) Qy = Qy + (ey * ey) * C.inv_Ty;
  }
  const int ci = min(3, max(0, n - 9));
  const float Cn = (ci == 0) ? C.C_nhits[0] : (ci == 1 ? C.C_nhits[1] : (ci == 2 ? C.C_nhits[2] : C.C_nhits[3]));
  const float Q = (Qx / (float)(n - 3) + Qy / (float)(n_uv - 2)) * Cn; /* Eq. (6) */
  if (DEBUG && enough && A.dbg.cand_quality) A.dbg.cand_quality[(size_t)seed * NT + lane] = ty_ok ? Q : -2.0f;

  /* accept Q < T_Q, keep the lowest Q; ties -> earlier in (chi2,set,h0,h2) order */
  const bool valid = enough && ty_ok && (Q < C.T_Q);
  unsigned long long qk = valid ? (((unsigned long long)__float_as_uint(Q) << 32) | (unsigned)lane) : ~0ull;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long other = __shfl_xor_sync(FULL, qk, o);
    qk = other < qk ? other : qk;
  }
  if (qk == ~0ull) {
    if (lane == 0) A.ws_nh[seed] = 0;
    return;
  }
  const int winner = (int)(qk & 31u);
  /* record: hit indices need the window bases (lanes 0..11), so every lane shuffles */
#pragma unroll
  for (int l = 0; l < NL; ++l) {
    const uint32_t wsel = (l < 4) ? cw0 : (l < 8 ? cw1 : cw2);
    const unsigned code = (wsel >> (8 * (l & 3))) & 0xFFu;
    const int f_l = __shfl_sync(FULL, wf, l);
    if (lane == winner) W.rec[l] = (code != NO_HIT) ? (int32_t)(h0 + f_l + code) : -1;
  }
  if (lane == winner) {
    /* ---- a6 (cont.): momentum from the slope change (Eq. 9) and the state at z_state */
    const float a = a0 + da, t = t0 + dt, c = c0 + dc;
    const float t_ref = t * 0.001f;
    const float dslope = t_ref - tx;
    const float F = C.poly[0] + dslope * (C.poly[1] + dslope * (C.poly[2] + dslope * (C.poly[3] + dslope * C.poly[4])));
    W.rec[12] = (int32_t)seed;
    W.rec[13] = n;
    W.rec[14] = __float_as_int((a + t * C.ds) + c * C.ws);
    W.rec[15] = __float_as_int((y + ty * C.dz_state) + (dy0 + dtym * C.ds));
    W.rec[16] = __float_as_int((t + c * C.dws) * 0.001f);
    W.rec[17] = __float_as_int(ty + dtym * 0.001f);
    W.rec[18] = __float_as_int(dslope / F);
    W.rec[19] = __float_as_int(Q);
    A.ws_nh[seed] = n;
  }
  __syncwarp();
  if (lane < REC_WORDS) A.ws_rec[(size_t)seed * REC_WORDS + lane] = W.rec[lane];
  __syncwarp();
}

template <bool DEBUG>
__global__ void __launch_bounds__(CTA_THREADS) lf_track_kernel(const __grid_constant__ Consts C,
                                                               const __grid_constant__ TrackArgs A) {
  CtaShared& S = *reinterpret_cast<CtaShared*>(lf_smem);
  float* buf = stage_buf();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) mbar_init(&S.mbar, 1);
  if (tid < NL) {
    S.g_tana[tid] = C.tana[tid];
    S.g_dzs[tid] = C.dzs[tid];
    S.g_dzm[tid] = C.dzm[tid];
    S.g_d[tid] = C.d[tid];
    S.g_w[tid] = C.w[tid];
  }
  __syncthreads();
  uint32_t phase = 0;
  for (;;) {
    if (tid == 0) {
      S.ev = (int)atomicAdd(A.ticket, 1u);
      S.next_seed = 0;
    }
    __syncthreads(); /* (A) previous event fully retired: buf, seg, counters reusable */
    const uint32_t ev = (uint32_t)S.ev;
    if (ev >= A.n_events) break;
    const uint32_t* so = A.seg_off + (size_t)ev * NSEG;
    const uint32_t h0 = so[0], h1 = so[NSEG];
    if (tid <= NSEG) S.seg[tid] = (int)(so[tid] - h0);
    const int nh = (int)(h1 - h0);
    const float* gsrc = A.hx + h0;
    const bool staged = nh + 4 <= A.stage_cap;
    const int skew = (int)((reinterpret_cast<uintptr_t>(gsrc) >> 2) & 3);
    if (staged) {
      /* Stage the event: hit i lives at buf[skew + i]; the 16-byte aligned interior goes by TMA. */
      const int head = min(nh, (4 - skew) & 3);
      const int bulk = (nh - head) & ~3;
      const int tail = nh - head - bulk;
      if (tid == 0 && bulk > 0) {
        fence_proxy_async();
        mbar_expect_tx(&S.mbar, (uint32_t)bulk * 4u);
        bulk_g2s(buf + skew + head, gsrc + head, (uint32_t)bulk * 4u, &S.mbar);
      }
      if (tid < head) buf[skew + tid] = gsrc[tid];
      if (tid >= 32 && tid < 32 + tail) buf[skew + head + bulk + (tid - 32)] = gsrc[head + bulk + (tid - 32)];
      if (bulk > 0) {
        mbar_wait(&S.mbar, phase);
        phase ^= 1u;
      }
    }
    __syncthreads(); /* (B) seg table and head/tail hits visible */
    const uint32_t s0 = A.seed_off[ev], s1 = A.seed_off[ev + 1];
    WarpScratch& W = S.ws[warp];
    if (staged) {
      const HitView<true> hv{skew};
      for (;;) {
        int k = 0;
        if (lane == 0) k = atomicAdd(&S.next_seed, 1);
        k = __shfl_sync(FULL, k, 0);
        if (s0 + (uint32_t)k >= s1) break;
        process_seed<DEBUG>(C, A, S, hv, h0, s0 + (uint32_t)k, W, lane);
      }
    } else {
      const HitView<false> hv{gsrc};
      for (;;) {
        int k = 0;
        if (lane == 0) k = atomicAdd(&S.next_seed, 1);
        k = __shfl_sync(FULL, k, 0);
        if (s0 + (uint32_t)k >= s1) break;
        process_seed<DEBUG>(C, A, S, hv, h0, s0 + (uint32_t)k, W, lane);
      }
    }
    __syncthreads(); /* (C) every seed of the event has its ws_nh flag */
    /* rank the event's tracks in seed order (a7, first half) */
    const int ns = (int)(s1 - s0);
    int base = 0;
    for (int c = 0; c < ns; c += CTA_THREADS) {
      const int i = c + tid;
      const bool flag = (i < ns) && (__ldcg(A.ws_nh + s0 + i) > 0);
      const unsigned m = __ballot_sync(FULL, flag);
      if (lane == 0) S.warp_tot[warp] = __popc(m);
      __syncthreads();
      int off = 0, tot = 0;
#pragma unroll
      for (int wq = 0; wq < WARPS_PER_CTA; ++wq) {
        const int tq = S.warp_tot[wq];
        off += (wq < warp) ? tq : 0;
        tot += tq;
      }
      if (i < ns) {
        A.ws_rank[s0 + i] = flag ? (base + off + __popc(m & ((1u << lane) - 1u))) : -1;
        A.ws_event[s0 + i] = (int32_t)ev;
      }
      base += tot;
      __syncthreads();
    }
    if (tid == 0) A.ev_count[ev] = (uint32_t)base;
  }
}

/* Exclusive scan of per-event track counts (single CTA); also re-arms the event ticket. */
__global__ void __launch_bounds__(1024) lf_scan_kernel(const uint32_t* __restrict__ ev_count, uint32_t n_events,
                                                       uint32_t* __restrict__ ev_off_ws, uint32_t* __restrict__ out_off,
                                                       uint32_t* __restrict__ n_tracks, uint32_t* ticket) {
  __shared__ uint32_t warp_tot[32];
  __shared__ uint32_t carry;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) carry = 0;
  __syncthreads();
  for (uint32_t c = 0; c < n_events; c += 1024) {
    const uint32_t i = c + tid;
    const uint32_t v = (i < n_events) ? ev_count[i] : 0u;
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(FULL, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      uint32_t wt = warp_tot[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(FULL, wt, o);
        if (lane >= o) wt += t;
      }
      warp_tot[lane] = wt; /* inclusive over warps */
    }
    __syncthreads();
    const uint32_t excl = carry + (warp > 0 ? warp_tot[warp - 1] : 0u) + (incl - v);
    if (i < n_events) {
      ev_off_ws[i] = excl;
      out_off[i] = excl;
    }
    __syncthreads();
    if (tid == 0) carry += warp_tot[31];
    __syncthreads();
  }
  if (tid == 0) {
    out_off[n_events] = carry;
    *n_tracks = carry;
    *ticket = 0u;
  }
}

/* Stream compaction (a7): one thread per (seed, record word); coalesced reads of the per-seed
 * records, dense SoA writes in (event, seed) order. */
__global__ void __launch_bounds__(256) lf_compact_kernel(const int32_t* __restrict__ ws_rec, const int32_t* __restrict__ ws_rank,
                                                         const int32_t* __restrict__ ws_event, const uint32_t* __restrict__ ev_off,
                                                         size_t n_seeds, int32_t* __restrict__ hit_idx, int32_t* __restrict__ seed_idx,
                                                         int32_t* __restrict__ n_hits, float* __restrict__ state, float* __restrict__ quality) {
  const size_t gid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= n_seeds * REC_WORDS) return;
  const size_t seed = gid / REC_WORDS;
  const int wd = (int)(gid - seed * REC_WORDS);
  const int rank = ws_rank[seed];
  if (rank < 0) return;
  const size_t dst = (size_t)ev_off[ws_event[seed]] + (size_t)rank;
  const int32_t v = ws_rec[gid];
  if (wd < 12) hit_idx[dst * NL + wd] = v;
  else if (wd == 12) seed_idx[dst] = v;
  else if (wd == 13) n_hits[dst] = v;
  else if (wd < 19) state[dst * 5 + (wd - 14)] = __int_as_float(v);
  else quality[dst] = __int_as_float(v);
}

} // namespace lf
