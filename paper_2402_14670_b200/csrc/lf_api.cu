/*
 * lf_api.cu -- C-ABI entry points of include/lf.h: handle management, host-side constants,
 * launch sequence.  No torch types; the caller's framework only supplies device memory and a stream.
 */
#include "../../include/lf.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "lf_kernels.cuh"

namespace {

thread_local std::string g_create_error;
constexpr size_t PROF_RING = 256;
constexpr int N_PROF_EV = LF_N_KERNELS + 1;
/* lf_run_host pipelines the batch in chunks of events: H2D of chunk c+1, kernels of chunk c and D2H of
 * chunk c-1 overlap (PCIe is full duplex).  At most HOST_MAX_CHUNKS chunks of at least HOST_CHUNK_EVENTS. */
constexpr int HOST_MAX_CHUNKS = 16;
constexpr size_t HOST_CHUNK_EVENTS = 2048; /* measured on config 3: 8-10 chunks beat 16 (11.1 vs 11.6 ms) */

/* One batch in flight through the host path (lf_run_host = slot 0; lf_host_submit / lf_host_collect: LF_HOST_SLOTS of them,
 * so that the copies of the next batch run while this one is finished): its device staging, events and bookkeeping. */
struct HostSlot {
  float* seeds = nullptr;      /* 5 * max_seeds */
  uint32_t* seed_off = nullptr;
  float* hits = nullptr;
  uint16_t* hits16 = nullptr;  /* hit_storage = 1: the caller's packed copy */
  float* origin16 = nullptr;
  uint32_t* seg_off = nullptr;
  int32_t *hit_idx = nullptr, *seed_idx = nullptr, *n_hits = nullptr;
  float *state = nullptr, *quality = nullptr;
  uint32_t *ev_off = nullptr, *n_tracks = nullptr; /* ne + HOST_MAX_CHUNKS + 1; HOST_MAX_CHUNKS */
  uint32_t* pinned_count = nullptr; /* host, pinned: HOST_MAX_CHUNKS counts, then the chunk-relative event offsets */
  cudaEvent_t ev_start = nullptr, ev_done = nullptr, ev_h2d[HOST_MAX_CHUNKS] = {}, ev_comp[HOST_MAX_CHUNKS] = {}, ev_cnt[HOST_MAX_CHUNKS] = {};
  bool ready = false;
  /* the submitted batch, until it has been collected */
  bool pending = false;
  cudaStream_t st = nullptr; /* the stream its kernels were enqueued on */
  lf_tracks out = {};
  size_t n_events = 0;
  int n_chunks = 0;
  size_t bounds[HOST_MAX_CHUNKS + 1] = {}; /* first event of every chunk */
  size_t first_seed[HOST_MAX_CHUNKS + 1] = {};
};
struct HostBufs {
  cudaStream_t s_h2d = nullptr, s_cnt = nullptr, s_d2h = nullptr; /* library-owned copy streams, shared by the slots */
  HostSlot slot[LF_HOST_SLOTS];
};

} // namespace

struct lf_handle {
  lf::Consts C;
  lf_geometry G;
  lf_params P;
  size_t max_events, max_seeds, max_hits;
  int device;
  int sm_count, stage_cap;
  int ext_chunk;   /* rows the extension kernel stages at a time: 256, or 128 if that keeps one more CTA per SM */
  int win_threads; /* threads per CTA of the window kernel: 256, or 512 if that keeps more warps per SM (large stages) */
  int stage_cap_x; /* the seeding kernel stages the six x layers only: about half an event */
  int regs[4], grid[4], ctas_per_sm[4], smem_bytes[4]; /* window, seed, extend, fit kernels */
  unsigned long long* ev_state; /* look-back words of the fit kernel's stream compaction */
  /* workspace */
  __half* hx16;     /* hit_storage = 1 only: the library's own fp16 copy (when the caller gives none) */
  float* origin16;
  float* hx_scratch; /* hit_storage = 1 only: fp32 image of events that do not fit the stage (lf_kernels.cuh, fetch_event) */
  bool half2;       /* hit_storage = 1: the seeding kernel evaluates pairs of doublets in __half2 (seed_triplets_h2) */
  bool wide;        /* the wide build of the event kernels runs (no-UT mode, or caps beyond the narrow limits) */
  int sides;        /* followed tracks (rows) per seed: 2 in the no-UT mode */
  uint32_t* win;
  void* trip_code;
  uint8_t* n_trip;
  int32_t *ws_rec, *ws_nh, *ws_rank;
  uint32_t *ev_count, *ev_dup, *ev_acc, *tickets;
  unsigned long long* counters; /* LF_N_COUNTERS: written by the debug build of the kernels */
  bool counters_valid = false;  /* the most recent launch was a debug launch */
  bool tickets_dirty = false;   /* an lf_run failed between its first and its last launch: the event tickets, which the last
                                   CTA of the fit kernel re-arms, may be left advanced; the next launch zeroes them first */
  uint32_t* validate_res; /* 4 words: lf_validate_inputs' violation bits and offending indices */
  uint4* acc_rec;
  lf::FitLut* fit_lut;
  size_t workspace_bytes;
  HostBufs hb;
  size_t host_chunk_events = HOST_CHUNK_EVENTS;
  size_t last_events = 0; /* n_events of the most recent launch (lf_run_counters) */
  int last_kernels = -1;  /* kernels the most recent launch enqueued (lf_get_info); -1 = nothing launched yet */
  bool profiling = false;
  size_t prof_runs = 0;                 /* runs recorded since profiling was enabled */
  cudaEvent_t (*prof_ev)[N_PROF_EV] = nullptr;  /* ring of PROF_RING event sets */
  std::string err;
};

namespace {

lf_status fail(lf_handle* h, lf_status st, const std::string& msg) {
  if (h) h->err = msg; else g_create_error = msg;
  return st;
}

#define LF_CUDA(h, call)                                                                              \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess)                                                                            \
      return fail((h), LF_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));              \
  } while (0)

bool uv_layer(int l) { return (l & 3) == 1 || (l & 3) == 2; }

/* cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel function, not to a handle: a later lf_create
 * with a smaller stage must not lower it under a live handle.  Per (kernel, device) the library keeps the largest
 * value any handle has asked for and only ever raises the attribute. */
std::mutex g_attr_mutex;
constexpr int MAX_DEVICES = 64;
int g_attr_max[3][4][2][MAX_DEVICES]; /* [narrow / wide / narrow half2][kernel][debug][device] */

cudaError_t raise_dynamic_smem(const void* kernel, int wide, int k, int dbg, int device, int bytes) {
  std::lock_guard<std::mutex> lock(g_attr_mutex);
  int& cur = g_attr_max[wide][k][dbg][device < 0 || device >= MAX_DEVICES ? 0 : device];
  if (bytes <= cur) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess) cur = bytes;
  return e;
}

/* Host-side constants in fp32, one rounding per operation.
 * Built with -ffp-contract=off; volatile stores keep every intermediate a genuine float. */
void make_consts(const lf_geometry& G, const lf_params& P, lf::Consts& c) {
  std::memset(&c, 0, sizeof(c));
  const float one = 1.0f, milli = 0.001f;
  c.z_seed = G.z_seed; c.z_mag = G.z_mag; c.kick = G.kick;
  c.dr = G.d_ratio * 1000.0f;
  c.K[0] = G.k_first; c.K[1] = G.k_last;
  for (int i = 0; i < 5; ++i) c.poly[i] = G.qop_poly[i];
  c.polarity = G.polarity;
  c.mag_dz_seed = c.z_mag - c.z_seed;
  for (int l = 0; l < lf::NL; ++l) {
    c.z[l] = G.z[l];
    c.tana[l] = G.tan_alpha[l];
    c.inv_tan[l] = uv_layer(l) ? one / c.tana[l] : 0.0f;
    c.dzs[l] = c.z[l] - c.z_seed;
    c.dzm[l] = c.z[l] - c.z_mag;
    const float dz = c.z[l] - G.z_ref;
    c.d[l] = dz * milli;
    const float dd = c.d[l] * c.d[l];
    const float curv = one + c.dr * c.d[l];
    c.w[l] = dd * curv;
  }
  for (int s = 0; s < 2; ++s) {
    const int a = s ? 3 : 0, b = a + 4, cc = a + 8;
    c.inv_dz_ac[s] = one / (c.z[cc] - c.z[a]);
    c.zmag_a[s] = c.z_mag - c.z[a];
    c.inv_r[s] = one / (c.inv_dz_ac[s] * c.zmag_a[s]); /* bracket of the h2 interval only (not a decision) */
    c.inv_abs_zmag_a[s] = one / std::fabs(c.zmag_a[s]);  /* idem */
    c.tolmax_over_zmag[s] = P.mag_tol_max * c.inv_abs_zmag_a[s]; /* idem */
    c.D10[s] = c.d[b] - c.d[a];
    c.D20[s] = c.d[cc] - c.d[a];
    c.W10[s] = c.w[b] - c.w[a];
    c.W20[s] = c.w[cc] - c.w[a];
    const float p1 = c.W20[s] * c.D10[s];
    const float p2 = c.W10[s] * c.D20[s];
    c.inv_det[s] = one / (p1 - p2);
    c.inv_D10[s] = one / c.D10[s];
  }
  c.dz_state = G.z_state - c.z_seed;
  const float dzst = G.z_state - G.z_ref;
  c.ds = dzst * milli;
  const float ds2 = c.ds * c.ds;
  const float curv_s = one + c.dr * c.ds;
  c.ws = ds2 * curv_s;
  const float two_ds = 2.0f * c.ds;
  const float three_dr = 3.0f * c.dr;
  c.dws = two_ds + three_dr * ds2;
  c.T_triplet = P.T_triplet; c.T_x = P.T_x; c.T_uv_slope = P.T_uv_slope; c.T_uv_min = P.T_uv_min;
  c.T_ty = P.T_ty; c.inv_Tx = one / P.T_x; c.inv_Ty = one / P.T_y; c.T_Q = P.T_Q;
  for (int i = 0; i < 4; ++i) c.C_nhits[i] = P.C_nhits[i];
  c.n_window = P.n_window; c.n_triplets = P.n_triplets; c.min_hits = P.min_hits;
  c.xtol_base = P.xtol_base; c.xtol_inv_p = P.xtol_inv_p; c.x_asym = P.x_asym; c.uv_half_width = P.uv_half_width;
  c.p_same_bend = P.p_same_bend; c.mag_tol_base = P.mag_tol_base; c.mag_tol_inv_p = P.mag_tol_inv_p;
  c.mag_tol_tx = P.mag_tol_tx; c.mag_tol_max = P.mag_tol_max;
  c.qop_mode = G.qop_mode;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 10; ++j) c.poly2d[i][j] = G.qop_poly2d[i][j];
  c.mode = P.mode;
  c.sides = (P.mode == 1) ? 2 : 1;
  if (P.mode == 1) {
    c.inv_p_min = one / P.velo_p_min;
    c.inv_pt_min = one / P.velo_pt_min;
    for (int i = 0; i < 8; ++i) c.xtol_poly[i] = P.xtol_poly[i];
    c.x_overlap = P.x_overlap;
  }
}

/* Geometry sums and cofactors of the two least-squares fits for every 12-bit hit-presence mask, in the
 * canonical fp32 order (sums over the present layers in ascending layer order; DESIGN.md "Canonical
 * arithmetic" a6).  Masks that cannot occur (singular systems) hold inf/nan and are never read. */
void make_fit_lut(const lf::Consts& c, lf::FitLut* lut) {
  for (unsigned m = 0; m < (1u << lf::NL); ++m) {
    volatile float S1 = 0.f, Sd = 0.f, Sw = 0.f, Sdd = 0.f, Sdw = 0.f, Sww = 0.f, U1 = 0.f, Ud = 0.f, Udd = 0.f;
    for (int l = 0; l < lf::NL; ++l) {
      if (!((m >> l) & 1u)) continue;
      const float dl = c.d[l], wl = c.w[l];
      const float dd = dl * dl, dw = dl * wl, ww = wl * wl;
      S1 = S1 + 1.0f; Sd = Sd + dl; Sw = Sw + wl; Sdd = Sdd + dd; Sdw = Sdw + dw; Sww = Sww + ww;
      if (uv_layer(l)) { U1 = U1 + 1.0f; Ud = Ud + dl; Udd = Udd + dd; }
    }
    auto mul = [](float a, float b) { volatile float r = a * b; return (float)r; };
    lf::FitLut& L = lut[m];
    L.C00 = mul(Sdd, Sww) - mul(Sdw, Sdw);
    L.C01 = mul(Sdw, Sw) - mul(Sd, Sww);
    L.C02 = mul(Sd, Sdw) - mul(Sdd, Sw);
    L.C11 = mul(S1, Sww) - mul(Sw, Sw);
    L.C12 = mul(Sd, Sw) - mul(S1, Sdw);
    L.C22 = mul(S1, Sdd) - mul(Sd, Sd);
    volatile float det = mul(S1, L.C00) + mul(Sd, L.C01);
    det = det + mul(Sw, L.C02);
    L.inv_det = 1.0f / det;
    L.pad0 = 0.f;
    L.U1 = U1; L.Ud = Ud; L.Udd = Udd;
    const float det2 = mul(U1, Udd) - mul(Ud, Ud);
    L.inv_det2 = 1.0f / det2;
  }
}

const char* validate(const lf_geometry& G, const lf_params& P) {
  if (G.n_layers != LF_N_LAYERS) return "geometry.n_layers must be 12";
  for (int l = 0; l < LF_N_LAYERS; ++l) {
    if (!std::isfinite(G.z[l]) || !std::isfinite(G.tan_alpha[l])) return "geometry: non-finite layer constant";
    if (l > 0 && !(G.z[l] > G.z[l - 1])) return "geometry.z must be strictly ascending";
    if (uv_layer(l) ? (G.tan_alpha[l] == 0.0f) : (G.tan_alpha[l] != 0.0f))
      return "geometry.tan_alpha must be 0 on x layers (0,3 mod 4) and non-zero on u/v layers (1,2 mod 4)";
  }
  if (!(G.z_mag > G.z_seed) || !(G.z[0] > G.z_mag)) return "geometry: need z_seed < z_mag < z[0]";
  {
    const float gf[] = {G.z_seed, G.z_mag, G.kick, G.z_ref, G.d_ratio, G.k_first, G.k_last, G.z_state,
                        G.qop_poly[0], G.qop_poly[1], G.qop_poly[2], G.qop_poly[3], G.qop_poly[4]};
    for (float v : gf)
      if (!std::isfinite(v)) return "geometry: non-finite constant";
    if (G.kick == 0.0f) return "geometry.kick must be non-zero (its sign is the bending direction)";
  }
  if (G.polarity != 1 && G.polarity != -1) return "geometry.polarity must be +1 or -1";
  if (G.qop_mode != 0 && G.qop_mode != 1) return "geometry.qop_mode must be 0 (constants) or 1 (2-D polynomials)";
  if (G.qop_mode == 1)
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j < ((i % 2 == 0) ? 10 : 6); ++j)
        if (!std::isfinite(G.qop_poly2d[i][j])) return "geometry.qop_poly2d: non-finite coefficient";
  if (P.n_window < 2 || P.n_window > LF_MAX_WINDOW_WIDE) return "params.n_window out of [2, LF_MAX_WINDOW_WIDE]";
  if (P.n_triplets < 1 || P.n_triplets > LF_MAX_TRIPLETS_WIDE) return "params.n_triplets out of [1, LF_MAX_TRIPLETS_WIDE]";
  if (P.mode != 0 && P.mode != 1) return "params.mode must be 0 (with UT) or 1 (no-UT)";
  if (P.mode == 1) {
    if (!(P.velo_p_min > 0) || !(P.velo_pt_min > 0)) return "params: velo_p_min and velo_pt_min must be positive";
    for (int i = 0; i < 8; ++i)
      if (!std::isfinite(P.xtol_poly[i])) return "params.xtol_poly: non-finite coefficient";
    if (!std::isfinite(P.x_overlap)) return "params.x_overlap: non-finite";
  }
  if (P.min_hits < 4 || P.min_hits > 12) return "params.min_hits out of [4, 12]";
  if (!(P.T_triplet > 0) || !(P.T_x > 0) || !(P.T_y > 0) || !(P.T_uv_min > 0) || !(P.T_Q > 0) || !(P.T_ty > 0))
    return "params: tolerances must be positive";
  if (P.hit_storage != 0 && P.hit_storage != 1) return "params.hit_storage must be 0 or 1";
  if (P.hit_storage == 1 && P.seed_arith != 0 && P.seed_arith != 1) return "params.seed_arith must be 0 (half2 pairs) or 1 (fp32)";
  {
    /* every tolerance is finite ("no cap" is a large finite number, not inf: the kernels bracket with it) */
    const float pf[] = {P.T_triplet, P.T_x, P.T_uv_slope, P.T_uv_min, P.T_ty, P.T_y, P.T_Q, P.C_nhits[0], P.C_nhits[1],
                        P.C_nhits[2], P.C_nhits[3], P.xtol_base, P.xtol_inv_p, P.x_asym, P.uv_half_width, P.p_same_bend,
                        P.mag_tol_base, P.mag_tol_inv_p, P.mag_tol_tx, P.mag_tol_max};
    for (float v : pf)
      if (!std::isfinite(v)) return "params: non-finite tolerance or constant";
    if (P.T_uv_slope < 0 || P.xtol_base < 0 || P.xtol_inv_p < 0 || P.x_asym < 0 || P.uv_half_width < 0 || P.p_same_bend < 0 ||
        P.mag_tol_base < 0 || P.mag_tol_inv_p < 0 || P.mag_tol_tx < 0 || P.mag_tol_max < 0)
      return "params: window and magnet tolerances must be >= 0";
    for (int i = 0; i < 4; ++i)
      if (!(P.C_nhits[i] > 0)) return "params.C_nhits must be positive";
  }
  return nullptr;
}

bool use_wide(const lf_params& P) {
  return P.mode == 1 || P.n_window > LF_MAX_WINDOW || P.n_triplets > LF_MAX_TRIPLETS;
}

template <bool DEBUG, bool WIDE>
lf_status launch_impl(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, lf_tracks* out,
                 const lf_debug* dbg, cudaStream_t st, size_t event_base = 0) {
  const bool prof = h->profiling;
  cudaEvent_t* pe = prof ? h->prof_ev[h->prof_runs % PROF_RING] : nullptr;
  if (h->tickets_dirty) LF_CUDA(h, cudaMemsetAsync(h->tickets, 0, (lf::N_TICKETS + 1) * sizeof(uint32_t), st));
  h->tickets_dirty = true; /* until every kernel of this run has been enqueued */
  if (prof) LF_CUDA(h, cudaEventRecord(pe[0], st));
  lf::EventArgs A;
  std::memset(&A, 0, sizeof(A));
  A.sx = seeds->x; A.sy = seeds->y; A.stx = seeds->tx; A.sty = seeds->ty; A.sqop = seeds->qop;
  A.seed_off = seeds->event_offsets;
  A.hx = hits->x; A.seg_off = hits->seg_offsets;
  A.n_events = (uint32_t)n_events;
  A.stage_cap = h->stage_cap;
  A.stage_cap_x = h->stage_cap_x;
  A.ext_chunk = h->ext_chunk;
  A.win = h->win; A.trip_code = h->trip_code; A.n_trip = h->n_trip;
  A.ws_rec = h->ws_rec; A.ws_nh = h->ws_nh; A.ws_rank = h->ws_rank;
  A.ev_count = h->ev_count;
  A.ev_dup = h->ev_dup;
  A.acc_rec = h->acc_rec; A.ev_acc = h->ev_acc; A.fit_lut = h->fit_lut;
  A.ev_state = h->ev_state;
  if (dbg) {
    A.dbg.win_first = dbg->win_first; A.dbg.win_count = dbg->win_count; A.dbg.n_triplets = dbg->n_triplets;
    A.dbg.trip_hits = dbg->trip_hits; A.dbg.trip_set = dbg->trip_set; A.dbg.trip_chi2 = dbg->trip_chi2;
    A.dbg.cand_hits = dbg->cand_hits; A.dbg.cand_quality = dbg->cand_quality;
  }
  if (DEBUG) {
    A.dbg.counters = h->counters;
    LF_CUDA(h, cudaMemsetAsync(h->counters, 0, LF_N_COUNTERS * sizeof(unsigned long long), st));
  }
  h->counters_valid = DEBUG;
  h->last_events = n_events;
  const bool work = n_events > 0;
  int n_kernels = work ? LF_N_KERNELS : 0; /* what this call enqueues (lf_get_info) */
  auto grid_of = [&](int k) { return (int)std::min<size_t>((size_t)h->grid[k], n_events); };
  const bool half_hits = h->P.hit_storage == 1;
  const __half* use16 = nullptr;
  const float* use_origin = nullptr;
  if (half_hits) {
    if (hits->x16 && hits->origin16) { /* the caller's fp16 copy */
      use16 = reinterpret_cast<const __half*>(hits->x16);
      use_origin = hits->origin16;
    } else { /* pack the fp32 hits (timed with the window kernel) */
      if (work && hits->n_hits > 0) {
        const int pg = (int)std::min<size_t>((size_t)h->sm_count * 8, n_events);
        lf::lf_pack_hits_kernel<<<pg, 256, 0, st>>>(hits->x, hits->seg_offsets, (uint32_t)n_events, (uint32_t)event_base, h->hx16,
                                                    h->origin16);
        ++n_kernels;
      }
      use16 = h->hx16;
      use_origin = h->origin16;
    }
    A.hx16 = use16;
    A.origin16 = use_origin;
    A.hx_scratch = h->hx_scratch;
    A.event_base = (uint32_t)event_base;
  }
  if (work) {
    A.ticket = h->tickets + 0;
    A.scratch_writer = 1; /* the window kernel decodes oversized events once for all four kernels */
    lf::lf_window_kernel<DEBUG, WIDE><<<grid_of(0), h->win_threads, h->smem_bytes[0], st>>>(h->C, A);
  }
  if (prof) LF_CUDA(h, cudaEventRecord(pe[1], st));
  A.scratch_writer = 0;
  A.stage_cap = h->stage_cap_x;
  if (work) {
    A.ticket = h->tickets + 1;
    if (!WIDE && h->half2) lf::lf_seed_kernel<DEBUG, false, true><<<grid_of(1), lf::SEED_THREADS, h->smem_bytes[1], st>>>(h->C, A);
    else lf::lf_seed_kernel<DEBUG, WIDE><<<grid_of(1), lf::SEED_THREADS, h->smem_bytes[1], st>>>(h->C, A);
  }
  if (prof) LF_CUDA(h, cudaEventRecord(pe[2], st));
  A.stage_cap = h->stage_cap;
  if (hits->x != nullptr) { /* extension and fit read the fp32 hits when the caller gave them */
    A.hx16 = nullptr;
    A.origin16 = nullptr;
  }
  if (work) {
    A.ticket = h->tickets + 2;
    lf::lf_extend_kernel<DEBUG, WIDE><<<grid_of(2), lf::FIT_THREADS, h->smem_bytes[2], st>>>(h->C, A);
  }
  if (prof) LF_CUDA(h, cudaEventRecord(pe[3], st));
  if (work) {
    /* a6 + a7: the fit kernel also scans the events' track counts (look-back) and writes the dense outputs */
    lf::TrackOut O;
    O.hit_idx = out->hit_idx; O.seed_idx = out->seed_idx; O.n_hits = out->n_hits; O.state = out->state; O.quality = out->quality;
    O.event_offsets = out->event_offsets; O.n_tracks = out->n_tracks;
    O.ev_state = h->ev_state; O.tickets = h->tickets;
    A.ticket = h->tickets + 3;
    lf::lf_fit_kernel<DEBUG, WIDE><<<grid_of(3), lf::FIT_THREADS, h->smem_bytes[3], st>>>(h->C, A, O);
  } else { /* no events: an empty track list */
    LF_CUDA(h, cudaMemsetAsync(out->event_offsets, 0, sizeof(uint32_t), st));
    LF_CUDA(h, cudaMemsetAsync(out->n_tracks, 0, sizeof(uint32_t), st));
  }
  if (prof) {
    LF_CUDA(h, cudaEventRecord(pe[4], st));
    ++h->prof_runs;
  }
  LF_CUDA(h, cudaGetLastError());
  h->tickets_dirty = false;
  h->last_kernels = n_kernels;
  return LF_OK;
}

template <bool DEBUG>
lf_status launch(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, lf_tracks* out,
                 const lf_debug* dbg, cudaStream_t st, size_t event_base = 0) {
  return h->wide ? launch_impl<DEBUG, true>(h, seeds, hits, n_events, out, dbg, st, event_base)
                 : launch_impl<DEBUG, false>(h, seeds, hits, n_events, out, dbg, st, event_base);
}

lf_status check_run_args(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, lf_tracks* out) {
  if (!h) return LF_ERR_INVALID_ARG;
  if (!seeds || !hits || !out) return fail(h, LF_ERR_INVALID_ARG, "lf_run: NULL seeds/hits/out");
  if (!seeds->event_offsets || !hits->seg_offsets || !out->event_offsets || !out->n_tracks)
    return fail(h, LF_ERR_INVALID_ARG, "lf_run: NULL offset table or n_tracks pointer");
  if (seeds->n_seeds > 0 && (!seeds->x || !seeds->y || !seeds->tx || !seeds->ty || (!seeds->qop && h->P.mode == 0)))
    return fail(h, LF_ERR_INVALID_ARG, "lf_run: NULL seed array");
  if (hits->n_hits > 0 && !hits->x && !(h->P.hit_storage == 1 && hits->x16 && hits->origin16))
    return fail(h, LF_ERR_INVALID_ARG, "lf_run: NULL hit array (x may be NULL only with hit_storage = 1 and x16 + origin16 given)");
  if (seeds->n_seeds > 0 && (!out->hit_idx || !out->seed_idx || !out->n_hits || !out->state || !out->quality))
    return fail(h, LF_ERR_INVALID_ARG, "lf_run: NULL output array");
  if ((reinterpret_cast<uintptr_t>(out->hit_idx) & 15u) != 0)
    return fail(h, LF_ERR_INVALID_ARG, "lf_run: out->hit_idx must be 16-byte aligned");
  if (n_events == 0 && (seeds->n_seeds != 0 || hits->n_hits != 0))
    return fail(h, LF_ERR_INVALID_ARG, "lf_run: n_events == 0 with non-empty seeds or hits");
  if (n_events > h->max_events || seeds->n_seeds > h->max_seeds || hits->n_hits > h->max_hits)
    return fail(h, LF_ERR_CAPACITY, "lf_run: batch exceeds the maxima given to lf_create");
  if (hits->n_hits >= (size_t)0x7fffffff) return fail(h, LF_ERR_CAPACITY, "lf_run: hit indices must fit int32");
  if (out->capacity < seeds->n_seeds)
    return fail(h, LF_ERR_CAPACITY, "lf_run: out->capacity must be >= seeds->n_seeds");
  return LF_OK;
}

} // namespace

extern "C" {

uint32_t lf_abi_version(void) { return LF_ABI_VERSION; }

size_t lf_sizeof(int which) {
  switch (which) {
    case 0: return sizeof(lf_geometry);
    case 1: return sizeof(lf_params);
    case 2: return sizeof(lf_seeds);
    case 3: return sizeof(lf_hits);
    case 4: return sizeof(lf_tracks);
    case 5: return sizeof(lf_debug);
    case 6: return sizeof(lf_info);
    default: return 0;
  }
}

const char* lf_last_error(const lf_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

lf_status lf_create(const lf_geometry* geometry, const lf_params* params, size_t max_events, size_t max_seeds,
                    size_t max_hits, lf_handle** out) {
  if (!geometry || !params || !out) return fail(nullptr, LF_ERR_INVALID_ARG, "lf_create: NULL argument");
  *out = nullptr;
  if (const char* why = validate(*geometry, *params)) return fail(nullptr, LF_ERR_INVALID_ARG, std::string("lf_create: ") + why);
  if (params->hit_storage == 1 && use_wide(*params))
    return fail(nullptr, LF_ERR_UNSUPPORTED, "lf_create: hit_storage = 1 needs mode 0 with n_window <= 32 and n_triplets <= 16");
  if (max_hits >= (size_t)0x7fffffff || max_seeds >= (size_t)0x7fffffff || max_events >= (size_t)0x7fffffff / LF_N_LAYERS / 2)
    return fail(nullptr, LF_ERR_CAPACITY, "lf_create: maxima must fit 32-bit indices");

  lf_handle* h = new (std::nothrow) lf_handle();
  if (!h) return fail(nullptr, LF_ERR_CUDA, "lf_create: out of host memory");
  h->G = *geometry; h->P = *params;
  h->max_events = max_events; h->max_seeds = max_seeds; h->max_hits = max_hits;
  make_consts(*geometry, *params, h->C);
  h->wide = use_wide(*params);
  h->half2 = params->hit_storage == 1 && params->seed_arith != 1;
  h->sides = h->C.sides;

  auto bail = [&](lf_status st, const std::string& msg) { g_create_error = msg; lf_destroy(h); return st; };
#define LF_CREATE_CUDA(call)                                                                     \
  do {                                                                                           \
    cudaError_t e_ = (call);                                                                     \
    if (e_ != cudaSuccess) return bail(LF_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)

  LF_CREATE_CUDA(cudaGetDevice(&h->device));
  cudaDeviceProp prop;
  LF_CREATE_CUDA(cudaGetDeviceProperties(&prop, h->device));
  h->sm_count = prop.multiProcessorCount;
  if (prop.major < 10) return bail(LF_ERR_UNSUPPORTED, "lf_create: this library is built for sm_100a (Blackwell) only");

  /* Shared-memory stage for one event's hits, sized from the maxima (include/lf.h, lf_create):
   * 1.25 x the mean event + 512 hits, clamped to [2048, 16384].  Larger events read global memory. */
  {
    const double mean_hits = (double)max_hits / (double)std::max<size_t>(max_events, 1);
    size_t cap = (size_t)(1.25 * mean_hits) + 512;
    cap = (cap + 255) & ~size_t(255);
    h->stage_cap = (int)std::min<size_t>(std::max<size_t>(cap, 2048), 16384);
  }
  const size_t stage_bytes = (size_t)lf::HDR_BYTES + (size_t)h->stage_cap * sizeof(float);
  h->stage_cap_x = (h->stage_cap / 2 + 256 + 255) & ~255; /* half an event + its fluctuation + the runs' alignment gaps */
  const size_t stage_bytes_x = (size_t)lf::HDR_BYTES + (size_t)h->stage_cap_x * sizeof(float);
  h->smem_bytes[0] = (int)stage_bytes;
  h->smem_bytes[1] = (int)(stage_bytes_x + (h->wide ? sizeof(lf::SeedTables<true, false>) : (h->half2 ? sizeof(lf::SeedTables<false, true>) : sizeof(lf::SeedTables<false, false>))));
  h->ext_chunk = lf::FIT_CHUNK;
  h->smem_bytes[2] = (int)(stage_bytes + lf::ext_tables_bytes(params->n_triplets, h->ext_chunk));
  h->smem_bytes[3] = (int)(stage_bytes + lf::FIT_TABLES_BYTES);
  const void* kern_n[4][2] = {{(const void*)lf::lf_window_kernel<false, false>, (const void*)lf::lf_window_kernel<true, false>},
                              {(const void*)lf::lf_seed_kernel<false, false>, (const void*)lf::lf_seed_kernel<true, false>},
                              {(const void*)lf::lf_extend_kernel<false, false>, (const void*)lf::lf_extend_kernel<true, false>},
                              {(const void*)lf::lf_fit_kernel<false, false>, (const void*)lf::lf_fit_kernel<true, false>}};
  const void* kern_w[4][2] = {{(const void*)lf::lf_window_kernel<false, true>, (const void*)lf::lf_window_kernel<true, true>},
                              {(const void*)lf::lf_seed_kernel<false, true>, (const void*)lf::lf_seed_kernel<true, true>},
                              {(const void*)lf::lf_extend_kernel<false, true>, (const void*)lf::lf_extend_kernel<true, true>},
                              {(const void*)lf::lf_fit_kernel<false, true>, (const void*)lf::lf_fit_kernel<true, true>}};
  const void* kern_h2[2] = {(const void*)lf::lf_seed_kernel<false, false, true>, (const void*)lf::lf_seed_kernel<true, false, true>};
  if (h->half2) { kern_n[1][0] = kern_h2[0]; kern_n[1][1] = kern_h2[1]; }
  const void* (*kern)[2] = h->wide ? kern_w : kern_n;
  int threads[4] = {lf::WIN_THREADS, lf::SEED_THREADS, lf::FIT_THREADS, lf::FIT_THREADS};
  h->win_threads = lf::WIN_THREADS;
  for (int k = 0; k < 4; ++k) {
    if (k == 0) { /* window kernel: CTAs of 512 threads if they put more warps on an SM (a large stage limits the CTAs) */
      int occ = 0, occ_big = 0;
      for (int d = 0; d < 2; ++d)
        LF_CREATE_CUDA(raise_dynamic_smem(kern[k][d], h->wide ? 1 : 0, k, d, h->device, h->smem_bytes[k]));
      LF_CREATE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern[k][0], lf::WIN_THREADS, h->smem_bytes[k]));
      LF_CREATE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_big, kern[k][0], lf::WIN_THREADS_BIG, h->smem_bytes[k]));
      if (occ_big * lf::WIN_THREADS_BIG > occ * lf::WIN_THREADS) threads[0] = h->win_threads = lf::WIN_THREADS_BIG;
    }
    if (k == 2) { /* extension kernel: half-size row tables if they buy a resident CTA (large events) */
      const int small = (int)(stage_bytes + lf::ext_tables_bytes(params->n_triplets, lf::FIT_CHUNK / 2));
      int occ_big = 0, occ_small = 0;
      for (int d = 0; d < 2; ++d)
        LF_CREATE_CUDA(raise_dynamic_smem(kern[k][d], h->wide ? 1 : 0, k, d, h->device, h->smem_bytes[k]));
      LF_CREATE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_big, kern[k][0], threads[k], h->smem_bytes[k]));
      LF_CREATE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_small, kern[k][0], threads[k], small));
      if (occ_small > occ_big) {
        h->ext_chunk = lf::FIT_CHUNK / 2;
        h->smem_bytes[k] = small;
      }
    }
    for (int d = 0; d < 2; ++d)
      LF_CREATE_CUDA(raise_dynamic_smem(kern[k][d], h->wide ? 1 : (h->half2 && k == 1 ? 2 : 0), k, d, h->device, h->smem_bytes[k]));
    LF_CREATE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->ctas_per_sm[k], kern[k][0], threads[k], h->smem_bytes[k]));
    if (h->ctas_per_sm[k] < 1) return bail(LF_ERR_CUDA, "lf_create: an event kernel does not fit on an SM");
    h->grid[k] = h->sm_count * h->ctas_per_sm[k];
    cudaFuncAttributes fa;
    LF_CREATE_CUDA(cudaFuncGetAttributes(&fa, kern[k][0]));
    h->regs[k] = fa.numRegs;
  }

  const size_t ns = std::max<size_t>(max_seeds, 1), ne = std::max<size_t>(max_events, 1);
  const size_t nt = (size_t)params->n_triplets;
  const size_t nrows = ns * (size_t)h->sides; /* followed tracks */
  const size_t code_bytes = h->wide ? sizeof(uint32_t) : sizeof(uint16_t);
  if (params->hit_storage == 1) {
    const size_t nh = std::max<size_t>(max_hits, 1);
    LF_CREATE_CUDA(cudaMalloc(&h->hx16, nh * sizeof(__half)));
    LF_CREATE_CUDA(cudaMalloc(&h->origin16, lf_origin_slots(ne, nh) * sizeof(float)));
    LF_CREATE_CUDA(cudaMalloc(&h->hx_scratch, nh * sizeof(float)));
  }
  LF_CREATE_CUDA(cudaMalloc(&h->win, nrows * lf::WIN_ROW * sizeof(uint32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->trip_code, nrows * nt * code_bytes));
  LF_CREATE_CUDA(cudaMalloc(&h->n_trip, nrows));
  LF_CREATE_CUDA(cudaMalloc(&h->ws_rec, ns * lf::REC_WORDS * sizeof(int32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->ws_nh, ns * sizeof(int32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->ws_rank, ns * sizeof(int32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->ev_count, ne * sizeof(uint32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->ev_dup, ne * sizeof(uint32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->ev_acc, ne * sizeof(uint32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->acc_rec, nrows * nt * sizeof(uint4)));
  {
    std::vector<lf::FitLut> lut(1u << lf::NL);
    make_fit_lut(h->C, lut.data());
    LF_CREATE_CUDA(cudaMalloc(&h->fit_lut, lut.size() * sizeof(lf::FitLut)));
    LF_CREATE_CUDA(cudaMemcpy(h->fit_lut, lut.data(), lut.size() * sizeof(lf::FitLut), cudaMemcpyHostToDevice));
  }
  LF_CREATE_CUDA(cudaMalloc(&h->validate_res, 4 * sizeof(uint32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->counters, LF_N_COUNTERS * sizeof(unsigned long long)));
  LF_CREATE_CUDA(cudaMalloc(&h->tickets, (lf::N_TICKETS + 1) * sizeof(uint32_t)));
  LF_CREATE_CUDA(cudaMemset(h->tickets, 0, (lf::N_TICKETS + 1) * sizeof(uint32_t)));
  LF_CREATE_CUDA(cudaMalloc(&h->ev_state, ne * sizeof(unsigned long long)));
  h->workspace_bytes = nrows * (lf::WIN_ROW * 4 + nt * (code_bytes + sizeof(uint4)) + 1) + ns * (lf::REC_WORDS + 2) * 4 +
                       (3 * ne + 1 + lf::N_TICKETS) * sizeof(uint32_t) + ne * sizeof(unsigned long long) +
                       (sizeof(lf::FitLut) << lf::NL);
#undef LF_CREATE_CUDA
  *out = h;
  return LF_OK;
}

lf_status lf_destroy(lf_handle* h) {
  if (!h) return LF_OK;
  { /* a batch still in flight through the host path: let its copies and kernels finish before their memory goes */
    bool in_flight = false;
    for (const HostSlot& b : h->hb.slot) in_flight = in_flight || b.pending;
    if (in_flight) {
      for (const HostSlot& b : h->hb.slot)
        if (b.pending) cudaStreamSynchronize(b.st);
      if (h->hb.s_h2d) cudaStreamSynchronize(h->hb.s_h2d);
      if (h->hb.s_cnt) cudaStreamSynchronize(h->hb.s_cnt);
      if (h->hb.s_d2h) cudaStreamSynchronize(h->hb.s_d2h);
    }
  }
  cudaFree(h->hx16); cudaFree(h->origin16); cudaFree(h->hx_scratch);
  cudaFree(h->win); cudaFree(h->trip_code); cudaFree(h->n_trip);
  cudaFree(h->ws_rec); cudaFree(h->ws_nh); cudaFree(h->ws_rank);
  cudaFree(h->ev_count); cudaFree(h->ev_dup); cudaFree(h->ev_acc); cudaFree(h->acc_rec); cudaFree(h->fit_lut); cudaFree(h->tickets); cudaFree(h->ev_state);
  cudaFree(h->validate_res);
  cudaFree(h->counters);
  HostBufs& hb = h->hb;
  for (HostSlot& b : hb.slot) {
    cudaFree(b.seeds); cudaFree(b.seed_off); cudaFree(b.hits); cudaFree(b.hits16); cudaFree(b.origin16); cudaFree(b.seg_off);
    cudaFree(b.hit_idx); cudaFree(b.seed_idx); cudaFree(b.n_hits); cudaFree(b.state); cudaFree(b.quality);
    cudaFree(b.ev_off); cudaFree(b.n_tracks);
    if (b.pinned_count) cudaFreeHost(b.pinned_count);
    if (b.ev_start) cudaEventDestroy(b.ev_start);
    if (b.ev_done) cudaEventDestroy(b.ev_done);
    for (int c = 0; c < HOST_MAX_CHUNKS; ++c) {
      if (b.ev_h2d[c]) cudaEventDestroy(b.ev_h2d[c]);
      if (b.ev_comp[c]) cudaEventDestroy(b.ev_comp[c]);
      if (b.ev_cnt[c]) cudaEventDestroy(b.ev_cnt[c]);
    }
  }
  if (hb.s_h2d) cudaStreamDestroy(hb.s_h2d);
  if (hb.s_cnt) cudaStreamDestroy(hb.s_cnt);
  if (hb.s_d2h) cudaStreamDestroy(hb.s_d2h);
  if (h->prof_ev) {
    for (size_t i = 0; i < PROF_RING; ++i)
      for (cudaEvent_t e : h->prof_ev[i])
        if (e) cudaEventDestroy(e);
    delete[] h->prof_ev;
  }
  delete h;
  return LF_OK;
}

lf_status lf_get_info(const lf_handle* h, lf_info* out) {
  if (!h || !out) return LF_ERR_INVALID_ARG;
  out->kernels_per_run = h->last_kernels >= 0 ? h->last_kernels : LF_N_KERNELS + (h->P.hit_storage == 1 ? 1 : 0);
  const int threads[4] = {h->win_threads, lf::SEED_THREADS, lf::FIT_THREADS, lf::FIT_THREADS};
  for (int k = 0; k < 4; ++k) {
    out->regs[k] = h->regs[k];
    out->block[k] = threads[k];
    out->grid[k] = h->grid[k];
    out->ctas_per_sm[k] = h->ctas_per_sm[k];
    out->smem_bytes[k] = h->smem_bytes[k];
  }
  out->staged_hits_per_event = h->stage_cap - 4;
  out->sm_count = h->sm_count;
  out->workspace_bytes = h->workspace_bytes;
  return LF_OK;
}

lf_status lf_run_counters(lf_handle* h, uint64_t counters[LF_N_COUNTERS]) {
  if (!h || !counters) return LF_ERR_INVALID_ARG;
  for (int i = 0; i < LF_N_COUNTERS; ++i) counters[i] = 0;
  const size_t ne = h->last_events;
  if (ne == 0) return LF_OK;
  std::vector<uint32_t> acc(ne), dup(ne), cnt(ne);
  LF_CUDA(h, cudaDeviceSynchronize());
  LF_CUDA(h, cudaMemcpy(acc.data(), h->ev_acc, ne * sizeof(uint32_t), cudaMemcpyDeviceToHost));
  LF_CUDA(h, cudaMemcpy(dup.data(), h->ev_dup, ne * sizeof(uint32_t), cudaMemcpyDeviceToHost));
  LF_CUDA(h, cudaMemcpy(cnt.data(), h->ev_count, ne * sizeof(uint32_t), cudaMemcpyDeviceToHost));
  for (size_t e = 0; e < ne; ++e) {
    counters[0] += acc[e];
    counters[1] += dup[e] ? 1u : 0u;
    counters[7] += cnt[e];
  }
  if (h->counters_valid) {
    unsigned long long dev[LF_N_COUNTERS];
    LF_CUDA(h, cudaMemcpy(dev, h->counters, sizeof(dev), cudaMemcpyDeviceToHost));
    for (int i = 2; i <= 6; ++i) counters[i] = dev[i];
  }
  return LF_OK;
}

lf_status lf_set_profiling(lf_handle* h, int enabled) {
  if (!h) return LF_ERR_INVALID_ARG;
  if (enabled && !h->prof_ev) {
    h->prof_ev = new (std::nothrow) cudaEvent_t[PROF_RING][N_PROF_EV]();
    if (!h->prof_ev) return fail(h, LF_ERR_CUDA, "lf_set_profiling: out of host memory");
    for (size_t i = 0; i < PROF_RING; ++i)
      for (cudaEvent_t& e : h->prof_ev[i]) LF_CUDA(h, cudaEventCreate(&e));
  }
  h->profiling = enabled != 0;
  h->prof_runs = 0;
  return LF_OK;
}

lf_status lf_kernel_times(lf_handle* h, float ms[LF_N_KERNELS]) {
  if (!h || !ms) return LF_ERR_INVALID_ARG;
  if (!h->profiling || h->prof_runs == 0) return fail(h, LF_ERR_INVALID_ARG, "lf_kernel_times: no profiled run recorded");
  const size_t n = std::min<size_t>(h->prof_runs, PROF_RING);
  double acc[LF_N_KERNELS] = {};
  for (size_t r = 0; r < n; ++r)
    for (int i = 0; i < LF_N_KERNELS; ++i) {
      float t = 0.f;
      LF_CUDA(h, cudaEventElapsedTime(&t, h->prof_ev[r][i], h->prof_ev[r][i + 1]));
      acc[i] += t;
    }
  for (int i = 0; i < LF_N_KERNELS; ++i) ms[i] = (float)(acc[i] / (double)n);
  return LF_OK;
}

lf_status lf_run(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, lf_tracks* out,
                 void* cuda_stream) {
  const lf_status st = check_run_args(h, seeds, hits, n_events, out);
  if (st != LF_OK) return st;
  for (const HostSlot& b : h->hb.slot) /* the workspace is in use */
    if (b.pending) return fail(h, LF_ERR_INVALID_ARG, "lf_run: a batch submitted with lf_host_submit has not been collected");
  h->err.clear();
  return launch<false>(h, seeds, hits, n_events, out, nullptr, (cudaStream_t)cuda_stream);
}

lf_status lf_run_debug(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, lf_tracks* out,
                       const lf_debug* debug, void* cuda_stream) {
  const lf_status st = check_run_args(h, seeds, hits, n_events, out);
  if (st != LF_OK) return st;
  if (!debug) return fail(h, LF_ERR_INVALID_ARG, "lf_run_debug: NULL debug");
  for (const HostSlot& b : h->hb.slot)
    if (b.pending) return fail(h, LF_ERR_INVALID_ARG, "lf_run_debug: a batch submitted with lf_host_submit has not been collected");
  h->err.clear();
  return launch<true>(h, seeds, hits, n_events, out, debug, (cudaStream_t)cuda_stream);
}

lf_status lf_validate_inputs(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, void* cuda_stream) {
  if (!h) return LF_ERR_INVALID_ARG;
  if (!seeds || !hits || !seeds->event_offsets || !hits->seg_offsets)
    return fail(h, LF_ERR_INVALID_ARG, "lf_validate_inputs: NULL seeds/hits or offset table");
  if (seeds->n_seeds > 0 && (!seeds->x || !seeds->y || !seeds->tx || !seeds->ty || (!seeds->qop && h->P.mode == 0)))
    return fail(h, LF_ERR_INVALID_ARG, "lf_validate_inputs: NULL seed array");
  const bool only16 = !hits->x && h->P.hit_storage == 1 && hits->x16 && hits->origin16; /* the fp16 copy is the only input */
  if (hits->n_hits > 0 && !hits->x && !only16)
    return fail(h, LF_ERR_INVALID_ARG, "lf_validate_inputs: NULL hit array (x may be NULL only with hit_storage = 1 and x16 + origin16 given)");
  if (n_events > h->max_events || seeds->n_seeds > h->max_seeds || hits->n_hits > h->max_hits)
    return fail(h, LF_ERR_CAPACITY, "lf_validate_inputs: batch exceeds the maxima given to lf_create");
  h->err.clear();
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint32_t* res = h->validate_res; /* word 0: violation bits; words 1..3: smallest offending index of each kind */
  LF_CUDA(h, cudaMemsetAsync(res, 0, sizeof(uint32_t), st));
  LF_CUDA(h, cudaMemsetAsync(res + 1, 0xFF, 3 * sizeof(uint32_t), st));
  const int blocks = std::max(1, std::min<int>(h->sm_count * 8, (int)((n_events * lf::NSEG + 7) / 8) + 1));
  lf::lf_validate_kernel<<<blocks, 256, 0, st>>>(hits->x, only16 ? reinterpret_cast<const __half*>(hits->x16) : nullptr,
                                               only16 ? hits->origin16 : nullptr, hits->seg_offsets, (uint32_t)n_events, (uint32_t)hits->n_hits,
                                               seeds->event_offsets, (uint32_t)seeds->n_seeds, seeds->x, seeds->y, seeds->tx,
                                               seeds->ty, h->P.mode == 0 ? seeds->qop : nullptr, res);
  LF_CUDA(h, cudaGetLastError());
  uint32_t host[4] = {0, 0, 0, 0};
  LF_CUDA(h, cudaMemcpyAsync(host, res, sizeof(host), cudaMemcpyDeviceToHost, st));
  LF_CUDA(h, cudaStreamSynchronize(st));
  if (host[0] == 0) return LF_OK;
  std::string msg = "lf_validate_inputs:";
  if (host[0] & lf::BAD_SEG_OFFSETS) msg += " seg_offsets not monotone / not ending at n_hits (segment " + std::to_string(host[1]) + ");";
  if (host[0] & lf::BAD_HIT_ORDER) msg += " hits not ascending inside a segment (hit " + std::to_string(host[2]) + ");";
  if (host[0] & lf::BAD_HIT_VALUE) msg += " non-finite hit coordinate (hit " + std::to_string(host[2]) + ");";
  if (host[0] & lf::BAD_SEED_OFFSETS) msg += " seed event_offsets not monotone / not ending at n_seeds (event " + std::to_string(host[3]) + ");";
  if (host[0] & lf::BAD_SEED_VALUE) msg += " non-finite seed state (seed " + std::to_string(host[3]) + ");";
  return fail(h, LF_ERR_INVALID_ARG, msg);
}

size_t lf_origin_slots(size_t n_events, size_t n_hits) { return (n_hits >> lf::H16_SHIFT) + n_events * lf::NSEG + 2; }

lf_status lf_pack_hits(lf_handle* h, const lf_hits* hits, size_t n_events, uint16_t* x16_out, float* origin16_out,
                       void* cuda_stream) {
  if (!h) return LF_ERR_INVALID_ARG;
  if (!hits || !hits->seg_offsets || (hits->n_hits > 0 && (!hits->x || !x16_out)) || !origin16_out)
    return fail(h, LF_ERR_INVALID_ARG, "lf_pack_hits: NULL hits / offsets / output");
  h->err.clear();
  if (n_events == 0 || hits->n_hits == 0) return LF_OK;
  const int pg = (int)std::min<size_t>((size_t)h->sm_count * 8, n_events);
  lf::lf_pack_hits_kernel<<<pg, 256, 0, (cudaStream_t)cuda_stream>>>(hits->x, hits->seg_offsets, (uint32_t)n_events, 0u,
                                                                    reinterpret_cast<__half*>(x16_out), origin16_out);
  LF_CUDA(h, cudaGetLastError());
  return LF_OK;
}

lf_status lf_set_host_chunk_events(lf_handle* h, size_t min_events_per_chunk) {
  if (!h) return LF_ERR_INVALID_ARG;
  if (min_events_per_chunk == 0) return fail(h, LF_ERR_INVALID_ARG, "lf_set_host_chunk_events: must be >= 1");
  h->host_chunk_events = min_events_per_chunk;
  return LF_OK;
}

static lf_status host_submit(lf_handle* h, int slot, const lf_seeds* seeds, const lf_hits* hits, size_t n_events,
                             lf_tracks* out, void* cuda_stream, bool after_stream);
static lf_status host_collect(lf_handle* h, int slot);

/* an error in the middle of the pipeline: copies from / into the caller's host buffers may still be in flight on the
 * library's streams; drain them (and the caller's stream) before handing the buffers back */
static void host_drain(lf_handle* h, void* cuda_stream) {
  HostBufs& hb = h->hb;
  if (hb.s_h2d) cudaStreamSynchronize(hb.s_h2d);
  if (hb.s_cnt) cudaStreamSynchronize(hb.s_cnt);
  if (hb.s_d2h) cudaStreamSynchronize(hb.s_d2h);
  /* An error aborts EVERY batch in flight on the handle (include/lf.h): the kernels of each of them run on the stream it
   * was submitted on, which need not be `cuda_stream` (lf_host_collect has none to pass), so wait for those streams
   * before the slots are marked idle and the workspace is handed to the next lf_run. */
  for (HostSlot& b : hb.slot)
    if (b.pending) cudaStreamSynchronize(b.st);
  if (cuda_stream) cudaStreamSynchronize((cudaStream_t)cuda_stream);
  for (HostSlot& b : hb.slot) b.pending = false;
}

lf_status lf_run_host(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, lf_tracks* out,
                      void* cuda_stream) {
  const lf_status st0 = check_run_args(h, seeds, hits, n_events, out);
  if (st0 != LF_OK) return st0;
  h->err.clear();
  for (const HostSlot& b : h->hb.slot)
    if (b.pending) return fail(h, LF_ERR_INVALID_ARG, "lf_run_host: a batch submitted with lf_host_submit has not been collected");
  lf_status rs = host_submit(h, 0, seeds, hits, n_events, out, cuda_stream, true);
  if (rs == LF_OK) rs = host_collect(h, 0);
  if (rs == LF_ERR_CUDA) host_drain(h, cuda_stream);
  return rs;
}

lf_status lf_host_submit(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, lf_tracks* out,
                         void* cuda_stream, int slot) {
  const lf_status st0 = check_run_args(h, seeds, hits, n_events, out);
  if (st0 != LF_OK) return st0;
  if (slot < 0 || slot >= LF_HOST_SLOTS) return fail(h, LF_ERR_INVALID_ARG, "lf_host_submit: slot out of range");
  if (h->hb.slot[slot].pending) return fail(h, LF_ERR_INVALID_ARG, "lf_host_submit: the slot holds a batch that has not been collected");
  h->err.clear();
  const lf_status rs = host_submit(h, slot, seeds, hits, n_events, out, cuda_stream, false);
  if (rs == LF_ERR_CUDA) host_drain(h, cuda_stream); /* failed half-way: nothing stays in flight (argument errors enqueue nothing) */
  return rs;
}

lf_status lf_host_collect(lf_handle* h, int slot) {
  if (!h) return LF_ERR_INVALID_ARG;
  if (slot < 0 || slot >= LF_HOST_SLOTS) return fail(h, LF_ERR_INVALID_ARG, "lf_host_collect: slot out of range");
  if (!h->hb.slot[slot].pending) return fail(h, LF_ERR_INVALID_ARG, "lf_host_collect: no batch was submitted to the slot");
  h->err.clear();
  const lf_status rs = host_collect(h, slot);
  if (rs != LF_OK) host_drain(h, nullptr);
  return rs;
}

/* First half of the host path: everything that needs no answer from the device.  Enqueues the host -> device copies of
 * the whole batch (library stream), the kernels of every chunk (caller's stream, each chunk behind its copy) and the small
 * copies that bring every chunk's track count back (library stream); returns without waiting. */
static lf_status host_submit(lf_handle* h, int slot, const lf_seeds* seeds, const lf_hits* hits, size_t n_events,
                             lf_tracks* out, void* cuda_stream, bool after_stream) {
  const uint32_t* so = seeds->event_offsets; /* HOST tables: the chunking reads them */
  const uint32_t* go = hits->seg_offsets;
  if (so[0] != 0 || go[0] != 0 || so[n_events] != seeds->n_seeds || go[n_events * lf::NSEG] != hits->n_hits)
    return fail(h, LF_ERR_INVALID_ARG, "lf_run_host: offset tables do not match n_seeds / n_hits");
  HostBufs& hb = h->hb;
  HostSlot& b = hb.slot[slot];
  cudaStream_t st = (cudaStream_t)cuda_stream;
  for (const HostSlot& o : hb.slot) /* the batches in flight share the workspace: their kernels must run one after the other */
    if (o.pending && o.st != st)
      return fail(h, LF_ERR_INVALID_ARG, "lf_host_submit: batches in flight on one handle must use the same cuda_stream");
  b.out = *out;
  b.n_events = n_events;
  b.n_chunks = 0;
  b.st = st;
  b.pending = true;
  if (n_events == 0) return LF_OK;
  const bool packed = h->P.hit_storage == 1 && hits->x16 && hits->origin16; /* the caller ships the fp16 copy */
  if (!hb.s_h2d) LF_CUDA(h, cudaStreamCreateWithFlags(&hb.s_h2d, cudaStreamNonBlocking));
  if (!hb.s_cnt) LF_CUDA(h, cudaStreamCreateWithFlags(&hb.s_cnt, cudaStreamNonBlocking));
  if (!hb.s_d2h) LF_CUDA(h, cudaStreamCreateWithFlags(&hb.s_d2h, cudaStreamNonBlocking));
  if (!b.ready) {
    /* First use of the slot.  Every member is allocated only while it is still null, so that a submit that ran out of
     * memory part-way leaks nothing: the next one completes the set (and lf_destroy frees whatever exists). */
    const size_t ns = std::max<size_t>(h->max_seeds, 1), ne = std::max<size_t>(h->max_events, 1);
    const size_t nh = std::max<size_t>(h->max_hits, 1);
#define LF_SLOT_ALLOC(member, bytes) \
    do { if (!(member)) LF_CUDA(h, cudaMalloc(&(member), (bytes))); } while (0)
#define LF_SLOT_EVENT(member) \
    do { if (!(member)) LF_CUDA(h, cudaEventCreateWithFlags(&(member), cudaEventDisableTiming)); } while (0)
    LF_SLOT_ALLOC(b.seeds, 5 * ns * sizeof(float));
    LF_SLOT_ALLOC(b.seed_off, (ne + 1) * sizeof(uint32_t));
    LF_SLOT_ALLOC(b.hits, nh * sizeof(float));
    if (h->P.hit_storage == 1) {
      LF_SLOT_ALLOC(b.hits16, nh * sizeof(uint16_t));
      LF_SLOT_ALLOC(b.origin16, lf_origin_slots(ne, nh) * sizeof(float));
    }
    LF_SLOT_ALLOC(b.seg_off, (ne * lf::NSEG + 1) * sizeof(uint32_t));
    LF_SLOT_ALLOC(b.hit_idx, ns * lf::NL * sizeof(int32_t));
    LF_SLOT_ALLOC(b.seed_idx, ns * sizeof(int32_t));
    LF_SLOT_ALLOC(b.n_hits, ns * sizeof(int32_t));
    LF_SLOT_ALLOC(b.state, ns * 5 * sizeof(float));
    LF_SLOT_ALLOC(b.quality, ns * sizeof(float));
    LF_SLOT_ALLOC(b.ev_off, (ne + HOST_MAX_CHUNKS + 1) * sizeof(uint32_t));
    LF_SLOT_ALLOC(b.n_tracks, HOST_MAX_CHUNKS * sizeof(uint32_t));
    if (!b.pinned_count) LF_CUDA(h, cudaMallocHost(&b.pinned_count, (ne + 2 * HOST_MAX_CHUNKS + 1) * sizeof(uint32_t)));
    LF_SLOT_EVENT(b.ev_start);
    LF_SLOT_EVENT(b.ev_done);
    for (int c = 0; c < HOST_MAX_CHUNKS; ++c) {
      LF_SLOT_EVENT(b.ev_h2d[c]);
      LF_SLOT_EVENT(b.ev_comp[c]);
      LF_SLOT_EVENT(b.ev_cnt[c]);
    }
#undef LF_SLOT_ALLOC
#undef LF_SLOT_EVENT
    b.ready = true;
  }
  const size_t stride = std::max<size_t>(h->max_seeds, 1);
  /* Chunk boundaries.  The pipeline is bound by the host->device copies, so what is left after the last byte has
   * arrived (kernels + device->host copy of the LAST chunk) is pure latency: equal chunks of at least
   * host_chunk_events events, the last of them cut into four pieces of 40 / 27 / 18 / 15 % so that this tail is short
   * while every piece's kernels still hide behind the next piece's copy. */
  size_t* bounds = b.bounds;
  int n_chunks = 0;
  {
    const int base = (int)std::min<size_t>(HOST_MAX_CHUNKS - 3, std::max<size_t>(1, n_events / h->host_chunk_events));
    for (int c = 0; c < base; ++c) bounds[n_chunks++] = (size_t)(((unsigned long long)n_events * (unsigned)c) / (unsigned)base);
    const size_t last0 = bounds[n_chunks - 1], last_n = n_events - last0;
    if (last_n >= 64) {
      bounds[n_chunks++] = last0 + (last_n * 40) / 100;
      bounds[n_chunks++] = last0 + (last_n * 67) / 100;
      bounds[n_chunks++] = last0 + (last_n * 85) / 100;
    }
    bounds[n_chunks] = n_events;
  }
  b.n_chunks = n_chunks;
  for (int c = 0; c <= n_chunks; ++c) b.first_seed[c] = so[bounds[c]];
  auto chunk_begin = [&](int c) { return bounds[c]; };

  /* lf_run_host: the copy streams start after whatever the caller queued on `cuda_stream` before this call.
   * lf_host_submit: they start at once, so that this batch's copies run under the previous batch's kernels. */
  if (after_stream) {
    LF_CUDA(h, cudaEventRecord(b.ev_start, st));
    LF_CUDA(h, cudaStreamWaitEvent(hb.s_h2d, b.ev_start, 0));
    LF_CUDA(h, cudaStreamWaitEvent(hb.s_cnt, b.ev_start, 0));
    LF_CUDA(h, cudaStreamWaitEvent(hb.s_d2h, b.ev_start, 0));
  }

  /* ---- host -> device: the offset tables once, then seeds and hits chunk by chunk */
  LF_CUDA(h, cudaMemcpyAsync(b.seed_off, so, (n_events + 1) * sizeof(uint32_t), cudaMemcpyHostToDevice, hb.s_h2d));
  LF_CUDA(h, cudaMemcpyAsync(b.seg_off, go, (n_events * lf::NSEG + 1) * sizeof(uint32_t), cudaMemcpyHostToDevice, hb.s_h2d));
  /* the seeds of the whole batch go first, in five copies (15 % of the input bytes): per-chunk seed copies would add
   * 5 x n_chunks small transfers, each with its fixed cost, to the stream that bounds the pipeline */
  const float* src[5] = {seeds->x, seeds->y, seeds->tx, seeds->ty, seeds->qop};
  for (int i = 0; i < 5 && seeds->n_seeds > 0; ++i)
    if (src[i]) /* qop may be NULL in the no-UT mode */
      LF_CUDA(h, cudaMemcpyAsync(b.seeds + i * stride, src[i], seeds->n_seeds * sizeof(float), cudaMemcpyHostToDevice, hb.s_h2d));
  for (int c = 0; c < n_chunks; ++c) {
    const size_t e0 = chunk_begin(c), e1 = chunk_begin(c + 1);
    const size_t g0 = go[e0 * lf::NSEG], g1 = go[e1 * lf::NSEG];
    if (g1 > g0 && hits->x)
      LF_CUDA(h, cudaMemcpyAsync(b.hits + g0, hits->x + g0, (g1 - g0) * sizeof(float), cudaMemcpyHostToDevice, hb.s_h2d));
    if (g1 > g0 && packed) { /* the packed copy of the chunk: its halves and the origin slots its segments own */
      LF_CUDA(h, cudaMemcpyAsync(b.hits16 + g0, hits->x16 + g0, (g1 - g0) * sizeof(uint16_t), cudaMemcpyHostToDevice, hb.s_h2d));
      const size_t o0 = (g0 >> lf::H16_SHIFT) + e0 * lf::NSEG, o1 = (g1 >> lf::H16_SHIFT) + e1 * lf::NSEG + 1;
      LF_CUDA(h, cudaMemcpyAsync(b.origin16 + o0, hits->origin16 + o0, (o1 - o0) * sizeof(float), cudaMemcpyHostToDevice, hb.s_h2d));
    }
    LF_CUDA(h, cudaEventRecord(b.ev_h2d[c], hb.s_h2d));
  }
  /* ---- kernels on the caller's stream, chunk by chunk; the counts follow on their own stream */
  uint32_t* pin_cnt = b.pinned_count;
  uint32_t* pin_off = b.pinned_count + HOST_MAX_CHUNKS; /* chunk c's n+1 relative offsets start at e0 + c */
  for (int c = 0; c < n_chunks; ++c) {
    const size_t e0 = chunk_begin(c), e1 = chunk_begin(c + 1);
    const size_t s0 = so[e0], s1 = so[e1], g0 = go[e0 * lf::NSEG], g1 = go[e1 * lf::NSEG];
    LF_CUDA(h, cudaStreamWaitEvent(st, b.ev_h2d[c], 0));
    lf_seeds ds = {b.seeds, b.seeds + stride, b.seeds + 2 * stride, b.seeds + 3 * stride, b.seeds + 4 * stride,
                   b.seed_off + e0, s1 - s0};
    lf_hits dh = {hits->x ? b.hits : nullptr, b.seg_off + e0 * lf::NSEG, g1 - g0, packed ? b.hits16 : nullptr,
                  packed ? b.origin16 : nullptr};
    lf_tracks dt = {b.hit_idx + s0 * lf::NL, b.seed_idx + s0, b.n_hits + s0, b.state + s0 * 5, b.quality + s0,
                    b.ev_off + e0 + c, b.n_tracks + c, stride - s0};
    const lf_status rs = launch<false>(h, &ds, &dh, e1 - e0, &dt, nullptr, st, e0);
    if (rs != LF_OK) return rs;
    LF_CUDA(h, cudaEventRecord(b.ev_comp[c], st));
    LF_CUDA(h, cudaStreamWaitEvent(hb.s_cnt, b.ev_comp[c], 0));
    LF_CUDA(h, cudaMemcpyAsync(pin_cnt + c, b.n_tracks + c, sizeof(uint32_t), cudaMemcpyDeviceToHost, hb.s_cnt));
    LF_CUDA(h, cudaMemcpyAsync(pin_off + e0 + c, b.ev_off + e0 + c, (e1 - e0) * sizeof(uint32_t), cudaMemcpyDeviceToHost, hb.s_cnt));
    LF_CUDA(h, cudaEventRecord(b.ev_cnt[c], hb.s_cnt));
  }
  return LF_OK;
}

/* Second half: as soon as a chunk's count is known its tracks go to their final dense position in the caller's arrays;
 * returns when the batch's last byte has arrived.  Does not wait for anything queued behind the batch. */
static lf_status host_collect(lf_handle* h, int slot) {
  HostBufs& hb = h->hb;
  HostSlot& b = hb.slot[slot];
  lf_tracks* out = &b.out;
  const size_t n_events = b.n_events;
  b.pending = false;
  if (n_events == 0) {
    out->event_offsets[0] = 0;
    *out->n_tracks = 0;
    return LF_OK;
  }
  uint32_t* pin_cnt = b.pinned_count;
  uint32_t* pin_off = b.pinned_count + HOST_MAX_CHUNKS;
  size_t running = 0;
  for (int c = 0; c < b.n_chunks; ++c) {
    const size_t e0 = b.bounds[c], e1 = b.bounds[c + 1];
    const size_t s0 = b.first_seed[c];
    LF_CUDA(h, cudaEventSynchronize(b.ev_cnt[c]));
    const size_t nt = pin_cnt[c];
    if (nt > 0) {
      LF_CUDA(h, cudaMemcpyAsync(out->hit_idx + running * lf::NL, b.hit_idx + s0 * lf::NL, nt * lf::NL * sizeof(int32_t), cudaMemcpyDeviceToHost, hb.s_d2h));
      LF_CUDA(h, cudaMemcpyAsync(out->seed_idx + running, b.seed_idx + s0, nt * sizeof(int32_t), cudaMemcpyDeviceToHost, hb.s_d2h));
      LF_CUDA(h, cudaMemcpyAsync(out->n_hits + running, b.n_hits + s0, nt * sizeof(int32_t), cudaMemcpyDeviceToHost, hb.s_d2h));
      LF_CUDA(h, cudaMemcpyAsync(out->state + running * 5, b.state + s0 * 5, nt * 5 * sizeof(float), cudaMemcpyDeviceToHost, hb.s_d2h));
      LF_CUDA(h, cudaMemcpyAsync(out->quality + running, b.quality + s0, nt * sizeof(float), cudaMemcpyDeviceToHost, hb.s_d2h));
    }
    const uint32_t* rel = pin_off + e0 + c;
    for (size_t e = e0; e < e1; ++e) out->event_offsets[e] = (uint32_t)(running + rel[e - e0]);
    running += nt;
  }
  out->event_offsets[n_events] = (uint32_t)running;
  *out->n_tracks = (uint32_t)running;
  /* the batch's kernels are done (its last count has arrived); wait for its last copy, not for the streams, which may
   * already hold the next batch */
  LF_CUDA(h, cudaEventRecord(b.ev_done, hb.s_d2h));
  LF_CUDA(h, cudaEventSynchronize(b.ev_done));
  return LF_OK;
}

} /* extern "C" */

/* ============================================================================================
 * lf_windows_static (include/lf.h): the search-window stage (a1 + a2) for callers that cannot allocate.
 *
 * The window kernel needs global memory besides the caller's inputs and outputs: its 64-byte window rows, the events'
 * equal-neighbour flags and look-back words, and the event ticket its persistent CTAs draw from.  lf_run takes that from
 * the workspace lf_create allocated.  Here it lives in the array below, which is part of the library's image: the driver
 * reserves it on every GPU that loads the library and keeps it until the process exits, so this entry point never
 * calls cudaMalloc / cudaFree (nor anything else that allocates device memory) and needs no handle.
 *
 * `lf_static_scratch` as written in HOST code is only the host-side shadow of the symbol, not an address the GPU can
 * use: the device address comes from cudaGetSymbolAddress, asked once per device with that device current (below).
 * ============================================================================================ */
namespace {
constexpr size_t STATIC_WIN_BYTES = (size_t)LF_STATIC_MAX_ROWS * lf::WIN_ROW * sizeof(uint32_t);  /* window rows */
constexpr size_t STATIC_STATE_BYTES = (size_t)LF_STATIC_MAX_EVENTS * sizeof(unsigned long long);  /* look-back words */
constexpr size_t STATIC_DUP_BYTES = (size_t)LF_STATIC_MAX_EVENTS * sizeof(uint32_t);              /* equal-neighbour flags */
constexpr size_t STATIC_TICKET_BYTES = 256;                                                        /* the event ticket */
constexpr size_t STATIC_SCRATCH_BYTES = STATIC_WIN_BYTES + STATIC_STATE_BYTES + STATIC_DUP_BYTES + STATIC_TICKET_BYTES;
static_assert(STATIC_SCRATCH_BYTES == LF_STATIC_SCRATCH_BYTES, "include/lf.h states the size of the static scratch");
constexpr int STATIC_STAGE_CAP = 8192; /* floats of shared memory for one event's hits: header + 32 KB stays under the 48 KB a
                                          kernel may use without raising an attribute; larger events read global memory */
struct StaticDevice {
  unsigned char* scratch = nullptr; /* device address of lf_static_scratch on this device */
  int sm_count = 0;
  bool ready = false;
};
StaticDevice g_static_dev[MAX_DEVICES];
std::mutex g_static_mutex;
} // namespace

static __device__ __align__(256) unsigned char lf_static_scratch[LF_STATIC_SCRATCH_BYTES];

extern "C" lf_status lf_windows_static(const lf_geometry* geometry, const lf_params* params, const lf_seeds* seeds,
                                       const lf_hits* hits, size_t n_events, int32_t* win_first, int32_t* win_count,
                                       void* cuda_stream) {
  /* ---- argument checks: all of them before the first CUDA call */
  if (!geometry || !params || !seeds || !hits)
    return fail(nullptr, LF_ERR_INVALID_ARG, "lf_windows_static: NULL geometry/params/seeds/hits");
  if (const char* why = validate(*geometry, *params)) return fail(nullptr, LF_ERR_INVALID_ARG, std::string("lf_windows_static: ") + why);
  if (params->hit_storage != 0)
    return fail(nullptr, LF_ERR_UNSUPPORTED, "lf_windows_static: fp32 hits only (hit_storage = 1 needs a scratch image of the hits)");
  const size_t sides = params->mode == 1 ? 2 : 1;
  if (n_events > (size_t)LF_STATIC_MAX_EVENTS || seeds->n_seeds > (size_t)LF_STATIC_MAX_ROWS / sides) {
    char msg[256];
    std::snprintf(msg, sizeof(msg),
                  "lf_windows_static: %zu events / %zu followed tracks exceed the static scratch (LF_STATIC_MAX_EVENTS = %d, "
                  "LF_STATIC_MAX_ROWS = %d): split the batch, or use lf_create + lf_run_debug",
                  n_events, seeds->n_seeds * sides, LF_STATIC_MAX_EVENTS, LF_STATIC_MAX_ROWS);
    return fail(nullptr, LF_ERR_CAPACITY, msg);
  }
  if (hits->n_hits >= (size_t)0x7fffffff) return fail(nullptr, LF_ERR_CAPACITY, "lf_windows_static: hit indices must fit int32");
  if (n_events == 0) {
    if (seeds->n_seeds != 0 || hits->n_hits != 0)
      return fail(nullptr, LF_ERR_INVALID_ARG, "lf_windows_static: n_events == 0 with non-empty seeds or hits");
    return LF_OK; /* nothing to write */
  }
  if (!seeds->event_offsets || !hits->seg_offsets) return fail(nullptr, LF_ERR_INVALID_ARG, "lf_windows_static: NULL offset table");
  if (seeds->n_seeds > 0 && (!seeds->x || !seeds->y || !seeds->tx || !seeds->ty || (!seeds->qop && params->mode == 0)))
    return fail(nullptr, LF_ERR_INVALID_ARG, "lf_windows_static: NULL seed array");
  if (hits->n_hits > 0 && !hits->x) return fail(nullptr, LF_ERR_INVALID_ARG, "lf_windows_static: NULL hit array");
  if (seeds->n_seeds > 0 && (!win_first || !win_count)) return fail(nullptr, LF_ERR_INVALID_ARG, "lf_windows_static: NULL output array");

  /* ---- once per device, with that device current: where the static array lives on it */
  int device = 0;
  LF_CUDA(nullptr, cudaGetDevice(&device));
  if (device < 0 || device >= MAX_DEVICES) return fail(nullptr, LF_ERR_UNSUPPORTED, "lf_windows_static: device index beyond the library's table");
  StaticDevice sd;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& slot = g_static_dev[device];
    if (!slot.ready) {
      int major = 0;
      LF_CUDA(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
      if (major < 10) return fail(nullptr, LF_ERR_UNSUPPORTED, "lf_windows_static: this library is built for sm_100a (Blackwell) only");
      LF_CUDA(nullptr, cudaDeviceGetAttribute(&slot.sm_count, cudaDevAttrMultiProcessorCount, device));
      unsigned char* ptr = nullptr;
      LF_CUDA(nullptr, cudaGetSymbolAddress((void**)&ptr, lf_static_scratch));
      if (!ptr) return fail(nullptr, LF_ERR_CUDA, "lf_windows_static: cudaGetSymbolAddress returned no address");
      /* The shared-memory limit of a kernel is a property of the kernel, and an lf_create with a small stage may have set
       * it below what this entry point launches with: raise it through the library's raise-only table (no later
       * lf_create can lower it again).  Sets a function attribute; allocates nothing. */
      const int smem_bytes = lf::HDR_BYTES + STATIC_STAGE_CAP * (int)sizeof(float);
      LF_CUDA(nullptr, raise_dynamic_smem((const void*)lf::lf_window_kernel<true, false>, 0, 0, 1, device, smem_bytes));
      LF_CUDA(nullptr, raise_dynamic_smem((const void*)lf::lf_window_kernel<true, true>, 1, 0, 1, device, smem_bytes));
      slot.scratch = ptr;
      slot.ready = true;
    }
    sd = slot;
  }

  lf::Consts consts;
  make_consts(*geometry, *params, consts);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint32_t* ticket = reinterpret_cast<uint32_t*>(sd.scratch + STATIC_WIN_BYTES + STATIC_STATE_BYTES + STATIC_DUP_BYTES);
  lf::EventArgs A;
  std::memset(&A, 0, sizeof(A));
  A.sx = seeds->x; A.sy = seeds->y; A.stx = seeds->tx; A.sty = seeds->ty; A.sqop = seeds->qop;
  A.seed_off = seeds->event_offsets;
  A.hx = hits->x; A.seg_off = hits->seg_offsets;
  A.n_events = (uint32_t)n_events;
  A.stage_cap = STATIC_STAGE_CAP;
  A.stage_cap_x = STATIC_STAGE_CAP;
  A.win = reinterpret_cast<uint32_t*>(sd.scratch);
  A.ev_state = reinterpret_cast<unsigned long long*>(sd.scratch + STATIC_WIN_BYTES);
  A.ev_dup = reinterpret_cast<uint32_t*>(sd.scratch + STATIC_WIN_BYTES + STATIC_STATE_BYTES);
  A.ticket = ticket;
  A.dbg.win_first = win_first;
  A.dbg.win_count = win_count;
  /* The array keeps what the previous call left.  Only the ticket must start at zero (the CTAs count events up from
   * it); window rows, flags and look-back words are written by the kernel before anybody reads them. */
  LF_CUDA(nullptr, cudaMemsetAsync(ticket, 0, sizeof(uint32_t), st));
  const int grid = (int)std::min<size_t>((size_t)sd.sm_count * 4, n_events);
  const size_t smem = (size_t)lf::HDR_BYTES + (size_t)STATIC_STAGE_CAP * sizeof(float);
  if (use_wide(*params)) lf::lf_window_kernel<true, true><<<grid, lf::WIN_THREADS, smem, st>>>(consts, A);
  else lf::lf_window_kernel<true, false><<<grid, lf::WIN_THREADS, smem, st>>>(consts, A);
  LF_CUDA(nullptr, cudaGetLastError());
  return LF_OK;
}
