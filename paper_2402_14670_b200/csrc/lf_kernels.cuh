/*
 * lf_kernels.cuh -- sm_100a device code of the Looking Forward hot path (include/lf.h, a1..a7).
 *
 * Execution model.  Four event kernels share one skeleton: persistent CTAs take events from an
 * atomic ticket; the event's 24 x-sorted hit segments are contiguous in HBM, so 1-D bulk async copies (TMA:
 * cp.async.bulk + mbarrier, SASS UBLKCP) stage them into shared memory (fetch_event: the whole event; fetch_event_x:
 * the six x layers in four runs, for the seeding kernel).  Each kernel then maps threads to the work item of its stage:
 *
 *   lf_window_kernel  a1/a2  one thread per (followed track, layer): one branch-free binary search over the segment
 *                            for the window centre, two short ones for the edges, n_window cap; writes a 64-byte row
 *                            per followed track: 12 packed windows + x_mag, tx, q/p, flags.
 *   lf_seed_kernel    a3     one warp per followed track.  For a fixed h0 the h2 hits that pass the magnet-opening
 *                            cut form a contiguous x interval: lanes = h0 bracket a conservative superset by two
 *                            shuffle searches; a warp prefix scan of the bracket sizes re-maps the work to lanes =
 *                            candidate doublets, where the exact fp32 predicate decides (bit-exact with the
 *                            all-pairs definition) and the closest h1 / chi2 cut follow in the same lane; rank
 *                            selection on (chi2, candidate order) keeps the n smallest, sorted.  seed_triplets_h2
 *                            is the same with pairs of doublets evaluated in __half2 (hit_storage = 1);
 *                            seed_triplets_wide handles windows of up to 64 hits and the no-UT tuning.
 *   lf_extend_kernel  a4/a5  one thread per triplet: parabola through the triplet, closest hit in the 9 other windows
 *                            (three searches in lockstep per station), chi2 cuts, hit-count rule; accepted
 *                            candidates are ballot-compacted in (seed, k) order into 16-byte records.
 *   lf_fit_kernel     a6/a7  one thread per accepted record: both least-squares fits (geometry sums from a
 *                            per-presence-mask LUT), Q, lowest (Q, k) per seed by shared-memory atomicMin; the winning
 *                            thread writes the 20-word track record; the CTA lists the event's tracks in seed order.
 *                            Stream compaction in the same kernel: a decoupled look-back over the events' track counts
 *                            gives every event its offset in the dense output, and the CTA that fitted the event copies
 *                            its tracks there (no scan kernel, no compaction kernel).
 *   lf_pack_hits_kernel, lf_validate_kernel: fp16 copy of the hits (hit_storage = 1); input preconditions.
 *
 * Arithmetic contract: fp32, one rounding per operation, in the order DESIGN.md "Canonical
 * arithmetic" lists (compile with -fmad=false, no fast-math; '/' is IEEE division; explicit __fmaf_rn appears only
 * where a value brackets a search and decides nothing).  This file is written from PAPER.md + DESIGN.md and shares
 * nothing with oracle/.
 */
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

namespace lf {

constexpr int NL = 12;
constexpr int NSEG = 24;
constexpr int H16_SHIFT = 3;   /* fp16 hit storage: 2^H16_SHIFT hits share one fp32 origin (include/lf.h, lf_pack_hits) */
constexpr int WIN_ROW = 16;    /* words per followed track in the window table: 12 packed windows + x_mag, tx, q/p, flags */
constexpr uint32_t ROW_LOW_P = 1u; /* flags: the seed's momentum is below p_same_bend (filter 1 applies) */
constexpr int REC_WORDS = 20;  /* 12 hit idx, seed, n_hits, 5 state, Q */
constexpr int TRIP_BUF = 64;   /* per-warp triplet key buffer */
constexpr int MAX_NT = 16;     /* == LF_MAX_TRIPLETS (narrow kernels) */
constexpr int MAX_NT_WIDE = 32; /* == LF_MAX_TRIPLETS_WIDE */
constexpr int WIN_THREADS = 256;     /* window kernel: threads per CTA ... */
constexpr int WIN_THREADS_BIG = 512; /* ... or, when a large stage leaves few CTAs per SM, this many (lf_create picks) */
/* Two builds of every event kernel (template parameter WIDE):
 *   narrow  n_window <= 32, n_triplets <= 16, one followed track ("row") per seed: the with-UT tuning; a search
 *           window fits one hit per lane, window-relative hit indices take 5 bits;
 *   wide    n_window <= 64, n_triplets <= 32, `sides` rows per seed (row = seed*sides + side): the no-UT tuning
 *           (two window sides per VELO track, 64 hits, 20 triplets), and the with-UT
 *           tuning with caps beyond the narrow limits (sides = 1). */
template <bool WIDE>
struct Fmt {
  static constexpr int WB = WIDE ? 7 : 6;             /* bits of the hit count in a packed window word */
  static constexpr uint32_t WMASK = (1u << WB) - 1u;
  static constexpr int IB = WIDE ? 6 : 5;             /* bits of a window-relative hit index in a triplet code */
  static constexpr uint32_t IMASK = (1u << IB) - 1u;
  static constexpr int EDGE_STEPS = WIDE ? 7 : 6;     /* window-edge searches span n_window + 1 hits */
  static constexpr uint32_t TOPB = WIDE ? 256u : 128u; /* first stride (bytes) of a search inside one window */
  static constexpr int KB = WIDE ? 5 : 4;             /* bits of the triplet index k */
  /* tag of a candidate record: seed inside the event | layer set << 25 | window side << 26 | k << 27 */
  static constexpr int SIE_BITS = 25;
  static constexpr uint32_t SIE = (1u << SIE_BITS) - 1u;
  static constexpr int SET_SHIFT = 25, SIDE_SHIFT = 26, K_SHIFT = 27;
  typedef typename std::conditional<WIDE, uint32_t, uint16_t>::type code_t; /* stored triplet code */
};
constexpr int SEED_WARPS = 8;
constexpr int SEED_THREADS = SEED_WARPS * 32;
constexpr int FIT_THREADS = 256;
constexpr int FIT_CHUNK = 256; /* most rows of one event whose windows the extension kernel stages at a time (<= FIT_THREADS, even);
                                 EventArgs.ext_chunk is the handle's choice, 256 or 128 */
constexpr int N_TICKETS = 4; /* window, seed, extend, fit */
constexpr unsigned FULL = 0xffffffffu;
constexpr float INTERVAL_MARGIN = 0.1f; /* mm added to the magnet tolerance when bracketing h2 (superset only) */

/* Geometry-derived constants and tunables, computed once on the host in fp32 (lf_api.cu). */
struct Consts {
  float z[NL], tana[NL], inv_tan[NL], dzs[NL], dzm[NL], d[NL], w[NL];
  float z_seed, z_mag, kick, dr, K[2], poly[5], mag_dz_seed;
  float inv_dz_ac[2], zmag_a[2], inv_r[2], inv_abs_zmag_a[2], tolmax_over_zmag[2], D10[2], D20[2], W10[2], W20[2], inv_det[2], inv_D10[2];
  float dz_state, ds, ws, dws;
  int polarity;
  float T_triplet, T_x, T_uv_slope, T_uv_min, T_ty, inv_Tx, inv_Ty, T_Q, C_nhits[4];
  int n_window, n_triplets, min_hits;
  float xtol_base, xtol_inv_p, x_asym, uv_half_width;
  float p_same_bend, mag_tol_base, mag_tol_inv_p, mag_tol_tx, mag_tol_max;
  /* no-UT tuning */
  int mode, sides;                 /* mode 1: sides = 2 (LEFT / RIGHT windows of Eq. 8) */
  float inv_p_min, inv_pt_min;     /* 1 / velo_p_min, 1 / velo_pt_min */
  float xtol_poly[8], x_overlap;   /* Eq. (7) / Table 5; Eq. (8) */
  /* full Eq. (9) */
  int qop_mode;
  float poly2d[5][10];
};

struct FitLut;

struct DebugOut {
  int32_t *win_first, *win_count, *n_triplets, *trip_hits, *trip_set;
  float* trip_chi2;
  int32_t* cand_hits;
  float* cand_quality;
  unsigned long long* counters; /* LF_N_COUNTERS work counters of the debug build (include/lf.h, lf_run_counters) */
};

/* Arguments common to the three event kernels + the per-stage tables (library workspace). */
struct EventArgs {
  const float *sx, *sy, *stx, *sty, *sqop;
  const uint32_t* seed_off;
  const float* hx;
  const uint32_t* seg_off;
  /* hit_storage = 1: fp16 copy of the hits (block-offset encoding, see lf_pack_hits_kernel); the window
   * and seed kernels stage from it when hx16 != nullptr */
  const __half* hx16;
  const float* origin16;
  uint32_t event_base;  /* index of the launch's first event in the arrays hx16 / origin16 were packed for (lf_run_host chunks) */
  float* hx_scratch;    /* hit_storage = 1: fp32 image of the events that do not fit the stage (decoded once, by the kernel
                           launched with scratch_writer != 0; read by all of them through HitView<false>) */
  int scratch_writer;
  uint32_t n_events;
  int stage_cap;        /* floats of shared memory available for one event's hits */
  int stage_cap_x;      /* the stage of the seeding kernel (fetch_event_x), known to the kernel that writes the fp16 scratch image */
  int ext_chunk;        /* extension kernel: rows staged at a time (lf_create picks the size that keeps most CTAs per SM) */
  uint32_t* ticket;     /* this kernel's event ticket */
  /* per followed track ("row" = seed*sides + side; narrow kernels: row = seed) */
  uint32_t* win;        /* n_rows*WIN_ROW: 12 x ((first_in_event << WB) | count), then x_mag, tx, q/p (mode 1: the assumed
                           1/p), flags */
  void* trip_code;      /* n_rows*NT Fmt::code_t: set<<3IB | h0<<2IB | h2<<IB | h1 (window-relative), sorted */
  uint8_t* n_trip;      /* n_rows */
  int32_t* ws_rec;      /* n_seeds * REC_WORDS */
  int32_t* ws_nh;       /* n_seeds: 1 if the seed has a track, else 0 */
  int32_t* ws_rank;     /* n_seeds: the events' track lists: entry (first seed of the event + r) = seed of the event's r-th track */
  uint32_t* ev_count;   /* n_events */
  uint4* acc_rec;       /* n_rows*NT: candidates that passed the hit-count rule: 3 words of hit codes (byte l = hit of
                           layer l inside its window, 0xFF = none), then the tag seed inside the event | layer set << 25 |
                           window side << 26 | k << 27; dense per event */
  uint32_t* ev_acc;     /* n_events: number of such records of the event */
  const struct FitLut* fit_lut; /* 4096: per presence mask */
  uint32_t* ev_dup;     /* n_events: written by the window kernel, != 0 if two neighbouring staged hits are equal */
  unsigned long long* ev_state; /* n_events: look-back words of the fit kernel's stream compaction, zeroed by the window kernel */
  DebugOut dbg;
};

/* Head of the dynamic shared memory of every event kernel; the staged hits follow it. */
struct __align__(16) CtaHeader {
  unsigned long long mbar;
  int seg[NSEG + 1];
  int ev;
  int nsteps; /* binary-search steps that cover the event's longest segment */
  int warp_tot[8];
  int dup; /* != 0: the event may hold equal neighbouring hits (closest_hit must resolve runs of ties) */
  int blk_pref[NSEG + 1]; /* fp16 hit storage: decode trips (32 hits each, one per warp pass) in front of each segment of the event */
  int xdelta[NL];         /* seeding kernel: hit i of an x layer l lives at stage position i - xdelta[l] (fetch_event_x) */
};
constexpr int HDR_BYTES = (sizeof(CtaHeader) + 15) & ~15;

struct EventCtx {
  uint32_t ev, h0;
  int nh, skew;
  bool staged;
  const float* gview; /* the event's hits in global memory (events that do not fit the stage) */
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

/* The one dynamic shared-memory array: CtaHeader, staged hits, then the kernel's own tables. */
extern __shared__ __align__(16) unsigned char lf_smem[];
__device__ __forceinline__ float* stage_buf() { return reinterpret_cast<float*>(lf_smem + HDR_BYTES); }

/* View of the current event's hits, indexed event-relative.  Staged: shared memory (LDS);
 * fallback for events larger than the stage buffer: read-only global loads. */
__device__ __forceinline__ float lds_f32(uint32_t addr) {
  float v;
  asm("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
  return v;
}
/* Besides operator[], a view hands out positions (`pos_t`) for searches whose steps are "advance, bound check,
 * load, compare, select": 32-bit shared-memory byte addresses for the staged hits, pointers otherwise. */
template <bool STAGED>
struct HitView;
template <>
struct HitView<true> {
  uint32_t base; /* shared-memory byte address of hit 0 of the event */
  __device__ __forceinline__ explicit HitView(int skew) : base(smem_u32(stage_buf()) + 4u * (uint32_t)skew) {}
  __device__ __forceinline__ float operator[](int i) const { return lds_f32(base + 4u * (uint32_t)i); }
  typedef uint32_t pos_t;
  __device__ __forceinline__ pos_t pos(int i) const { return base + 4u * (uint32_t)i; }
  static __device__ __forceinline__ pos_t adv(pos_t p, int n) { return p + 4u * (uint32_t)n; }
  static __device__ __forceinline__ float before(pos_t p) { return lds_f32(p - 4u); } /* the hit in front of p */
  static __device__ __forceinline__ float at(pos_t p) { return lds_f32(p); }
  static __device__ __forceinline__ int diff(pos_t a, pos_t b) { return (int)(a - b) >> 2; }
};
template <>
struct HitView<false> {
  const float* p;
  __device__ __forceinline__ explicit HitView(const float* first) : p(first) {}
  __device__ __forceinline__ float operator[](int i) const { return __ldg(p + i); }
  typedef const float* pos_t;
  __device__ __forceinline__ pos_t pos(int i) const { return p + i; }
  static __device__ __forceinline__ pos_t adv(pos_t q, int n) { return q + n; }
  static __device__ __forceinline__ float before(pos_t q) { return __ldg(q - 1); }
  static __device__ __forceinline__ float at(pos_t q) { return __ldg(q); }
  static __device__ __forceinline__ int diff(pos_t a, pos_t b) { return (int)(a - b); }
};

/* Branch-free binary search over the x-sorted positions [a, e): a + number of leading hits with x < v
 * (INCLUSIVE == false: lower bound) or x <= v (true: upper bound).  Needs 2^NSTEPS > e - a. */
template <int NSTEPS, bool INCLUSIVE, class HV>
__device__ __forceinline__ typename HV::pos_t bound_pos(typename HV::pos_t a, typename HV::pos_t e, float v) {
  typename HV::pos_t p = a;
#pragma unroll
  for (int s = NSTEPS - 1; s >= 0; --s) {
    const typename HV::pos_t q = HV::adv(p, 1 << s);
    if (q <= e) {
      const float xm = HV::before(q);
      if (INCLUSIVE ? (xm <= v) : (xm < v)) p = q;
    }
  }
  return p;
}
template <class HV>
__device__ __forceinline__ typename HV::pos_t lower_pos(typename HV::pos_t a, typename HV::pos_t e, float v, int nsteps) {
  if (nsteps <= 8) return bound_pos<8, false, HV>(a, e, v);
  typename HV::pos_t p = a;
  for (int s = nsteps - 1; s >= 0; --s) {
    const typename HV::pos_t q = HV::adv(p, 1 << s);
    if (q <= e && HV::before(q) < v) p = q;
  }
  return p;
}

/* Takes the next event and stages its hits.  Called by every thread of the CTA; returns false when
 * the batch is exhausted.  Hit i of the event then lives at stage_buf()[skew + i].  `while_loading` is called once by
 * every thread of an event that was taken, after the bulk copy has been issued and before anybody waits for it: work
 * that does not touch the stage hides behind the copy's latency (the extension and fit kernels pull the event's tables
 * into L2 there; the fit kernel also resolves the output offset of an earlier event). */
struct NoHook {
  __device__ __forceinline__ void operator()() const {}
};
template <class Hook = NoHook>
__device__ __forceinline__ bool fetch_event(const EventArgs& A, uint32_t& phase, EventCtx& E, Hook while_loading = Hook()) {
  CtaHeader& H = *reinterpret_cast<CtaHeader*>(lf_smem);
  float* buf = stage_buf();
  const int tid = threadIdx.x;
  __syncthreads(); /* previous event fully retired: header, stage buffer and tables reusable */
  if (tid == 0) H.ev = (int)atomicAdd(A.ticket, 1u);
  __syncthreads();
  E.ev = (uint32_t)H.ev;
  if (E.ev >= A.n_events) return false;
  const uint32_t* so = A.seg_off + (size_t)E.ev * NSEG;
  E.h0 = so[0];
  E.nh = (int)(so[NSEG] - E.h0);
  if (tid <= NSEG) H.seg[tid] = (int)(so[tid] - E.h0);
  if (tid < 32) { /* longest segment -> number of binary-search steps */
    int len = (tid < NSEG) ? (int)(so[tid + 1] - so[tid]) : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) len = max(len, __shfl_xor_sync(FULL, len, o));
    if (tid == 0) H.nsteps = 32 - __clz(len);
  }
  if (tid == 32) H.dup = (int)A.ev_dup[E.ev]; /* meaningful in the seed and fit kernels only */
  const float* gsrc = A.hx + E.h0;
  E.staged = E.nh + 4 <= A.stage_cap;
  const bool from16 = A.hx16 != nullptr;
  E.skew = from16 ? 0 : (int)((reinterpret_cast<uintptr_t>(gsrc) >> 2) & 3);
  E.gview = from16 ? A.hx_scratch + E.h0 : gsrc;
  if (from16) {
    /* fp16 hit storage (lf_pack_hits_kernel): x~ = origin(block of 8 hits) + half.  One warp decodes one trip of 32 hits
     * (counted from the start of each segment) at a time: a 64-byte load of halves, the origins, 32 fp32 stores into the
     * stage (or, for an event larger than the stage, into the library's fp32 scratch image, once per lf_run). */
    if (tid < 32) {
      const int nb = (tid < NSEG) ? (int)((so[tid + 1] - so[tid] + 31u) >> 5) : 0;
      int incl = nb;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, o);
        if (tid >= o) incl += v;
      }
      if (tid <= NSEG) H.blk_pref[tid] = incl - nb; /* entry NSEG = all blocks of the event */
    }
    __syncthreads();
    /* The scratch writer (the window kernel) also decodes into the scratch image every event that the seeding kernel's
     * half-size x-layer stage cannot hold (its runs take at most 24 floats of alignment gaps). */
    bool to_scratch = false;
    if (A.scratch_writer) {
      const int nx = (int)((so[2] - so[0]) + (so[10] - so[6]) + (so[18] - so[14]) + (so[24] - so[22]));
      to_scratch = !E.staged || nx + 28 > A.stage_cap_x;
    }
    if (E.staged || to_scratch) {
      float* scr = A.hx_scratch + E.h0;
      const int lane = tid & 31, n_blk = H.blk_pref[NSEG];
      const int pref = (lane < NSEG) ? H.blk_pref[lane] : 0x7FFFFFFF;
      for (int blk = tid >> 5; blk < n_blk; blk += (int)(blockDim.x >> 5)) {
        const int sg = __popc(__ballot_sync(FULL, pref <= blk)) - 1; /* the last segment that starts at or before blk */
        const int b = blk - H.blk_pref[sg];
        const uint32_t S = so[sg];
        const int i = 32 * b + lane;
        if (i < (int)(so[sg + 1] - S)) {
          const float v = __ldg(A.origin16 + ((S >> H16_SHIFT) + ((A.event_base + E.ev) * NSEG + (uint32_t)sg) + (uint32_t)(i >> H16_SHIFT))) +
                          __half2float(A.hx16[S + i]);
          if (E.staged) buf[(int)(S - E.h0) + i] = v;
          if (to_scratch) scr[(int)(S - E.h0) + i] = v;
        }
      }
      if (to_scratch) __threadfence(); /* the scratch image is read back by this CTA and by the later kernels */
    }
  } else if (E.staged) {
    /* the 16-byte aligned interior goes by TMA, the ragged head/tail by plain loads */
    const int head = min(E.nh, (4 - E.skew) & 3);
    const int bulk = (E.nh - head) & ~3;
    const int tail = E.nh - head - bulk;
    if (tid == 0 && bulk > 0) {
      fence_proxy_async();
      mbar_expect_tx(&H.mbar, (uint32_t)bulk * 4u);
      bulk_g2s(buf + E.skew + head, gsrc + head, (uint32_t)bulk * 4u, &H.mbar);
    }
    if (tid < head) buf[E.skew + tid] = gsrc[tid];
    if (tid >= 32 && tid < 32 + tail) buf[E.skew + head + bulk + (tid - 32)] = gsrc[head + bulk + (tid - 32)];
    while_loading();
    if (bulk > 0) {
      if (tid == 0) mbar_wait(&H.mbar, phase); /* one thread polls; the barrier below publishes */
      phase ^= 1u;
    }
  }
  if (from16 || !E.staged) while_loading();
  __syncthreads();
  return true;
}

/* fetch_event for the seeding kernel, which touches the six x layers only (0, 3, 4, 7, 8, 11): they form
 * four contiguous runs of the event's hits, staged back to back by four bulk copies, so that the stage holds half an
 * event and large events keep their CTAs per SM.  Hit i (event-relative) of x layer l then lives at stage position
 * i - H.xdelta[l]; for an event that does not fit even so, xdelta = 0 and the hits are read from global memory. */
__device__ __forceinline__ bool fetch_event_x(const EventArgs& A, uint32_t& phase, EventCtx& E) {
  CtaHeader& H = *reinterpret_cast<CtaHeader*>(lf_smem);
  float* buf = stage_buf();
  const int tid = threadIdx.x;
  __syncthreads();
  if (tid == 0) H.ev = (int)atomicAdd(A.ticket, 1u);
  __syncthreads();
  E.ev = (uint32_t)H.ev;
  if (E.ev >= A.n_events) return false;
  const uint32_t* so = A.seg_off + (size_t)E.ev * NSEG;
  E.h0 = so[0];
  E.nh = (int)(so[NSEG] - E.h0);
  if (tid == 32) H.dup = (int)A.ev_dup[E.ev];
  const bool from16 = A.hx16 != nullptr;
  E.skew = 0;
  E.gview = from16 ? A.hx_scratch + E.h0 : A.hx + E.h0;
  /* the four runs: segments [0,2), [6,10), [14,18), [22,24); stage base of run r keeps the 16-byte phase of its source */
  int rs[4], rn[4], rb[4];
  {
    const int sa[4] = {0, 6, 14, 22}, sb[4] = {2, 10, 18, 24};
    int pos = 0;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      rs[r] = (int)(so[sa[r]] - E.h0);
      rn[r] = (int)(so[sb[r]] - so[sa[r]]);
      const int sk = from16 ? 0 : (int)((reinterpret_cast<uintptr_t>(A.hx + E.h0 + rs[r]) >> 2) & 3);
      rb[r] = pos + sk;
      pos = (rb[r] + rn[r] + 3) & ~3;
    }
    E.staged = pos + 4 <= A.stage_cap;
  }
  if (tid < NL) {
    const int r = (tid == 0) ? 0 : ((tid <= 4) ? 1 : ((tid <= 8) ? 2 : 3)); /* run of layer tid (x layers only matter) */
    H.xdelta[tid] = E.staged ? ((r == 0 ? rs[0] - rb[0] : (r == 1 ? rs[1] - rb[1] : (r == 2 ? rs[2] - rb[2] : rs[3] - rb[3])))) : 0;
  }
  if (from16) {
    if (tid < 32) {
      const int nb = (tid < NSEG) ? (int)((so[tid + 1] - so[tid] + 31u) >> 5) : 0;
      int incl = nb;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, o);
        if (tid >= o) incl += v;
      }
      if (tid <= NSEG) H.blk_pref[tid] = incl - nb;
    }
    __syncthreads();
    if (E.staged) { /* oversized events were decoded into the scratch image by the window kernel */
      const int lane = tid & 31, n_blk = H.blk_pref[NSEG];
      const int pref = (lane < NSEG) ? H.blk_pref[lane] : 0x7FFFFFFF;
      for (int blk = tid >> 5; blk < n_blk; blk += (int)(blockDim.x >> 5)) {
        const int sg = __popc(__ballot_sync(FULL, pref <= blk)) - 1;
        const int l = sg >> 1;
        if ((l & 3) != 0 && (l & 3) != 3) continue; /* a u/v layer: not staged here */
        const int b = blk - H.blk_pref[sg];
        const uint32_t S = so[sg];
        const int i = 32 * b + lane;
        if (i < (int)(so[sg + 1] - S))
          buf[(int)(S - E.h0) - H.xdelta[l] + i] =
              __ldg(A.origin16 + ((S >> H16_SHIFT) + ((A.event_base + E.ev) * NSEG + (uint32_t)sg) + (uint32_t)(i >> H16_SHIFT))) +
              __half2float(A.hx16[S + i]);
      }
    }
  } else if (E.staged) {
    /* per run: the 16-byte aligned interior by TMA, the ragged head / tail (at most 3 hits each) by plain loads */
    const float* g0 = A.hx + E.h0;
    int head[4], bulk[4];
    uint32_t bytes = 0;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      head[r] = min(rn[r], (4 - (rb[r] & 3)) & 3);
      bulk[r] = (rn[r] - head[r]) & ~3;
      bytes += (uint32_t)bulk[r] * 4u;
    }
    if (tid == 0 && bytes > 0) {
      fence_proxy_async();
      mbar_expect_tx(&H.mbar, bytes);
#pragma unroll
      for (int r = 0; r < 4; ++r)
        if (bulk[r] > 0) bulk_g2s(buf + rb[r] + head[r], g0 + rs[r] + head[r], (uint32_t)bulk[r] * 4u, &H.mbar);
    }
    if (tid >= 64 && tid < 96) {
      const int r = (tid - 64) >> 3, e = (tid - 64) & 7; /* e < 4: head element e; else tail element e - 4 */
      const int hd = (r == 0) ? head[0] : ((r == 1) ? head[1] : ((r == 2) ? head[2] : head[3]));
      const int bk = (r == 0) ? bulk[0] : ((r == 1) ? bulk[1] : ((r == 2) ? bulk[2] : bulk[3]));
      const int n = (r == 0) ? rn[0] : ((r == 1) ? rn[1] : ((r == 2) ? rn[2] : rn[3]));
      const int s_ = (r == 0) ? rs[0] : ((r == 1) ? rs[1] : ((r == 2) ? rs[2] : rs[3]));
      const int b_ = (r == 0) ? rb[0] : ((r == 1) ? rb[1] : ((r == 2) ? rb[2] : rb[3]));
      const int i = (e < 4) ? e : hd + bk + (e - 4);
      if ((e < 4) ? (e < hd) : (i < n)) buf[b_ + i] = g0[s_ + i];
    }
    if (bytes > 0) {
      if (tid == 0) mbar_wait(&H.mbar, phase);
      phase ^= 1u;
    }
  }
  __syncthreads();
  return true;
}

/* Closest hit to `pred` in the x-sorted window [f, f+n), n <= 32: first x >= pred by binary search,
 * then compare the two neighbours; ties -> lower index, including runs of equal distance on the low
 * side (equals a linear argmin with strict '<'); such a run needs two equal neighbouring hits, so the
 * walk is skipped when the event has none (`dup` == false).  Returns the event-relative index, or -1 if
 * n == 0, and in `dist` the distance |x - pred| of that hit (x - pred and pred - x round to the same
 * magnitude, so dist*dist is bit-identical to (x - pred)^2).  Generic version (global-memory view). */
template <bool WIDE, class HV>
__device__ __forceinline__ int closest_hit(const HV& hx, int f, int n, float pred, bool dup, float& dist) {
  if (n <= 0) return -1;
  const int e = f + n;
  int pos = f;
#pragma unroll
  for (int s = Fmt<WIDE>::EDGE_STEPS - 1; s >= 0; --s) {
    const int probe = pos + (1 << s);
    if (probe <= e && hx[probe - 1] < pred) pos = probe;
  }
  if (pos == f) {
    dist = hx[f] - pred;
    return f;
  }
  int k = pos - 1;
  const float dk = pred - hx[k];
  if (pos < e) {
    const float dh = hx[pos] - pred;
    if (!(dk <= dh)) {
      dist = dh;
      return pos;
    }
  }
  dist = dk;
  if (dup) /* only events with equal neighbouring hits can have a run of ties */
    while (k > f && (pred - hx[k - 1]) == dk) --k;
  return k;
}

/* The same on the staged hits: positions are 32-bit shared-memory byte addresses, so one search step is
 * add, bound check, LDS, compare, select. */
template <bool WIDE>
__device__ __forceinline__ int closest_hit(const HitView<true>& hx, int f, int n, float pred, bool dup, float& dist) {
  if (n <= 0) return -1;
  const uint32_t a = hx.base + 4u * (uint32_t)f;
  const uint32_t end = a + 4u * (uint32_t)n;
  uint32_t p = a;
#pragma unroll
  for (uint32_t s = Fmt<WIDE>::TOPB; s >= 4u; s >>= 1) {
    const uint32_t q = p + s;
    if (q <= end && lds_f32(q - 4u) < pred) p = q;
  }
  if (p == a) {
    dist = lds_f32(a) - pred;
    return f;
  }
  const float dk = pred - lds_f32(p - 4u);
  if (p < end) {
    const float dh = lds_f32(p) - pred;
    if (!(dk <= dh)) {
      dist = dh;
      return f + (int)((p - a) >> 2);
    }
  }
  dist = dk;
  uint32_t k = p - 4u;
  if (dup)
    while (k > a && (pred - lds_f32(k - 4u)) == dk) k -= 4u;
  return f + (int)((k - a) >> 2);
}

/* G independent closest-hit searches in lockstep, branch-free: the G chains of dependent LDS overlap
 * (instruction-level parallelism instead of occupancy).  ww[g] is the packed window (first << 6 | count),
 * krel[g] the index of the closest hit inside its window (-1 and dist = +inf if the window is empty). */
template <int G, bool WIDE>
__device__ __forceinline__ void closest_group(const HitView<true>& hx, const uint32_t (&ww)[G], const float (&pred)[G],
                                              bool dup, int (&krel)[G], float (&dist)[G]) {
  const float INF = __int_as_float(0x7f800000);
  const uint32_t base = hx.base;
  uint32_t a[G], end[G], p[G];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    a[g] = base + 4u * (ww[g] >> Fmt<WIDE>::WB);
    end[g] = a[g] + 4u * (ww[g] & Fmt<WIDE>::WMASK);
    p[g] = a[g];
  }
#pragma unroll
  for (uint32_t s = Fmt<WIDE>::TOPB; s >= 4u; s >>= 1) {
#pragma unroll
    for (int g = 0; g < G; ++g) {
      const uint32_t q = p[g] + s;
      const float x = (q <= end[g]) ? lds_f32(q - 4u) : INF;
      p[g] = (x < pred[g]) ? q : p[g];
    }
  }
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const float xl = (p[g] > a[g]) ? lds_f32(p[g] - 4u) : -INF;
    const float xh = (p[g] < end[g]) ? lds_f32(p[g]) : INF;
    const float dk = pred[g] - xl, dh = xh - pred[g];
    const bool right = !(dk <= dh); /* ties -> lower index */
    uint32_t k = right ? p[g] : p[g] - 4u;
    dist[g] = right ? dh : dk;
    if (dup && !right)
      while (k > a[g] && (pred[g] - lds_f32(k - 4u)) == dk) k -= 4u;
    krel[g] = (int)(k - a[g]) >> 2;
  }
}
template <int G, bool WIDE>
__device__ __forceinline__ void closest_group(const HitView<false>& hx, const uint32_t (&ww)[G], const float (&pred)[G],
                                              bool dup, int (&krel)[G], float (&dist)[G]) {
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int f = (int)(ww[g] >> Fmt<WIDE>::WB);
    dist[g] = __int_as_float(0x7f800000);
    const int k = closest_hit<WIDE>(hx, f, (int)(ww[g] & Fmt<WIDE>::WMASK), pred[g], dup, dist[g]);
    krel[g] = (k < 0) ? -1 : k - f;
  }
}

/* ============================================================================================
 * a1/a2: search windows.  One thread per (seed, layer, edge).
 * ============================================================================================ */
template <bool DEBUG, bool WIDE, bool STAGED>
__device__ __forceinline__ void windows_of_event(const Consts& C, const EventArgs& A, const CtaHeader& H,
                                                 const EventCtx& E, const HitView<STAGED>& hx) {
  typedef HitView<STAGED> HV;
  typedef typename HV::pos_t pos_t;
  typedef Fmt<WIDE> F;
  const int tid = threadIdx.x;
  const uint32_t s0 = A.seed_off[E.ev], s1 = A.seed_off[E.ev + 1];
  const int sides = WIDE ? C.sides : 1;
  const int per_seed = sides * NL;
  const int n_items = (int)(s1 - s0) * per_seed;
  const int nsteps = H.nsteps;
  const bool pol_pos = C.polarity > 0;
  const int halfw = C.n_window / 2, reach = C.n_window + 1;
  for (int it = tid; it < n_items; it += (int)blockDim.x) {
    const int q12 = it / NL; /* (seed, side) pair; sides is 1 or 2, so no division by a run-time value */
    const int layer = it - q12 * NL;
    const int sl = WIDE ? (q12 >> (sides >> 1)) : q12;
    const int side = WIDE ? (q12 & (sides - 1)) : 0;
    const uint32_t seed = s0 + (uint32_t)sl;
    const size_t row = (size_t)seed * sides + side;
    const float x = __ldg(A.sx + seed), y = __ldg(A.sy + seed), tx = __ldg(A.stx + seed), ty = __ldg(A.sty + seed);
    const int zone = (ty >= 0.0f) ? 1 : 0;
    float lo, hi;
    if (WIDE && C.mode == 1) {
      /* no-UT: straight-line extrapolation of the VELO track, assumed minimum momentum,
       * x_tol of Eq. (7), double-sided windows of Eq. (8) */
      const float s2 = tx * tx + ty * ty;
      const float sin_theta = sqrtf(s2 / (1.0f + s2));
      const float inv_p = fminf(C.inv_p_min, sin_theta * C.inv_pt_min);
      const float xe = x + tx * C.dzs[layer];
      float ctr = xe, tol;
      if (is_uv(layer)) {
        const float yl = y + ty * C.dzs[layer];
        ctr = xe + yl * C.tana[layer];
        tol = C.uv_half_width;
      } else {
        const float* c = C.xtol_poly;
        tol = inv_p * (((c[0] + tx * (c[1] + c[2] * tx)) + (ty * ty) * (c[3] + tx * (c[4] + c[5] * tx))) +
                       inv_p * (c[6] * tx + c[7] * inv_p));
      }
      lo = (side == 0) ? ctr - tol : ctr - C.x_overlap;
      hi = (side == 0) ? ctr + C.x_overlap : ctr + tol;
    } else {
      /* a1: pT-kick extrapolation */
      const float qop = __ldg(A.sqop + seed);
      const float aq = fmaxf(fabsf(qop), 1e-6f);
      const float x_mag = x + tx * C.mag_dz_seed;
      const float txp = tx + C.kick * qop;
      const float xc = x_mag + txp * C.dzm[layer];
      if (!is_uv(layer)) { /* PAPER.md:181-200, Eq. (3) */
        const float x_tol = C.xtol_base + C.xtol_inv_p * aq;
        const bool q_pos = qop > 0.0f;
        const float a_left = (q_pos == pol_pos) ? C.x_asym : 0.0f;
        const float a_right = (q_pos != pol_pos) ? C.x_asym : 0.0f;
        lo = (xc - x_tol) - a_left;
        hi = (xc + x_tol) + a_right;
      } else {
        const float yl = y + ty * C.dzs[layer];
        const float ctr = xc + yl * C.tana[layer];
        lo = ctr - C.uv_half_width;
        hi = ctr + C.uv_half_width;
      }
    }
    const int sb = H.seg[layer * 2 + zone], se = H.seg[layer * 2 + zone + 1];
    /* a2.  With c = lower_bound(mid) the window [first, last) = [lower_bound(lo), upper_bound(hi))
     * is capped to [max(first, c - n/2), min(last, c + n/2)) iff it holds more than n = n_window hits.  Both
     * the test and the result only need first and last clipped to c -/+ (n + 1), so after one search over
     * the segment the two edges are short searches next to c (lo <= mid <= hi puts c inside the window;
     * an empty interval lo > hi, possible in the no-UT mode with a negative x_tol, gives first >= last = empty). */
    const pos_t pb = hx.pos(sb), pe = hx.pos(se);
    const float midv = (lo + hi) * 0.5f;
    const pos_t pc = lower_pos<HV>(pb, pe, midv, nsteps);
    const int c = sb + HV::diff(pc, pb);
    const int fmin = max(sb, c - reach), lmax = min(se, c + reach);
    const pos_t pf = bound_pos<F::EDGE_STEPS, false, HV>(hx.pos(fmin), pc, lo);   /* first x >= lo, not below c - (n+1) */
    const pos_t pl = bound_pos<F::EDGE_STEPS, true, HV>(pc, hx.pos(lmax), hi);    /* first x > hi, not above c + (n+1) */
    int first = fmin + HV::diff(pf, hx.pos(fmin)), last = c + HV::diff(pl, pc);
    if (last - first > C.n_window) {
      first = max(first, c - halfw);
      last = min(last, c + halfw);
    }
    if (WIDE && last < first) last = first;
    A.win[row * WIN_ROW + layer] = ((uint32_t)first << F::WB) | (uint32_t)(last - first);
    if (layer == 0) {
      /* words 12..15 of the row: what the seeding kernel needs of the seed, so that it reads one 64-byte row */
      float q3 = 0.0f;
      uint32_t flags = 0u;
      if (WIDE && C.mode == 1) {
        const float s2 = tx * tx + ty * ty;
        q3 = fminf(C.inv_p_min, sqrtf(s2 / (1.0f + s2)) * C.inv_pt_min); /* the assumed 1/p */
      } else {
        q3 = __ldg(A.sqop + seed);
        const float pmom = 1.0f / fmaxf(fabsf(q3), 1e-6f);
        flags = (pmom < C.p_same_bend) ? ROW_LOW_P : 0u;
      }
      *reinterpret_cast<uint4*>(A.win + row * WIN_ROW + NL) =
          make_uint4(__float_as_uint(x + tx * C.mag_dz_seed), __float_as_uint(tx), __float_as_uint(q3), flags);
    }
    if (DEBUG) {
      if (A.dbg.win_first) A.dbg.win_first[row * NL + layer] = (int32_t)(E.h0 + first);
      if (A.dbg.win_count) A.dbg.win_count[row * NL + layer] = last - first;
      if (A.dbg.counters) atomicAdd(A.dbg.counters + 2, (unsigned long long)(last - first));
    }
  }
}

/* ev_dup[event] = 1 iff two neighbouring hits of the event (as the kernels see them) are equal.  Only then can
 * "closest hit" meet a run of equal distances, so the seed and fit kernels skip the tie walk otherwise.
 * Conservative across segment boundaries (a false positive only costs the walk). */
template <class HV>
__device__ __forceinline__ void flag_equal_neighbours(const EventArgs& A, const EventCtx& E, const HV& hx) {
  int dup = 0;
  for (int i = threadIdx.x; i + 1 < E.nh; i += (int)blockDim.x) dup |= (hx[i] == hx[i + 1]) ? 1 : 0;
  dup = __syncthreads_or(dup);
  if (threadIdx.x == 0) A.ev_dup[E.ev] = (uint32_t)dup;
}

template <bool DEBUG, bool WIDE>
__global__ void __launch_bounds__(WIN_THREADS_BIG, 4) lf_window_kernel(const __grid_constant__ Consts C,
                                                                const __grid_constant__ EventArgs A) {
  CtaHeader& H = *reinterpret_cast<CtaHeader*>(lf_smem);
  if (threadIdx.x == 0) mbar_init(&H.mbar, 1);
  uint32_t phase = 0;
  EventCtx E;
  while (fetch_event(A, phase, E)) {
    if (threadIdx.x == 0) A.ev_state[E.ev] = 0ull; /* re-arms the look-back word of the event (lf_fit_kernel) */
    if (E.staged) {
      flag_equal_neighbours(A, E, HitView<true>(E.skew));
      windows_of_event<DEBUG, WIDE, true>(C, A, H, E, HitView<true>(E.skew));
    } else {
      flag_equal_neighbours(A, E, HitView<false>(E.gview));
      windows_of_event<DEBUG, WIDE, false>(C, A, H, E, HitView<false>(E.gview));
    }
  }
}

/* ============================================================================================
 * a3: triplet seeding.  One warp per seed.
 * ============================================================================================ */
/* Closest hit to `pred` in the non-empty x-sorted window [f, e) of at most 2^EDGE_STEPS - 1 hits, branch-free: first
 * x >= pred by a binary search whose probes beyond the window read +inf, then the two neighbours; ties -> lower index
 * (equal to a linear argmin with strict '<'; the walk over a run of equal distances runs only in events that hold two
 * equal neighbouring hits).  Returns the event-relative index and, in `dist`, |x - pred| of that hit (x - pred and
 * pred - x round to the same magnitude, so dist*dist is bit-identical to (x - pred)^2).  An empty window gives dist = +inf. */
template <bool WIDE, class HV>
__device__ __forceinline__ int closest_in_window(const HV& hx, int f, int e, float pred, bool dup, float& dist) {
  typedef typename HV::pos_t pos_t;
  const float INF = __int_as_float(0x7f800000);
  const pos_t a = hx.pos(f), end = hx.pos(e);
  pos_t p = a;
#pragma unroll
  for (int s = Fmt<WIDE>::EDGE_STEPS - 1; s >= 0; --s) {
    const pos_t q = HV::adv(p, 1 << s);
    if (q <= end && HV::before(q) < pred) p = q;
  }
  const float xl = (p > a) ? HV::before(p) : -INF;
  const float xh = (p < end) ? HV::at(p) : INF;
  const float dk = pred - xl, dh = xh - pred;
  const bool right = !(dk <= dh); /* ties -> lower index */
  pos_t k = right ? p : HV::adv(p, -1);
  dist = right ? dh : dk;
  if (dup && !right)
    while (k > a && (pred - HV::before(k)) == dk) k = HV::adv(k, -1);
  return f + HV::diff(k, a);
}

/* Per-warp scratch of the narrow seeding kernel: the passing triplets in candidate order, i.e. ascending
 * (set, h0, h2): the chi2 bit pattern (non-negative floats order like their bit patterns) and the 16-bit code. */
struct __align__(16) SeedScratch {
  uint32_t chi2[TRIP_BUF];
  uint16_t code[TRIP_BUF];
  int4 setw[2]; /* per layer set: first and end of the h1 window, first of the h2 window (event-relative) */
};
/* + the per-h0 references of the half2 pair evaluation (hit_storage = 1): x2 of the first doublet of the h0 hit's
 * bracket and, for that doublet in fp32, its slope t, its opening at the magnet and its expected x1 */
struct __align__(16) SeedScratchH2 : SeedScratch {
  float4 ref[2][32];
};

/* Rank selection on the warp's triplets: keeps the `keep` smallest of `n` (<= TRIP_BUF) by the key (chi2, position in the
 * buffer) and leaves them SORTED ascending in W.chi2 / W.code [0, min(n, keep)).  The buffer is in candidate order and a
 * selection keeps it ordered by the full key, so the position stands for the (set, h0, h2) part of the order key of
 * DESIGN.md C9.  PAPER.md:221. */
__device__ __forceinline__ int count_less4(const uint32_t* v, uint32_t c) {
  const uint4 q = *reinterpret_cast<const uint4*>(v);
  return ((q.x < c) ? 1 : 0) + ((q.y < c) ? 1 : 0) + ((q.z < c) ? 1 : 0) + ((q.w < c) ? 1 : 0);
}
__device__ __forceinline__ int select_smallest(SeedScratch& W, int n, int keep, int lane) {
  const unsigned lt_mask = (1u << lane) - 1u;
  if (n <= 32) {
    /* P = 8, 16 or 32 key slots, 32 / P lanes per key: lane & (P-1) is the key, lane / P the part of the P slots it
     * compares with (16-byte groups; the slots beyond n are padded with all-ones, which no passing chi2 equals) */
    if (lane >= n) W.chi2[lane] = 0xFFFFFFFFu;
    __syncwarp();
    const int P = (n <= 8) ? 8 : ((n <= 16) ? 16 : 32);
    const int key = lane & (P - 1);
    const uint32_t c0 = W.chi2[key];
    const uint16_t d0 = W.code[key];
    int r;
    if (n <= 8) {
      const uint2 q = *reinterpret_cast<const uint2*>(&W.chi2[(lane >> 3) * 2]);
      r = ((q.x < c0) ? 1 : 0) + ((q.y < c0) ? 1 : 0);
      r += __shfl_xor_sync(FULL, r, 8);
      r += __shfl_xor_sync(FULL, r, 16);
    } else if (n <= 16) {
      r = count_less4(&W.chi2[(lane >> 4) * 8], c0) + count_less4(&W.chi2[(lane >> 4) * 8 + 4], c0);
      r += __shfl_xor_sync(FULL, r, 16);
    } else {
      r = 0;
      for (int j = 0; j < n; j += 4) r += count_less4(&W.chi2[j], c0);
    }
    /* equal chi2: the earlier candidate first */
    r += __popc(__match_any_sync(FULL, c0) & lt_mask & (unsigned)((1ull << P) - 1ull));
    __syncwarp();
    if (lane < n && r < keep) {
      W.chi2[r] = c0;
      W.code[r] = d0;
    }
  } else {
    const uint32_t c0 = W.chi2[lane];
    const uint16_t d0 = W.code[lane];
    const uint32_t c1 = (lane + 32 < n) ? W.chi2[lane + 32] : 0xFFFFFFFFu;
    const uint16_t d1 = W.code[lane + 32];
    int r0 = 0, r1 = 0;
    for (int j = 0; j < n; ++j) {
      const uint32_t cj = W.chi2[j];
      r0 += (cj < c0 || (cj == c0 && j < lane)) ? 1 : 0;
      r1 += (cj < c1 || (cj == c1 && j < lane + 32)) ? 1 : 0;
    }
    __syncwarp();
    if (r0 < keep) {
      W.chi2[r0] = c0;
      W.code[r0] = d0;
    }
    if (lane + 32 < n && r1 < keep) {
      W.chi2[r1] = c1;
      W.code[r1] = d1;
    }
  }
  __syncwarp();
  return n < keep ? n : keep;
}

/* The same on 64-bit keys (chi2 bits, code): the wide build. */
struct __align__(16) SeedScratch64 {
  unsigned long long trip[TRIP_BUF];
};
__device__ __forceinline__ int select_smallest(SeedScratch64& W, int n, int keep, int lane) {
  const unsigned long long k0 = (lane < n) ? W.trip[lane] : ~0ull;
  const unsigned long long k1 = (lane + 32 < n) ? W.trip[lane + 32] : ~0ull;
  int r0 = 0, r1 = 0;
  if (n <= 32) {
    for (int j = 0; j < n; ++j) r0 += (W.trip[j] < k0) ? 1 : 0;
  } else {
    for (int j = 0; j < n; ++j) {
      const unsigned long long kj = W.trip[j];
      r0 += (kj < k0) ? 1 : 0;
      r1 += (kj < k1) ? 1 : 0;
    }
  }
  __syncwarp();
  if (lane < n && r0 < keep) W.trip[r0] = k0;
  if (lane + 32 < n && r1 < keep) W.trip[r1] = k1;
  __syncwarp();
  return n < keep ? n : keep;
}

/* Number of the warp's 32 lane values `xv` (ascending over the lanes, +inf padded) that are < v
 * (INCLUSIVE == false) or <= v (true): binary search by shuffles, every lane with its own v. */
template <bool INCLUSIVE>
__device__ __forceinline__ int lanes_below(float xv, float v) {
  int probe = 15; /* the lane probed next = count so far + step - 1 (one update per step instead of two) */
#pragma unroll
  for (int s = 16; s >= 2; s >>= 1) {
    const float xm = __shfl_sync(FULL, xv, probe);
    const bool c = INCLUSIVE ? (xm <= v) : (xm < v);
    probe += (c ? s : 0) - (s >> 1);
  }
#pragma unroll
  for (int r = 0; r < 2; ++r) { /* step 1, then the 32nd lane: probe == count <= 31 */
    const float xm = __shfl_sync(FULL, xv, probe);
    if (INCLUSIVE ? (xm <= v) : (xm < v)) probe += 1;
  }
  return probe;
}

/* Per layer set: the constants a candidate doublet needs (shared memory, one 32-byte row per set, so that a lane
 * whose candidate belongs to either set fetches them with two 16-byte loads instead of a select per constant). */
struct __align__(16) SetConsts {
  float inv_dz, zmag_a, zb, za;
  float K;
  /* half2 pair evaluation (seed_triplets_h2): both halves hold inv_dz, r = inv_dz * zmag_a, c = inv_dz * (zb - za * K) */
  uint32_t inv_dz2, r2, c2;
};
__device__ __forceinline__ uint32_t h2_bits(float v) {
  const __half2 h = __float2half2_rn(v);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ __half2 h2_of(uint32_t bits) { return *reinterpret_cast<const __half2*>(&bits); }
__device__ __forceinline__ void fill_set_consts(const Consts& C, SetConsts* sc) {
  if (threadIdx.x < 2) {
    const int s = threadIdx.x;
    sc[s].inv_dz = C.inv_dz_ac[s];
    sc[s].zmag_a = C.zmag_a[s];
    sc[s].zb = C.z[s ? 7 : 4];
    sc[s].za = C.z[s ? 3 : 0];
    sc[s].K = C.K[s];
    sc[s].inv_dz2 = h2_bits(C.inv_dz_ac[s]);
    sc[s].r2 = h2_bits(C.inv_dz_ac[s] * C.zmag_a[s]);
    sc[s].c2 = h2_bits(C.inv_dz_ac[s] * (C.z[s ? 7 : 4] - C.z[s ? 3 : 0] * C.K[s]));
  }
}

struct SeedEventPtrs { /* the event's slices of the per-row tables */
  const uint32_t* rows;
  uint16_t* codes;
  uint8_t* n_trip;
  uint32_t s0;
};
template <bool DEBUG, class HV>
__device__ __forceinline__ void seed_triplets(const Consts& C, const EventArgs& A, const HV& hx, uint32_t h0,
                                              const SeedEventPtrs& EP, uint32_t k_seed, SeedScratch& W, const SetConsts* SC,
                                              int lane, bool dup) {
  constexpr bool STG = std::is_same<HV, HitView<true> >::value; /* staged hits: reading past a window is harmless */
  const int* XD = reinterpret_cast<const CtaHeader*>(lf_smem)->xdelta;
  const uint32_t* rowp = EP.rows + k_seed * WIN_ROW;
  /* the seed's row of the window table: lanes 0..11 hold the packed window of layer `lane`, lanes 12..15 x_mag, tx,
   * q/p and the flags (written by the window kernel) */
  const uint32_t winw = (lane < WIN_ROW) ? rowp[lane] : 0u;
  const float x_mag = __uint_as_float(__shfl_sync(FULL, winw, 12)), tx = __uint_as_float(__shfl_sync(FULL, winw, 13));
  const float qop = __uint_as_float(__shfl_sync(FULL, winw, 14));
  const bool low_p = (__shfl_sync(FULL, winw, 15) & ROW_LOW_P) != 0u;
  const float aq = fmaxf(fabsf(qop), 1e-6f);
  const float kq = C.kick * qop; /* expected slope change across the magnet (Eq. 2) */
  const unsigned lt_mask = (1u << lane) - 1u;
  const float tol0 = C.mag_tol_base + C.mag_tol_inv_p * aq;
  const float INF = __int_as_float(0x7f800000);
  /* ---- per layer set: lanes = h0.  |x0 + t*zmag_a - x_mag| < tol is linear in x2 (t = (x2-x0)*inv_dz, slope
   * r = inv_dz*zmag_a < 0) and tol <= tol_sup (tol is monotone in |t|), so the survivors lie inside
   * x2 in [x0 + (tol_sup - A)/r, x0 + (-tol_sup - A)/r], A = x0 - x_mag.  The margin in tol_sup (0.1 mm >> fp32
   * rounding of these expressions, which may therefore use fused multiply-adds: they bracket, they do not decide)
   * makes the bracket a strict superset; the h2 window sits one hit per lane, so both bracket ends are shuffle
   * searches. */
  const float tol0m = tol0 + INTERVAL_MARGIN, tolmaxm = C.mag_tol_max + INTERVAL_MARGIN;
  float x0s[2];
  unsigned cnt_p = 0, jlo_p = 0; /* set 0 in the low half-word, set 1 in the high one */
#pragma unroll
  for (int set = 0; set < 2; ++set) {
    const int la = set ? 3 : 0;
    const uint32_t wa = __shfl_sync(FULL, winw, la), wb = __shfl_sync(FULL, winw, la + 4), wc = __shfl_sync(FULL, winw, la + 8);
    /* window starts as positions of the compact x-layer stage (fetch_event_x) */
    const int fa = (int)(wa >> 6) - XD[la], na = (int)(wa & 63u), fb = (int)(wb >> 6) - XD[la + 4], nb = (int)(wb & 63u);
    const int fc = (int)(wc >> 6) - XD[la + 8], nc = (int)(wc & 63u);
    if (lane == set) W.setw[set] = make_int4(fb, fb + nb, fc, 0);
    const bool have = (lane < na) && (nb != 0); /* no h1 hit, no triplet */
    const float x0 = (STG || lane < na) ? hx[fa + lane] : 0.0f;
    const float x2r = (STG || lane < nc) ? hx[fc + lane] : 0.0f;
    const float x2v = (lane < nc) ? x2r : INF;
    /* a survivor has |A + t*zmag_a| < tol <= tol_max, so |t| <= (|A| + tol_max)/|zmag_a| =: tmax */
    const float Aoff = x0 - x_mag;
    const float tmax = __fmaf_rn(fabsf(Aoff), C.inv_abs_zmag_a[set], C.tolmax_over_zmag[set]);
    const float tol_sup = fminf(tolmaxm, __fmaf_rn(C.mag_tol_tx, tmax, tol0m));
    const float inv_r = C.inv_r[set];
    const int jlo = lanes_below<false>(x2v, __fmaf_rn(tol_sup - Aoff, inv_r, x0));           /* first x2 >= lower end */
    const int jhi = min(nc, lanes_below<true>(x2v, __fmaf_rn(-tol_sup - Aoff, inv_r, x0)));  /* first x2 > upper end; the
                                                                                     +inf padding lanes are not hits */
    const int cnt = have ? max(jhi - jlo, 0) : 0;
    x0s[set] = x0;
    cnt_p |= (unsigned)cnt << (16 * set);
    jlo_p |= (unsigned)jlo << (16 * set);
  }
  /* ---- dense lane-per-candidate evaluation over both sets: inclusive scan of the per-h0 counts */
  unsigned incl_p = cnt_p;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned v = __shfl_up_sync(FULL, incl_p, o);
    if (lane >= o) incl_p += v;
  }
  const unsigned tot_p = __shfl_sync(FULL, incl_p, 31);
  const int total0 = (int)(tot_p & 0xFFFFu), total = total0 + (int)(tot_p >> 16);
  __syncwarp(); /* W.setw */
  int tcount = 0;
  for (int base = 0; base < total; base += 32) {
    const int tau = base + lane;
    const bool act = tau < total;
    const int set = (tau >= total0) ? 1 : 0;
    const int ts = set ? tau - total0 : tau;
    const unsigned sel = set ? 0x4432u : 0x4410u; /* __byte_perm selector: this set's half-word */
    int owner = 15; /* ends as the number of lanes whose inclusive count is <= ts == the h0 lane owning candidate ts;
                       meanwhile the lane probed next (count so far + step - 1) */
#pragma unroll
    for (int s = 16; s >= 2; s >>= 1) {
      const unsigned v = __shfl_sync(FULL, incl_p, owner);
      owner += (((int)__byte_perm(v, 0u, sel) <= ts) ? s : 0) - (s >> 1);
    }
    {
      const unsigned v = __shfl_sync(FULL, incl_p, owner);
      if ((int)__byte_perm(v, 0u, sel) <= ts) owner += 1;
    }
    const unsigned ip = __shfl_sync(FULL, incl_p, owner), cp = __shfl_sync(FULL, cnt_p, owner);
    const unsigned jp = __shfl_sync(FULL, jlo_p, owner);
    const int before = (int)__byte_perm(ip, 0u, sel) - (int)__byte_perm(cp, 0u, sel);
    const int j = (int)__byte_perm(jp, 0u, sel) + (ts - before); /* h2 index inside its window */
    const float xa = __shfl_sync(FULL, x0s[0], owner), xb = __shfl_sync(FULL, x0s[1], owner);
    const float x0o = set ? xb : xa;
    bool pass = false;
    uint32_t chi2b = 0u, code = 0u;
    if (act) {
      /* the exact predicate is the definition */
      const float4 ca = *reinterpret_cast<const float4*>(&SC[set].inv_dz); /* inv_dz, zmag_a, zb, za */
      const int4 wv = W.setw[set];                                        /* fb, fb + nb, fc */
      const float x2 = hx[wv.z + j];
      const float t = (x2 - x0o) * ca.x;
      bool ok = true;
      if (low_p) ok = (t - tx) * kq > 0.0f; /* filter 1: same bending direction as the expected kick */
      const float x_at_mag = x0o + t * ca.y;
      const float tol = fminf(C.mag_tol_max, tol0 + C.mag_tol_tx * fabsf(t));
      ok = ok && (fabsf(x_at_mag - x_mag) < tol); /* filter 2: opening at the magnet centre */
      if (DEBUG && ok && A.dbg.counters) atomicAdd(A.dbg.counters + 4, 1ull);
      if (ok) {
        /* x1_expected, closest h1, chi2 cut */
        const float x1e = ca.z * t + (x0o - t * ca.w) * SC[set].K;
        float dx;
        const int k = closest_in_window<false>(hx, wv.x, wv.y, x1e, dup, dx);
        const float chi2 = dx * dx;
        if (chi2 < C.T_triplet) {
          pass = true;
          chi2b = __float_as_uint(chi2);
          code = (unsigned)((set << 15) | (owner << 10) | (j << 5) | (k - wv.x));
        }
      }
    }
    const unsigned m = __ballot_sync(FULL, pass);
    if (DEBUG && lane == 0 && A.dbg.counters) atomicAdd(A.dbg.counters + 5, (unsigned long long)__popc(m));
    if (m) {
      if (tcount > 32) tcount = select_smallest(W, tcount, C.n_triplets, lane);
      if (pass) {
        const int slot = tcount + __popc(m & lt_mask);
        W.chi2[slot] = chi2b;
        W.code[slot] = (uint16_t)code;
      }
      tcount += __popc(m);
      __syncwarp();
    }
  }
  if (tcount > 0) tcount = select_smallest(W, tcount, C.n_triplets, lane); /* sorted in (chi2,set,h0,h2) order */
  const int ntr = tcount;
  const int NT = C.n_triplets;
  if (lane == 0) EP.n_trip[k_seed] = (uint8_t)ntr;
  const bool mine = lane < ntr;
  const unsigned low = mine ? (unsigned)W.code[lane] : 0u;
  if (lane < NT) EP.codes[k_seed * (uint32_t)NT + (uint32_t)lane] = (uint16_t)low;
  if (DEBUG) {
    if (lane == 0 && A.dbg.counters) {
      atomicAdd(A.dbg.counters + 3, (unsigned long long)total);
      atomicAdd(A.dbg.counters + 6, (unsigned long long)ntr);
    }
    const size_t seed = (size_t)EP.s0 + k_seed;
    const int set = (low >> 15) & 1, la = set ? 3 : 0;
    const int fa = (int)(__shfl_sync(FULL, winw, la) >> 6), fb = (int)(__shfl_sync(FULL, winw, la + 4) >> 6);
    const int fc = (int)(__shfl_sync(FULL, winw, la + 8) >> 6);
    if (lane == 0 && A.dbg.n_triplets) A.dbg.n_triplets[seed] = ntr;
    if (lane < NT) {
      const size_t o = (size_t)seed * NT + lane;
      if (A.dbg.trip_set) A.dbg.trip_set[o] = mine ? set : -1;
      if (A.dbg.trip_chi2) A.dbg.trip_chi2[o] = mine ? __uint_as_float(W.chi2[lane]) : -1.0f;
      if (A.dbg.trip_hits) {
        A.dbg.trip_hits[o * 3 + 0] = mine ? (int32_t)(h0 + fa + ((low >> 10) & 31)) : -1;
        A.dbg.trip_hits[o * 3 + 1] = mine ? (int32_t)(h0 + fb + (low & 31)) : -1;
        A.dbg.trip_hits[o * 3 + 2] = mine ? (int32_t)(h0 + fc + ((low >> 5) & 31)) : -1;
      }
    }
  }
  __syncwarp();
}

/* a3 with fp16 hit storage (params.hit_storage = 1; "Using fp16 allows us to use half-2 vectorized instructions
 * ... processing two combinations at a time"): the same scheme as seed_triplets, but a lane evaluates a PAIR of
 * neighbouring doublets (h0, j0) and (h0, j0 + 1) of one h0 hit with __half2 arithmetic.  To keep binary16 accurate the
 * pair works on small quantities: per h0 hit the first doublet of its bracket is evaluated in fp32 (slope t_ref, opening
 * at the magnet m_ref, expected x1 e_ref) and a doublet of the bracket differs from it by d = x2 - x2_ref < 2 * 41 mm:
 *   t = t_ref + d * inv_dz,  opening = m_ref + d * (inv_dz * zmag_a),  x1_expected = e_ref + d * inv_dz * (zb - za * K),
 * all three exact identities of PAPER.md:210-215.  The closest h1 and the chi2 are fp32 on the decoded hits.  Decisions
 * are taken in binary16 here, so this kernel is judged by BASELINE.json configs[2]'s rule, not bit for bit. */
template <bool DEBUG, class HV>
__device__ __forceinline__ void seed_triplets_h2(const Consts& C, const EventArgs& A, const HV& hx, uint32_t h0,
                                                 const SeedEventPtrs& EP, uint32_t k_seed, SeedScratchH2& W, const SetConsts* SC,
                                                 int lane, bool dup) {
  constexpr bool STG = std::is_same<HV, HitView<true> >::value;
  const int* XD = reinterpret_cast<const CtaHeader*>(lf_smem)->xdelta;
  const uint32_t* rowp = EP.rows + k_seed * WIN_ROW;
  const uint32_t winw = (lane < WIN_ROW) ? rowp[lane] : 0u;
  const float x_mag = __uint_as_float(__shfl_sync(FULL, winw, 12)), tx = __uint_as_float(__shfl_sync(FULL, winw, 13));
  const float qop = __uint_as_float(__shfl_sync(FULL, winw, 14));
  const bool low_p = (__shfl_sync(FULL, winw, 15) & ROW_LOW_P) != 0u;
  const float aq = fmaxf(fabsf(qop), 1e-6f);
  const float kq = C.kick * qop;
  const unsigned lt_mask = (1u << lane) - 1u;
  const float tol0 = C.mag_tol_base + C.mag_tol_inv_p * aq;
  const float INF = __int_as_float(0x7f800000);
  const float tol0m = tol0 + INTERVAL_MARGIN, tolmaxm = C.mag_tol_max + INTERVAL_MARGIN;
  unsigned slots_p = 0, cnt_p = 0, jlo_p = 0; /* set 0 in the low half-word, set 1 in the high one */
#pragma unroll
  for (int set = 0; set < 2; ++set) {
    const int la = set ? 3 : 0;
    const uint32_t wa = __shfl_sync(FULL, winw, la), wb = __shfl_sync(FULL, winw, la + 4), wc = __shfl_sync(FULL, winw, la + 8);
    /* window starts as positions of the compact x-layer stage (fetch_event_x) */
    const int fa = (int)(wa >> 6) - XD[la], na = (int)(wa & 63u), fb = (int)(wb >> 6) - XD[la + 4], nb = (int)(wb & 63u);
    const int fc = (int)(wc >> 6) - XD[la + 8], nc = (int)(wc & 63u);
    if (lane == set) W.setw[set] = make_int4(fb, fb + nb, fc, fc + nc);
    const bool have = (lane < na) && (nb != 0);
    const float x0 = (STG || lane < na) ? hx[fa + lane] : 0.0f;
    const float x2r = (STG || lane < nc) ? hx[fc + lane] : 0.0f;
    const float x2v = (lane < nc) ? x2r : INF;
    const float Aoff = x0 - x_mag;
    const float tmax = __fmaf_rn(fabsf(Aoff), C.inv_abs_zmag_a[set], C.tolmax_over_zmag[set]);
    const float tol_sup = fminf(tolmaxm, __fmaf_rn(C.mag_tol_tx, tmax, tol0m));
    const float inv_r = C.inv_r[set];
    const int jlo = lanes_below<false>(x2v, __fmaf_rn(tol_sup - Aoff, inv_r, x0));
    const int jhi = min(nc, lanes_below<true>(x2v, __fmaf_rn(-tol_sup - Aoff, inv_r, x0)));
    const int cnt = have ? max(jhi - jlo, 0) : 0;
    /* the bracket's first doublet in fp32: the reference of the h0 hit's pairs */
    const float x2ref = __shfl_sync(FULL, x2r, min(jlo, 31));
    const float t_ref = (x2ref - x0) * C.inv_dz_ac[set];
    const float m_ref = (x0 + t_ref * C.zmag_a[set]) - x_mag;
    const float e_ref = C.z[set ? 7 : 4] * t_ref + (x0 - t_ref * C.z[set ? 3 : 0]) * C.K[set];
    W.ref[set][lane] = make_float4(x2ref, t_ref, m_ref, e_ref);
    slots_p |= (unsigned)((cnt + 1) >> 1) << (16 * set);
    cnt_p |= (unsigned)cnt << (16 * set);
    jlo_p |= (unsigned)jlo << (16 * set);
  }
  /* ---- dense lane-per-PAIR evaluation over both sets: inclusive scan of the per-h0 pair counts */
  unsigned incl_p = slots_p;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned v = __shfl_up_sync(FULL, incl_p, o);
    if (lane >= o) incl_p += v;
  }
  const unsigned tot_p = __shfl_sync(FULL, incl_p, 31);
  const int total0 = (int)(tot_p & 0xFFFFu), total = total0 + (int)(tot_p >> 16);
  __syncwarp(); /* W.setw, W.ref */
  /* seed constants of the pair arithmetic, both halves equal */
  const __half2 tx2 = __float2half2_rn(tx), tol02 = __float2half2_rn(tol0), tolmax2 = __float2half2_rn(C.mag_tol_max);
  const __half2 txc2 = __float2half2_rn(C.mag_tol_tx), sgn2 = __float2half2_rn(kq > 0.0f ? 1.0f : (kq < 0.0f ? -1.0f : 0.0f));
  const __half2 zero2 = __float2half2_rn(0.0f);
  int tcount = 0, n_eval = 0, n_ok = 0, n_pass = 0;
  for (int base = 0; base < total; base += 32) {
    const int tau = base + lane;
    const bool act = tau < total;
    const int set = (tau >= total0) ? 1 : 0;
    const int ts = set ? tau - total0 : tau;
    const unsigned sel = set ? 0x4432u : 0x4410u;
    int owner = 15;
#pragma unroll
    for (int s = 16; s >= 2; s >>= 1) {
      const unsigned v = __shfl_sync(FULL, incl_p, owner);
      owner += (((int)__byte_perm(v, 0u, sel) <= ts) ? s : 0) - (s >> 1);
    }
    {
      const unsigned v = __shfl_sync(FULL, incl_p, owner);
      if ((int)__byte_perm(v, 0u, sel) <= ts) owner += 1;
    }
    const unsigned ip = __shfl_sync(FULL, incl_p, owner), sp = __shfl_sync(FULL, slots_p, owner);
    const unsigned jp = __shfl_sync(FULL, jlo_p, owner), cp = __shfl_sync(FULL, cnt_p, owner);
    const int before = (int)__byte_perm(ip, 0u, sel) - (int)__byte_perm(sp, 0u, sel);
    const int pair = ts - before;                                   /* pair of the h0 hit's bracket */
    const int j0 = (int)__byte_perm(jp, 0u, sel) + 2 * pair;       /* h2 index of its first doublet */
    const bool two = 2 * pair + 1 < (int)__byte_perm(cp, 0u, sel); /* the pair's second doublet exists */
    bool ok[2] = {false, false};
    float x1e[2] = {0.0f, 0.0f};
    int4 wv = make_int4(0, 0, 0, 0);
    if (act) {
      wv = W.setw[set]; /* fb, fb + nb, fc, fc + nc */
      const float4 ref = W.ref[set][owner]; /* x2_ref, t_ref, m_ref, e_ref */
      const float x2a = hx[wv.z + j0];
      const float x2b = (STG || two) ? hx[wv.z + j0 + 1] : x2a;
      /* two combinations at a time */
      const __half2 d2 = __floats2half2_rn(x2a - ref.x, x2b - ref.x);
      const __half2 t2 = __hfma2(d2, h2_of(SC[set].inv_dz2), __float2half2_rn(ref.y));
      const __half2 m2 = __hfma2(d2, h2_of(SC[set].r2), __float2half2_rn(ref.z));
      const __half2 tol2 = __hmin2(tolmax2, __hfma2(__habs2(t2), txc2, tol02));
      unsigned okm = __hlt2_mask(__habs2(m2), tol2);                                        /* filter 2 */
      if (low_p) okm &= __hgt2_mask(__hmul2(__hsub2(t2, tx2), sgn2), zero2);                 /* filter 1 */
      const __half2 e2 = __hmul2(d2, h2_of(SC[set].c2));
      x1e[0] = ref.w + __low2float(e2);
      x1e[1] = ref.w + __high2float(e2);
      ok[0] = (okm & 0xFFFFu) != 0u;
      ok[1] = two && (okm >> 16) != 0u;
    }
    if (DEBUG) {
      n_eval += __popc(__ballot_sync(FULL, act)) + __popc(__ballot_sync(FULL, act && two));
      n_ok += __popc(__ballot_sync(FULL, ok[0])) + __popc(__ballot_sync(FULL, ok[1]));
    }
#pragma unroll
    for (int e = 0; e < 2; ++e) { /* the pair's doublets in turn: closest h1 and chi2 cut in fp32 */
      bool pass = false;
      uint32_t chi2b = 0u, code = 0u;
      if (ok[e]) {
        float dx;
        const int k = closest_in_window<false>(hx, wv.x, wv.y, x1e[e], dup, dx);
        const float chi2 = dx * dx;
        if (chi2 < C.T_triplet) {
          pass = true;
          chi2b = __float_as_uint(chi2);
          code = (unsigned)((set << 15) | (owner << 10) | ((j0 + e) << 5) | (k - wv.x));
        }
      }
      const unsigned m = __ballot_sync(FULL, pass);
      if (m) {
        if (DEBUG) n_pass += __popc(m);
        if (tcount > 32) tcount = select_smallest(W, tcount, C.n_triplets, lane);
        if (pass) {
          const int slot = tcount + __popc(m & lt_mask);
          W.chi2[slot] = chi2b;
          W.code[slot] = (uint16_t)code;
        }
        tcount += __popc(m);
        __syncwarp();
      }
    }
  }
  if (tcount > 0) tcount = select_smallest(W, tcount, C.n_triplets, lane);
  const int ntr = tcount;
  const int NT = C.n_triplets;
  if (lane == 0) EP.n_trip[k_seed] = (uint8_t)ntr;
  const bool mine = lane < ntr;
  const unsigned low = mine ? (unsigned)W.code[lane] : 0u;
  if (lane < NT) EP.codes[k_seed * (uint32_t)NT + (uint32_t)lane] = (uint16_t)low;
  if (DEBUG) {
    if (lane == 0 && A.dbg.counters) {
      atomicAdd(A.dbg.counters + 3, (unsigned long long)n_eval);
      atomicAdd(A.dbg.counters + 4, (unsigned long long)n_ok);
      atomicAdd(A.dbg.counters + 5, (unsigned long long)n_pass);
      atomicAdd(A.dbg.counters + 6, (unsigned long long)ntr);
    }
    const size_t seed = (size_t)EP.s0 + k_seed;
    const int set = (low >> 15) & 1, la = set ? 3 : 0;
    const int fa = (int)(__shfl_sync(FULL, winw, la) >> 6), fb = (int)(__shfl_sync(FULL, winw, la + 4) >> 6);
    const int fc = (int)(__shfl_sync(FULL, winw, la + 8) >> 6);
    if (lane == 0 && A.dbg.n_triplets) A.dbg.n_triplets[seed] = ntr;
    if (lane < NT) {
      const size_t o = (size_t)seed * NT + lane;
      if (A.dbg.trip_set) A.dbg.trip_set[o] = mine ? set : -1;
      if (A.dbg.trip_chi2) A.dbg.trip_chi2[o] = mine ? __uint_as_float(W.chi2[lane]) : -1.0f;
      if (A.dbg.trip_hits) {
        A.dbg.trip_hits[o * 3 + 0] = mine ? (int32_t)(h0 + fa + ((low >> 10) & 31)) : -1;
        A.dbg.trip_hits[o * 3 + 1] = mine ? (int32_t)(h0 + fb + (low & 31)) : -1;
        A.dbg.trip_hits[o * 3 + 2] = mine ? (int32_t)(h0 + fc + ((low >> 5) & 31)) : -1;
      }
    }
  }
  __syncwarp();
}

/* a3 in the wide build (windows of up to 64 hits, `sides` rows per seed).  One warp per
 * row.  Same scheme as seed_triplets over four groups of 32 h0 hits (layer set x half of the h0 window): lanes =
 * h0 bracket the h2 interval that can pass the magnet-opening cut (binary searches over the h2 window in shared
 * memory) and leave (running candidate count, bracket start, x0) in the warp's scratch; then ONE dense pass maps
 * lanes to candidate doublets (binary search of the candidate number in the 128 running counts), where the exact
 * fp32 predicate decides and closest h1 / chi2 cut follow in the same lane.  In the no-UT mode the assumed 1/p
 * of PAPER.md:289 stands where q/p stood and the same-bend filter does not exist (a VELO track has no momentum
 * or charge). */
struct __align__(16) SeedScratchWide {
  unsigned long long trip[TRIP_BUF];
  uint32_t incl[128]; /* entry e = set*64 + h0: candidates of entries 0..e */
  uint32_t jx[128];   /* first h2 index of the bracket | candidates before the entry << 8 */
  float x0[128];
};
__device__ __forceinline__ SeedScratch64& trip_part(SeedScratchWide& W) { return *reinterpret_cast<SeedScratch64*>(W.trip); }

template <bool DEBUG, class HV>
__device__ __forceinline__ void seed_triplets_wide(const Consts& C, const EventArgs& A, const HV& hx, uint32_t h0,
                                                   uint32_t seed, int side, SeedScratchWide& W, int lane, bool dup) {
  typedef Fmt<true> F;
  typedef typename HV::pos_t pos_t;
  const int* XD = reinterpret_cast<const CtaHeader*>(lf_smem)->xdelta;
  const size_t row = (size_t)seed * C.sides + side;
  const bool no_ut = C.mode == 1;
  /* the row of the window table: lanes 0..11 the packed windows, lanes 12..15 x_mag, tx, q/p (no-UT: the assumed 1/p of
   * PAPER.md:289) and the flags, written by the window kernel */
  const uint32_t winw = (lane < WIN_ROW) ? A.win[row * WIN_ROW + lane] : 0u;
  const float x_mag = __uint_as_float(__shfl_sync(FULL, winw, 12)), tx = __uint_as_float(__shfl_sync(FULL, winw, 13));
  const float q3 = __uint_as_float(__shfl_sync(FULL, winw, 14));
  const bool low_p = (__shfl_sync(FULL, winw, 15) & ROW_LOW_P) != 0u;
  const float aq = no_ut ? q3 : fmaxf(fabsf(q3), 1e-6f);
  const float kq = no_ut ? 0.0f : C.kick * q3; /* expected slope change across the magnet (Eq. 2) */
  const unsigned lt_mask = (1u << lane) - 1u;
  const float tol0 = C.mag_tol_base + C.mag_tol_inv_p * aq;
  /* ---- brackets: four groups of 32 h0 hits */
  int fbs[2], nbs[2], fcs[2];
  int total = 0; /* warp-uniform running number of candidate doublets */
#pragma unroll
  for (int set = 0; set < 2; ++set) {
    const int la = set ? 3 : 0;
    const uint32_t wa = __shfl_sync(FULL, winw, la), wb = __shfl_sync(FULL, winw, la + 4), wc = __shfl_sync(FULL, winw, la + 8);
    /* window starts as positions of the compact x-layer stage (fetch_event_x) */
    const int fa = (int)(wa >> F::WB) - XD[la], na = (int)(wa & F::WMASK), nc = (int)(wc & F::WMASK);
    fbs[set] = (int)(wb >> F::WB) - XD[la + 4];
    nbs[set] = (int)(wb & F::WMASK);
    fcs[set] = (int)(wc >> F::WB) - XD[la + 8];
    const bool set_on = na != 0 && nbs[set] != 0 && nc != 0; /* warp-uniform */
    const float inv_r = C.inv_r[set];
    const pos_t pc0 = hx.pos(fcs[set]), pc1 = hx.pos(fcs[set] + nc);
#pragma unroll
    for (int sub = 0; sub < 64; sub += 32) {
      const int e = set * 64 + sub + lane;
      if (!set_on || sub >= na) { /* warp-uniform: no candidates from this group */
        W.incl[e] = (uint32_t)total;
        continue;
      }
      const bool have = sub + lane < na;
      const float x0 = have ? hx[fa + sub + lane] : 0.0f;
      /* a survivor has |A + t*zmag_a| < tol <= tol_max, so |t| <= (|A| + tol_max)/|zmag_a| =: tmax (see seed_triplets) */
      const float Aoff = x0 - x_mag;
      const float tmax = (fabsf(Aoff) + C.mag_tol_max) * C.inv_abs_zmag_a[set];
      const float tol_sup = fminf(C.mag_tol_max, tol0 + C.mag_tol_tx * tmax) + INTERVAL_MARGIN;
      const int jlo = HV::diff(bound_pos<F::EDGE_STEPS, false, HV>(pc0, pc1, x0 + (tol_sup - Aoff) * inv_r), pc0);
      const int jhi = HV::diff(bound_pos<F::EDGE_STEPS, true, HV>(pc0, pc1, x0 + (-tol_sup - Aoff) * inv_r), pc0);
      const int cnt = have ? max(jhi - jlo, 0) : 0;
      int incl = cnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += v;
      }
      incl += total;
      W.incl[e] = (uint32_t)incl;
      W.jx[e] = (uint32_t)jlo | ((uint32_t)(incl - cnt) << 8);
      W.x0[e] = x0;
      total = __shfl_sync(FULL, incl, 31);
    }
  }
  __syncwarp();
  /* ---- dense lane-per-candidate evaluation over all groups */
  int tcount = 0;
  SeedScratch64& WT = trip_part(W);
  for (int base = 0; base < total; base += 32) {
    const int tau = base + lane;
    const bool act = tau < total;
    int e = 0; /* number of entries whose running count is <= tau == the entry owning candidate tau */
#pragma unroll
    for (int st = 64; st >= 1; st >>= 1)
      if (W.incl[e + st - 1] <= (uint32_t)tau) e += st;
    e = min(e, 127);
    bool pass = false;
    unsigned long long key = 0;
    if (act) {
      const uint32_t jx = W.jx[e];
      const float x0o = W.x0[e];
      const int set = e >> 6, h0i = e & 63;
      const int j = (int)(jx & 0xFFu) + (tau - (int)(jx >> 8)); /* h2 index inside its window */
      /* the exact predicate is the definition */
      const int fb = set ? fbs[1] : fbs[0], nb = set ? nbs[1] : nbs[0], fc = set ? fcs[1] : fcs[0];
      const float inv_dz = set ? C.inv_dz_ac[1] : C.inv_dz_ac[0], zmag_a = set ? C.zmag_a[1] : C.zmag_a[0];
      const float x2 = hx[fc + j];
      const float t = (x2 - x0o) * inv_dz;
      bool ok = true;
      if (low_p) ok = (t - tx) * kq > 0.0f; /* filter 1: same bending direction as the expected kick */
      const float x_at_mag = x0o + t * zmag_a;
      const float tol = fminf(C.mag_tol_max, tol0 + C.mag_tol_tx * fabsf(t));
      ok = ok && (fabsf(x_at_mag - x_mag) < tol); /* filter 2: opening at the magnet centre */
      if (DEBUG && ok && A.dbg.counters) atomicAdd(A.dbg.counters + 4, 1ull);
      if (ok) {
        const float zb = set ? C.z[7] : C.z[4], za = set ? C.z[3] : C.z[0], Kx1 = set ? C.K[1] : C.K[0];
        const float x1e = zb * t + (x0o - t * za) * Kx1;
        float dx;
        const int k = closest_in_window<true>(hx, fb, fb + nb, x1e, dup, dx);
        const float chi2 = dx * dx;
        if (chi2 < C.T_triplet) {
          pass = true;
          key = ((unsigned long long)__float_as_uint(chi2) << 32) |
                (unsigned)((set << (3 * F::IB)) | (h0i << (2 * F::IB)) | (j << F::IB) | (k - fb));
        }
      }
    }
    const unsigned m = __ballot_sync(FULL, pass);
    if (DEBUG && lane == 0 && A.dbg.counters) atomicAdd(A.dbg.counters + 5, (unsigned long long)__popc(m));
    if (m) {
      if (tcount > 32) tcount = select_smallest(WT, tcount, C.n_triplets, lane);
      if (pass) WT.trip[tcount + __popc(m & lt_mask)] = key;
      tcount += __popc(m);
      __syncwarp();
    }
  }
  if (tcount > 0) tcount = select_smallest(WT, tcount, C.n_triplets, lane); /* sorted in (chi2,set,h0,h2) order */
  const int ntr = tcount;
  const int NT = C.n_triplets;
  if (lane == 0) A.n_trip[row] = (uint8_t)ntr;
  const bool mine = lane < ntr;
  const unsigned long long key = mine ? WT.trip[lane] : 0ull;
  if (mine) static_cast<uint32_t*>(A.trip_code)[row * NT + lane] = (unsigned)key; /* codes beyond n_trip are never read */
  if (DEBUG) {
    if (lane == 0 && A.dbg.counters) {
      atomicAdd(A.dbg.counters + 3, (unsigned long long)total);
      atomicAdd(A.dbg.counters + 6, (unsigned long long)ntr);
    }
    const unsigned low = (unsigned)key;
    const int set = (low >> (3 * F::IB)) & 1, la = set ? 3 : 0;
    const int fa = (int)(__shfl_sync(FULL, winw, la) >> F::WB);
    const int fb = (set ? fbs[1] : fbs[0]) + XD[la + 4], fc = (set ? fcs[1] : fcs[0]) + XD[la + 8]; /* event-relative again */
    if (lane == 0 && A.dbg.n_triplets) A.dbg.n_triplets[row] = ntr;
    if (lane < NT) {
      const size_t o = row * NT + lane;
      if (A.dbg.trip_set) A.dbg.trip_set[o] = mine ? set : -1;
      if (A.dbg.trip_chi2) A.dbg.trip_chi2[o] = mine ? __uint_as_float((unsigned)(key >> 32)) : -1.0f;
      if (A.dbg.trip_hits) {
        A.dbg.trip_hits[o * 3 + 0] = mine ? (int32_t)(h0 + fa + ((low >> (2 * F::IB)) & F::IMASK)) : -1;
        A.dbg.trip_hits[o * 3 + 1] = mine ? (int32_t)(h0 + fb + (low & F::IMASK)) : -1;
        A.dbg.trip_hits[o * 3 + 2] = mine ? (int32_t)(h0 + fc + ((low >> F::IB) & F::IMASK)) : -1;
      }
    }
  }
  __syncwarp();
}

template <bool WIDE, bool H2>
struct __align__(16) SeedTables {
  int next_seed;
  int pad[3];
  SetConsts sc[2];
  typename std::conditional<WIDE, SeedScratchWide, typename std::conditional<H2, SeedScratchH2, SeedScratch>::type>::type ws[SEED_WARPS];
};

/* H2: the half2 pair evaluation of seed_triplets_h2 (narrow build, hit_storage = 1) */
template <bool DEBUG, bool WIDE, bool H2 = false>
__global__ void __launch_bounds__(SEED_THREADS, WIDE ? 4 : 5) lf_seed_kernel(const __grid_constant__ Consts C,
                                                                           const __grid_constant__ EventArgs A) {
  static_assert(!(WIDE && H2), "the half2 pair evaluation exists in the narrow build only");
  CtaHeader& H = *reinterpret_cast<CtaHeader*>(lf_smem);
  SeedTables<WIDE, H2>& T = *reinterpret_cast<SeedTables<WIDE, H2>*>(lf_smem + HDR_BYTES + (size_t)A.stage_cap * sizeof(float));
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    mbar_init(&H.mbar, 1);
    T.next_seed = 0;
  }
  fill_set_consts(C, T.sc); /* published by fetch_event's barriers */
  uint32_t phase = 0;
  EventCtx E;
  while (fetch_event_x(A, phase, E)) {
    const uint32_t s0 = A.seed_off[E.ev], s1 = A.seed_off[E.ev + 1];
    const int sides = WIDE ? C.sides : 1;
    const int n_rows = (int)(s1 - s0) * sides;
    auto& W = T.ws[warp];
    const bool dup = H.dup != 0;
    constexpr int PER_TICKET = WIDE ? 2 : 4;
    SeedEventPtrs EP;
    EP.rows = A.win + (size_t)s0 * WIN_ROW;
    EP.codes = static_cast<uint16_t*>(A.trip_code) + (size_t)s0 * C.n_triplets; /* narrow build only */
    EP.n_trip = A.n_trip + s0;
    EP.s0 = s0;
    /* the warps read one 64-byte row per followed track: pull the event's rows (two per 128-byte line) into L1 now */
    for (int i = threadIdx.x * 2; i < n_rows; i += SEED_THREADS * 2)
      asm volatile("prefetch.global.L1 [%0];" ::"l"(A.win + ((size_t)s0 * sides + i) * WIN_ROW));
    /* the warps of the CTA share the event's rows by tickets: PER_TICKET rows each while many are left, single rows for
     * the last 24, so that the warps reach the end of the event together */
    const int n_big = max(n_rows - 24, 0) / PER_TICKET;
    for (;;) {
      int t = 0;
      if (lane == 0) t = atomicAdd(&T.next_seed, 1);
      t = __shfl_sync(FULL, t, 0);
      int k = (t < n_big) ? t * PER_TICKET : n_big * PER_TICKET + (t - n_big);
      if (k >= n_rows) break;
      const int kend = (t < n_big) ? k + PER_TICKET : k + 1;
      for (; k < kend; ++k) {
        if constexpr (WIDE) {
          const int sh = sides >> 1; /* sides is 1 or 2: shifts instead of a division by a run-time value */
          const uint32_t seed = s0 + (uint32_t)(k >> sh);
          const int side = k & (sides - 1);
          if (E.staged) seed_triplets_wide<DEBUG>(C, A, HitView<true>(E.skew), E.h0, seed, side, W, lane, dup);
          else seed_triplets_wide<DEBUG>(C, A, HitView<false>(E.gview), E.h0, seed, side, W, lane, dup);
        } else if constexpr (H2) {
          if (E.staged) seed_triplets_h2<DEBUG>(C, A, HitView<true>(E.skew), E.h0, EP, (uint32_t)k, W, T.sc, lane, dup);
          else seed_triplets_h2<DEBUG>(C, A, HitView<false>(E.gview), E.h0, EP, (uint32_t)k, W, T.sc, lane, dup);
        } else {
          if (E.staged) seed_triplets<DEBUG>(C, A, HitView<true>(E.skew), E.h0, EP, (uint32_t)k, W, T.sc, lane, dup);
          else seed_triplets<DEBUG>(C, A, HitView<false>(E.gview), E.h0, EP, (uint32_t)k, W, T.sc, lane, dup);
        }
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) T.next_seed = 0; /* published by fetch_event's barriers */
  }
}

/* ============================================================================================
 * a4-a6: extension (lf_extend_kernel), then fit, quality, best per seed (lf_fit_kernel).
 * ============================================================================================ */

/* Hit codes of a candidate: byte l = window-relative index of the hit on layer l, 0xFF = none. */
struct CandHits {
  uint32_t w[3];
  int n, n_uv;
  bool enough;
};
__device__ __forceinline__ unsigned code_of(const CandHits& h, int l) { return (h.w[l >> 2] >> (8 * (l & 3))) & 0xFFu; }

/* Eq. (4) parameters: exact parabola through the three triplet hits. */
template <bool WIDE, class HV>
__device__ __forceinline__ void triplet_parabola(const Consts& C, const HV& hx, const uint32_t* winw, unsigned code,
                                                 float& a0, float& t0, float& c0) {
  typedef Fmt<WIDE> F;
  const int set = (code >> (3 * F::IB)) & 1, la = set ? 3 : 0;
  const float x0 = hx[(int)(winw[la] >> F::WB) + (int)((code >> (2 * F::IB)) & F::IMASK)];
  const float x1 = hx[(int)(winw[la + 4] >> F::WB) + (int)(code & F::IMASK)];
  const float x2 = hx[(int)(winw[la + 8] >> F::WB) + (int)((code >> F::IB) & F::IMASK)];
  const float X10 = x1 - x0, X20 = x2 - x0;
  const float D10 = set ? C.D10[1] : C.D10[0], D20 = set ? C.D20[1] : C.D20[0];
  const float W10 = set ? C.W10[1] : C.W10[0];
  c0 = (X20 * D10 - X10 * D20) * (set ? C.inv_det[1] : C.inv_det[0]);
  t0 = (X10 - c0 * W10) * (set ? C.inv_D10[1] : C.inv_D10[0]);
  a0 = (x0 - t0 * (set ? C.d[3] : C.d[0])) - c0 * (set ? C.w[3] : C.w[0]);
}

/* a4/a5: extension of one triplet to the 9 other layers + hit-count rule.
 * `geo` is the shared-memory copy of the per-layer constants: d, w, dzs, tana (12 floats each). */
template <bool WIDE, class HV>
__device__ __forceinline__ CandHits extend_candidate(const Consts& C, const HV& hx, const uint32_t* winw, const float* geo,
                                                  float y, float tx, float ty, unsigned code, bool dup) {
  typedef Fmt<WIDE> F;
  const int set = (code >> (3 * F::IB)) & 1;
  float a0, t0, c0;
  triplet_parabola<WIDE>(C, hx, winw, code, a0, t0, c0);
  const float T_uv = fmaxf(C.T_uv_min, C.T_uv_slope * (fabsf(tx) + fabsf(ty)));
  CandHits h;
  /* per station: the triplet's own hit (byte 0 for set 0, byte 3 for set 1) and the three other layers,
   * searched in lockstep */
  const unsigned trip[3] = {(code >> (2 * F::IB)) & F::IMASK, code & F::IMASK, (code >> F::IB) & F::IMASK};
  const unsigned tsh = set ? 24u : 0u, sh0 = set ? 0u : 8u;
  int n = 3, n_uv = 0;
  unsigned st_mask = 0;
#pragma unroll
  for (int st = 0; st < 3; ++st) {
    const int l0 = st * 4 + (1 - set); /* layers l0, l0+1, l0+2: set 0 -> u, v, x; set 1 -> x, u, v */
    uint32_t ww[3];
    float pred[3], dist[3];
    int krel[3];
#pragma unroll
    for (int g = 0; g < 3; ++g) {
      const int l = l0 + g;
      ww[g] = winw[l];
      pred[g] = (a0 + t0 * geo[l]) + c0 * geo[NL + l];
    }
    /* stereo layers: + y(z_l) * tan(alpha_l) */
    if (set) {
      pred[1] = pred[1] + (y + ty * geo[2 * NL + l0 + 1]) * geo[3 * NL + l0 + 1];
      pred[2] = pred[2] + (y + ty * geo[2 * NL + l0 + 2]) * geo[3 * NL + l0 + 2];
    } else {
      pred[0] = pred[0] + (y + ty * geo[2 * NL + l0]) * geo[3 * NL + l0];
      pred[1] = pred[1] + (y + ty * geo[2 * NL + l0 + 1]) * geo[3 * NL + l0 + 1];
    }
    closest_group<3, WIDE>(hx, ww, pred, dup, krel, dist);
    unsigned w = (trip[st] << tsh) | (0x00FFFFFFu << sh0);
#pragma unroll
    for (int g = 0; g < 3; ++g) {
      const bool uv = set ? (g != 0) : (g != 2);
      const float chi2 = dist[g] * dist[g];
      if (chi2 < (uv ? T_uv : C.T_x)) { /* an empty window gives chi2 = +inf */
        const unsigned sh = sh0 + 8u * (unsigned)g;
        w = (w & ~(0xFFu << sh)) | ((unsigned)krel[g] << sh);
        ++n;
        if (uv) { ++n_uv; st_mask |= 1u << st; }
      }
    }
    h.w[st] = w;
  }
  h.n = n;
  h.n_uv = n_uv;
  /* at least min_hits hits and at least one u/v hit per station */
  h.enough = (n >= C.min_hits) && (st_mask == 7u);
  return h;
}

/* Per-mask constants of the two least-squares fits (computed once in lf_create, fp32, the canonical order):
 * the geometry sums depend only on which layers hold a hit. */
struct __align__(16) FitLut {
  float C00, C01, C02, C11; /* cofactors of the 3x3 normal matrix of (1, d, w) over the present layers */
  float C12, C22, inv_det, pad0;
  float U1, Ud, Udd, inv_det2; /* 2x2 normal matrix of (1, d) over the present u/v layers */
};

/* ---- E: lf_extend_kernel (a4, a5).  One thread per triplet candidate of the event; candidates passing
 * the hit-count rule are written as 16-byte records, densely and in (seed, k) order, into the event's
 * slice of `acc_rec` (slice start = first seed of the event * n_triplets). */
struct ExtTables {
  float* geo;      /* 4*12: d, w, dzs, tana */
  uint32_t* win;   /* FIT_CHUNK*12 packed windows */
  float* sp;       /* FIT_CHUNK*4: y, tx, ty, (unused) */
  uint16_t* item;  /* FIT_CHUNK*NT: seed_local<<4 | k */
  int* wcnt;       /* 2 * 8: accepted candidates per warp, double-buffered by pass */
};
__host__ __device__ inline size_t ext_tables_bytes(int nt, int chunk) {
  return 4 * NL * 4 + (size_t)chunk * NL * 4 + (size_t)chunk * 4 * 4 + (((size_t)chunk * nt * 2 + 15) & ~size_t(15)) + 16 * 4;
}

template <bool DEBUG, bool WIDE, bool STAGED>
__device__ __forceinline__ void extend_event(const Consts& C, const EventArgs& A, CtaHeader& H, const EventCtx& E,
                                             const HitView<STAGED>& hx, const ExtTables& T) {
  typedef Fmt<WIDE> F;
  typedef typename F::code_t code_t;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t s0 = A.seed_off[E.ev], s1 = A.seed_off[E.ev + 1];
  const int sides = WIDE ? C.sides : 1;
  const int nr = (int)(s1 - s0) * sides;        /* rows (followed tracks) of the event */
  const size_t row0 = (size_t)s0 * sides;       /* first row of the event */
  const int NT = C.n_triplets;
  const bool dup = H.dup != 0;
  const code_t* trip_code = static_cast<const code_t*>(A.trip_code);
  uint4* rec = A.acc_rec + row0 * NT;
  uint32_t ev_acc = 0;
  int parity = 0;
  const int CH = A.ext_chunk;
  for (int cb = 0; cb < nr; cb += CH) { /* the chunk size is even: a chunk starts on a seed boundary */
    const int cn = min(CH, nr - cb);
    const size_t rbase = row0 + (size_t)cb;
    /* ---- stage the chunk's windows, seed parameters and candidate counts */
    for (int i = tid; i < cn * WIN_ROW; i += FIT_THREADS)
      if ((i & (WIN_ROW - 1)) < NL) T.win[(i >> 4) * NL + (i & (WIN_ROW - 1))] = A.win[rbase * WIN_ROW + i];
    int my_n = 0;
    if (tid < cn) {
      const size_t row = rbase + (size_t)tid;
      const uint32_t seed = WIDE ? (uint32_t)(row >> (sides >> 1)) : (uint32_t)row; /* sides is 1 or 2 */
      T.sp[tid * 4 + 0] = __ldg(A.sy + seed);
      T.sp[tid * 4 + 1] = __ldg(A.stx + seed);
      T.sp[tid * 4 + 2] = __ldg(A.sty + seed);
      my_n = (int)A.n_trip[row];
      A.ws_nh[seed] = 0; /* set by the fit kernel if the seed gets a track */
      if (DEBUG) {
        for (int k = my_n; k < NT; ++k) {
          if (A.dbg.cand_quality) A.dbg.cand_quality[row * NT + k] = -1.0f;
          if (A.dbg.cand_hits)
            for (int l = 0; l < NL; ++l) A.dbg.cand_hits[(row * NT + k) * NL + l] = -1;
        }
      }
    }
    /* exclusive prefix of candidate counts over the chunk (FIT_CHUNK <= FIT_THREADS) */
    int incl = my_n;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int v = __shfl_up_sync(FULL, incl, o);
      if (lane >= o) incl += v;
    }
    if (lane == 31) H.warp_tot[warp] = incl;
    __syncthreads();
    int woff = 0, total = 0;
#pragma unroll
    for (int wq = 0; wq < FIT_THREADS / 32; ++wq) {
      const int tq = H.warp_tot[wq];
      woff += (wq < warp) ? tq : 0;
      total += tq;
    }
    const int excl = woff + incl - my_n;
    if (tid < cn) {
      for (int k = 0; k < my_n; ++k) T.item[excl + k] = (uint16_t)((tid << F::KB) | k);
    }
    __syncthreads();
    /* ---- one thread per candidate; the accepted ones are appended in candidate order.  The candidate's item and its
     * triplet code are fetched one pass ahead. */
    const unsigned KM = (1u << F::KB) - 1u;
    unsigned im = (tid < total) ? T.item[tid] : 0u;
    unsigned code = (tid < total) ? (unsigned)trip_code[(rbase + (size_t)(im >> F::KB)) * NT + (im & KM)] : 0u;
    for (int base = 0; base < total; base += FIT_THREADS) {
      const int it = base + tid;
      const bool more = it + FIT_THREADS < total;
      const unsigned im_next = more ? T.item[it + FIT_THREADS] : 0u;
      const unsigned code_next = more ? (unsigned)trip_code[(rbase + (size_t)(im_next >> F::KB)) * NT + (im_next & KM)] : 0u;
      bool enough = false;
      CandHits h;
      unsigned tag = 0;
      if (it < total) {
        const int rl = (int)(im >> F::KB), k = (int)(im & KM);
        const size_t row = rbase + (size_t)rl;
        h = extend_candidate<WIDE>(C, hx, T.win + rl * NL, T.geo, T.sp[rl * 4 + 0], T.sp[rl * 4 + 1], T.sp[rl * 4 + 2], code, dup);
        enough = h.enough;
        /* seed inside the event, (side,) candidate index */
        const int re = cb + rl;
        const unsigned set_bit = ((code >> (3 * F::IB)) & 1u) << F::SET_SHIFT;
        tag = WIDE ? ((unsigned)(re >> (sides >> 1)) | set_bit | ((unsigned)(re & (sides - 1)) << F::SIDE_SHIFT) | ((unsigned)k << F::K_SHIFT))
                   : ((unsigned)re | set_bit | ((unsigned)k << F::K_SHIFT));
        if (DEBUG) {
          if (A.dbg.cand_hits)
            for (int l = 0; l < NL; ++l) {
              const unsigned cd = code_of(h, l);
              A.dbg.cand_hits[(row * NT + k) * NL + l] = (cd != 0xFFu) ? (int32_t)(E.h0 + (T.win[rl * NL + l] >> F::WB) + cd) : -1;
            }
          if (A.dbg.cand_quality && !enough) A.dbg.cand_quality[row * NT + k] = -1.0f;
        }
      }
      im = im_next;
      code = code_next;
      const unsigned m = __ballot_sync(FULL, enough);
      int* wc = T.wcnt + parity * 8;
      if (lane == 0) wc[warp] = __popc(m);
      __syncthreads();
      int off = 0, tot = 0;
#pragma unroll
      for (int wq = 0; wq < FIT_THREADS / 32; ++wq) {
        const int tq = wc[wq];
        off += (wq < warp) ? tq : 0;
        tot += tq;
      }
      if (enough) rec[ev_acc + (uint32_t)(off + __popc(m & ((1u << lane) - 1u)))] = make_uint4(h.w[0], h.w[1], h.w[2], tag);
      ev_acc += (uint32_t)tot;
      parity ^= 1;
    }
    __syncthreads(); /* the tables are restaged by the next chunk */
  }
  if (tid == 0) A.ev_acc[E.ev] = ev_acc;
}

template <bool DEBUG, bool WIDE>
__global__ void __launch_bounds__(FIT_THREADS, 4) lf_extend_kernel(const __grid_constant__ Consts C,
                                                                   const __grid_constant__ EventArgs A) {
  CtaHeader& H = *reinterpret_cast<CtaHeader*>(lf_smem);
  unsigned char* tb = lf_smem + HDR_BYTES + (size_t)A.stage_cap * sizeof(float);
  const int NT = C.n_triplets;
  ExtTables T;
  T.geo = reinterpret_cast<float*>(tb);
  tb += 4 * NL * 4;
  T.win = reinterpret_cast<uint32_t*>(tb);
  tb += (size_t)A.ext_chunk * NL * 4;
  T.sp = reinterpret_cast<float*>(tb);
  tb += (size_t)A.ext_chunk * 16;
  T.item = reinterpret_cast<uint16_t*>(tb);
  tb += ((size_t)A.ext_chunk * NT * 2 + 15) & ~size_t(15);
  T.wcnt = reinterpret_cast<int*>(tb);
  if (threadIdx.x == 0) mbar_init(&H.mbar, 1);
  if (threadIdx.x < NL) {
    T.geo[threadIdx.x] = C.d[threadIdx.x];
    T.geo[NL + threadIdx.x] = C.w[threadIdx.x];
    T.geo[2 * NL + threadIdx.x] = C.dzs[threadIdx.x];
    T.geo[3 * NL + threadIdx.x] = C.tana[threadIdx.x];
  }
  uint32_t phase = 0;
  EventCtx E = {};
  /* while the event's hits are on their way: pull its per-row tables (window rows, triplet counts and codes, seed
   * parameters; written by the earlier kernels, so in DRAM by now) into L2 */
  auto prefetch_tables = [&]() {
    const int tid = threadIdx.x;
    const uint32_t s0 = A.seed_off[E.ev], s1 = A.seed_off[E.ev + 1];
    const int sides = WIDE ? C.sides : 1;
    const size_t row0 = (size_t)s0 * sides, n_rows = (size_t)(s1 - s0) * sides;
    const char* rows = reinterpret_cast<const char*>(A.win + row0 * WIN_ROW);
    for (size_t o = (size_t)tid * 128; o < n_rows * WIN_ROW * 4; o += (size_t)FIT_THREADS * 128)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(rows + o));
    const size_t cbytes = n_rows * NT * sizeof(typename Fmt<WIDE>::code_t);
    const char* codes = static_cast<const char*>(A.trip_code) + row0 * NT * sizeof(typename Fmt<WIDE>::code_t);
    for (size_t o = (size_t)tid * 128; o < cbytes; o += (size_t)FIT_THREADS * 128)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(codes + o));
    if (tid < 8) {
      if ((size_t)tid * 128 < n_rows) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.n_trip + row0 + (size_t)tid * 128));
    } else if (tid >= 32 && tid < 32 + 3 * 8) {
      const int a = (tid - 32) >> 3;
      const size_t o = (size_t)((tid - 32) & 7) * 32;
      const float* base = (a == 0) ? A.sy : ((a == 1) ? A.stx : A.sty);
      if (o < (size_t)(s1 - s0)) asm volatile("prefetch.global.L2 [%0];" ::"l"(base + s0 + o));
    }
  };
  while (fetch_event(A, phase, E, prefetch_tables)) {
    if (E.staged) extend_event<DEBUG, WIDE, true>(C, A, H, E, HitView<true>(E.skew), T);
    else extend_event<DEBUG, WIDE, false>(C, A, H, E, HitView<false>(E.gview), T);
  }
}

/* Coefficients c_0..c_4 of Eq. (9) for a seed with slopes (tx, ty): constants, or 2-D polynomials
 * in the slopes over the terms the field symmetries allow (term order: include/lf.h, lf_geometry.qop_poly2d).
 * Even i: sum_j a_ij mono_j over 10 monomials in u = tx^2, v = ty^2; odd i: tx * (sum over the first 6). */
__device__ __forceinline__ void eq9_coefficients(const Consts& C, float tx, float ty, float (&c)[5]) {
  if (C.qop_mode == 0) {
#pragma unroll
    for (int i = 0; i < 5; ++i) c[i] = C.poly[i];
    return;
  }
  const float u = tx * tx, v = ty * ty;
  const float uu = u * u, uv = u * v, vv = v * v;
  const float mono[10] = {1.0f, u, v, uu, uv, vv, uu * u, uu * v, u * vv, vv * v};
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    const int n_terms = (i % 2 == 0) ? 10 : 6;
    float acc = C.poly2d[i][0];
#pragma unroll
    for (int j = 1; j < n_terms; ++j) acc = acc + C.poly2d[i][j] * mono[j];
    c[i] = (i % 2 == 0) ? acc : tx * acc;
  }
}

/* ---- F: lf_fit_kernel (a6, a7).  One thread per accepted candidate, a pass of FIT_THREADS records at a
 * time; the records of a seed are adjacent and a pass ends on a seed boundary, so after one barrier the lowest
 * (Q, k) of every seed is known (64-bit atomicMin in shared memory) and the winning thread still holds its fit
 * in registers: it writes the 20-word track record (q/p from Eq. 9, state at z_state).  Then the CTA ranks the
 * event's tracks in seed order into the event's dense track list.
 *
 * a7 (stream compaction) without a scan or a compaction kernel: the events' track counts are scanned by a decoupled
 * look-back over `ev_state` (64-bit words: flag << 32 | value; flag 1 = the event's own count, 2 = inclusive prefix).
 * A CTA publishes its event's count when the event is done and resolves the event's prefix TWO events later, inside
 * the next-but-one fetch_event while the bulk copy of the new event's hits is in flight: the look-back then meets
 * counts that were published long ago and does not wait on a running event.  No deadlock either way: tickets are handed
 * out in event order, so every lower-numbered event is owned by a CTA that is running or done, and publishing a count
 * waits on nothing.  With the prefix known the CTA copies the event's tracks from its per-seed records (L2-resident:
 * it wrote them two events ago) to their final dense position, in (event, seed) order; the last CTA out re-arms the
 * event tickets. */
struct TrackOut {
  int32_t *hit_idx, *seed_idx, *n_hits;
  float *state, *quality;
  uint32_t *event_offsets, *n_tracks;
  unsigned long long* ev_state; /* n_events look-back words, zeroed by the window kernel of the same lf_run */
  uint32_t* tickets;            /* N_TICKETS event tickets + the count of CTAs of this kernel that are done */
};
/* CTA-wide scalars that live across events (kept out of registers) */
enum { TM_EXCL = 0,                                 /* exclusive prefix of the event being resolved */
       TM_OLD_EV, TM_OLD_S0, TM_OLD_N, TM_OLD_SLOT, /* the event finished two events ago (ev + 1; 0 = none): resolved in
                                                       the next fetch_event */
       TM_NEW_EV, TM_NEW_S0, TM_NEW_N, TM_NEW_SLOT, /* the event finished last */
       TM_SLOT,                                     /* track-list slot of the current event (0..2) */
       TM_WORDS = 12 };
constexpr int LIST_CAP = 384; /* tracks of an event whose list is also kept in shared memory until the event is copied out */
struct FitTables {
  unsigned long long* best; /* 2 * FIT_THREADS: lowest (Q bits << 32 | k) per seed of the pass, double-buffered */
  int* next_b;              /* 2: first left-over record of a pass (consumed one barrier later) */
  int* wcnt;                /* 2 * 8: seed changes per warp */
  uint32_t* misc;           /* TM_WORDS */
  uint32_t* list;           /* 3 * LIST_CAP: the track lists (seeds) of the current event and of the two still to be copied out */
};
constexpr size_t FIT_TABLES_BYTES = 2 * FIT_THREADS * 8 + 16 + 16 * 4 + TM_WORDS * 4 + 3 * LIST_CAP * 4;

__device__ __forceinline__ unsigned long long ld_state(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_state(unsigned long long* p, unsigned long long v) {
  asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

/* Decoupled look-back by one warp: exclusive prefix of event `ev` over ev_state; publishes the inclusive prefix. */
__device__ __forceinline__ uint32_t lookback_publish(unsigned long long* state, int ev, uint32_t n, int lane) {
  uint32_t excl = 0;
  for (int idx = ev - 1; idx >= 0; idx -= 32) {
    const int j = idx - lane;
    unsigned long long v;
    do { /* every lower-numbered event belongs to a CTA that is running or done: its count arrives */
      v = (j >= 0) ? ld_state(state + j) : (2ull << 32);
    } while (__any_sync(FULL, (uint32_t)(v >> 32) == 0u));
    const unsigned pm = __ballot_sync(FULL, (uint32_t)(v >> 32) == 2u);
    const int first = pm ? (__ffs(pm) - 1) : 31; /* the nearest event whose inclusive prefix is known */
    uint32_t c = (lane <= first) ? (uint32_t)v : 0u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(FULL, c, o);
    excl += c;
    if (pm) break;
  }
  if (lane == 0) st_state(state + ev, (2ull << 32) | (unsigned long long)(excl + n));
  return excl;
}

/* a7, second half: the tracks of a resolved event go from the per-seed records to their dense final position.  One
 * thread per track: its five 16-byte loads are in flight together (one L2 round trip per event instead of one per load);
 * `list` is the event's track list in shared memory, or nullptr if it did not fit (then the global copy is read). */
__device__ __forceinline__ void copy_out_event(const EventArgs& A, const TrackOut& O, const uint32_t* list, uint32_t s0, int n,
                                               uint32_t excl) {
  for (int t = threadIdx.x; t < n; t += FIT_THREADS) {
    const uint32_t seed = list ? list[t] : (uint32_t)__ldcg(A.ws_rank + s0 + t);
    const int4* src = reinterpret_cast<const int4*>(A.ws_rec) + (size_t)seed * (REC_WORDS / 4);
    const int4 h0 = __ldcg(src), h1 = __ldcg(src + 1), h2 = __ldcg(src + 2), p0 = __ldcg(src + 3), p1 = __ldcg(src + 4);
    const size_t dst = (size_t)excl + (size_t)t;
    int4* hd = reinterpret_cast<int4*>(O.hit_idx) + dst * 3;
    hd[0] = h0;
    hd[1] = h1;
    hd[2] = h2;
    O.seed_idx[dst] = p0.x;
    O.n_hits[dst] = p0.y;
    float* sd = O.state + dst * 5;
    sd[0] = __int_as_float(p0.z);
    sd[1] = __int_as_float(p0.w);
    sd[2] = __int_as_float(p1.x);
    sd[3] = __int_as_float(p1.y);
    sd[4] = __int_as_float(p1.z);
    O.quality[dst] = __int_as_float(p1.w);
  }
}

template <bool DEBUG, bool WIDE, bool STAGED>
__device__ __forceinline__ int fit_event(const Consts& C, const EventArgs& A, CtaHeader& H, const EventCtx& E,
                                         const HitView<STAGED>& hx, const FitTables& T) {
  typedef Fmt<WIDE> F;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t s0 = A.seed_off[E.ev], s1 = A.seed_off[E.ev + 1];
  const int ns = (int)(s1 - s0);
  const int sides = WIDE ? C.sides : 1;
  const int NT = C.n_triplets;
  const uint4* rec = A.acc_rec + (size_t)s0 * sides * NT;
  const int n_acc = (int)A.ev_acc[E.ev];
  const unsigned SIE = F::SIE;
  int parity = 0;
  for (int b = 0; b < n_acc; parity ^= 1) {
    unsigned long long* best = T.best + parity * FIT_THREADS;
    int* wc = T.wcnt + parity * 8;
    best[tid] = ~0ull;
    const int t = b + tid;
    const bool have = t < n_acc;
    const uint4 r = have ? __ldg(rec + t) : make_uint4(0, 0, 0, 0xFFFFFFFFu);
    if (t + FIT_THREADS < n_acc) /* the next pass starts at most FIT_THREADS records further: pull its lines into L1 */
      asm volatile("prefetch.global.L1 [%0];" ::"l"(rec + t + FIT_THREADS));
    const unsigned sie = r.w & SIE;
    const int k = (int)(r.w >> F::K_SHIFT);
    /* wide: the records of a seed's sides are adjacent (side 0 first) and compete for the seed's track */
    const int side = WIDE ? (int)((r.w >> F::SIDE_SHIFT) & 1u) : 0;
    unsigned prev_sie = __shfl_up_sync(FULL, sie, 1);
    if (lane == 0) prev_sie = (tid > 0 && have) ? (__ldg(&rec[t - 1].w) & SIE) : 0xFFFFFFFEu;
    /* a seed whose records continue in the next pass is left to that pass (a seed has < FIT_THREADS records) */
    const unsigned nxt_sie = (b + FIT_THREADS < n_acc) ? (__ldg(&rec[b + FIT_THREADS].w) & SIE) : 0xFFFFFFFEu;
    const bool mine = have && sie != nxt_sie;
    if (have && !mine && prev_sie != nxt_sie) T.next_b[parity] = t; /* first left-over record: single writer */
    const uint32_t seed = s0 + sie;
    /* dense index of the record's seed inside the pass: number of seed changes up to this record */
    const unsigned chg = __ballot_sync(FULL, have && sie != prev_sie);
    if (lane == 0) wc[warp] = __popc(chg);
    __syncthreads();
    if (tid == 0) T.next_b[parity ^ 1] = 0x7FFFFFFF; /* re-armed for the next pass; its readers are past the barrier */
    if (nxt_sie != 0xFFFFFFFEu && tid < 96) {
      /* the next pass fits seeds nxt_sie, nxt_sie + 1, ...: pull their window rows (two per 128-byte line) and seed
       * parameters towards L1 while this pass computes */
      const uint32_t ps = s0 + nxt_sie;
      const void* pf;
      if (tid < 64) pf = A.win + ((size_t)ps * sides + 2 * tid) * WIN_ROW;
      else pf = ((tid < 72) ? A.sy : ((tid < 80) ? A.stx : A.sty)) + ps + 32 * (tid & 7);
      const bool inside = (tid < 64) ? (ps * sides + 2 * tid < s1 * sides) : (ps + 32 * (tid & 7) < s1);
      if (inside) asm volatile("prefetch.global.L1 [%0];" ::"l"(pf));
    }
    int slot = __popc(chg & ((2u << lane) - 1u)) - 1;
#pragma unroll
    for (int wq = 0; wq < FIT_THREADS / 32; ++wq) slot += (wq < warp) ? wc[wq] : 0;
    /* ---- the fit, sums in ascending layer order */
    float a0 = 0.f, t0 = 0.f, c0 = 0.f, da = 0.f, dt = 0.f, dc = 0.f, dy0 = 0.f, dtym = 0.f, Q = 0.f, y = 0.f, tx = 0.f, ty = 0.f;
    unsigned mask = 0;
    CandHits h;
    h.w[0] = r.x; h.w[1] = r.y; h.w[2] = r.z;
    unsigned long long key = ~0ull;
    if (mine) {
      const size_t row = (size_t)seed * sides + side;
      const uint4* wp = reinterpret_cast<const uint4*>(A.win + row * WIN_ROW);
      const uint4 w0 = __ldg(wp), w1 = __ldg(wp + 1), w2 = __ldg(wp + 2);
      uint32_t wf[NL]; /* event-relative hit index per layer (meaningless if the layer has no hit); dead after the first loop */
      wf[0] = w0.x; wf[1] = w0.y; wf[2] = w0.z; wf[3] = w0.w; wf[4] = w1.x; wf[5] = w1.y; wf[6] = w1.z; wf[7] = w1.w;
      wf[8] = w2.x; wf[9] = w2.y; wf[10] = w2.z; wf[11] = w2.w;
      y = __ldg(A.sy + seed);
      tx = __ldg(A.stx + seed);
      ty = __ldg(A.sty + seed);
#pragma unroll
      for (int l = 0; l < NL; ++l) {
        const unsigned cd = code_of(h, l);
        wf[l] = (wf[l] >> F::WB) + cd;
        mask |= (cd != 0xFFu) ? (1u << l) : 0u;
      }
      const int n = __popc(mask), n_uv = __popc(mask & 0x666u);
      {
        const int set = (int)((r.w >> F::SET_SHIFT) & 1u);
        const float x0 = hx[(int)(set ? wf[3] : wf[0])], x1 = hx[(int)(set ? wf[7] : wf[4])], x2 = hx[(int)(set ? wf[11] : wf[8])];
        const float X10 = x1 - x0, X20 = x2 - x0;
        const float D10 = set ? C.D10[1] : C.D10[0], D20 = set ? C.D20[1] : C.D20[0];
        const float W10 = set ? C.W10[1] : C.W10[0];
        c0 = (X20 * D10 - X10 * D20) * (set ? C.inv_det[1] : C.inv_det[0]);
        t0 = (X10 - c0 * W10) * (set ? C.inv_D10[1] : C.inv_D10[0]);
        a0 = (x0 - t0 * (set ? C.d[3] : C.d[0])) - c0 * (set ? C.w[3] : C.w[0]);
      }
      const float4* lut = reinterpret_cast<const float4*>(A.fit_lut + mask);
      const float4 LA = __ldg(lut), LB = __ldg(lut + 1), LY = __ldg(lut + 2);
      const float T_uv = fmaxf(C.T_uv_min, C.T_uv_slope * (fabsf(tx) + fabsf(ty)));
      const float inv_Tuv = 1.0f / T_uv;
      /* x fit on the residuals to the triplet parabola */
      float rr[NL];
      float Sr = 0.f, Sdr = 0.f, Swr = 0.f;
#pragma unroll
      for (int l = 0; l < NL; ++l) {
        const bool present = (mask >> l) & 1u;
        const float dl = C.d[l], wl = C.w[l];
        const float s_i = hx[present ? (int)wf[l] : 0];
        const float yt = is_uv(l) ? (y + ty * C.dzs[l]) * C.tana[l] : 0.0f;
        const float mm = s_i - yt;
        rr[l] = mm - ((a0 + t0 * dl) + c0 * wl);
        if (present) {
          Sr = Sr + rr[l];
          Sdr = Sdr + dl * rr[l];
          Swr = Swr + wl * rr[l];
        }
      }
      da = ((LA.x * Sr + LA.y * Sdr) + LA.z * Swr) * LB.z;
      dt = ((LA.y * Sr + LA.w * Sdr) + LB.x * Swr) * LB.z;
      dc = ((LA.z * Sr + LB.x * Sdr) + LB.y * Swr) * LB.z;
      float Qx = 0.f, Ur = 0.f, Udr = 0.f;
#pragma unroll
      for (int l = 0; l < NL; ++l) {
        const bool present = (mask >> l) & 1u;
        const float dl = C.d[l], wl = C.w[l];
        const float e = rr[l] - ((da + dt * dl) + dc * wl);
        const float chi2 = e * e;
        if (is_uv(l)) {
          rr[l] = e * C.inv_tan[l]; /* rho: y residual to the seed's straight line */
          if (present) {
            Qx = Qx + chi2 * inv_Tuv;
            Ur = Ur + rr[l];
            Udr = Udr + dl * rr[l];
          }
        } else if (present) {
          Qx = Qx + chi2 * C.inv_Tx;
        }
      }
      /* y line on the u/v hits */
      dy0 = (LY.z * Ur - LY.y * Udr) * LY.w;
      dtym = (LY.x * Udr - LY.y * Ur) * LY.w;
      const bool ty_ok = fabsf(dtym * 0.001f) < C.T_ty;
      float Qy = 0.f;
#pragma unroll
      for (int l = 0; l < NL; ++l) {
        if (!is_uv(l)) continue;
        const float ey = rr[l] - (dy0 + dtym * C.d[l]);
        if ((mask >> l) & 1u) Qy = Qy + (ey * ey) * C.inv_Ty;
      }
      const int ci = min(3, max(0, n - 9));
      const float Cn = (ci == 0) ? C.C_nhits[0] : (ci == 1 ? C.C_nhits[1] : (ci == 2 ? C.C_nhits[2] : C.C_nhits[3]));
      Q = (Qx / (float)(n - 3) + Qy / (float)(n_uv - 2)) * Cn; /* Eq. (6) */
      if (DEBUG && A.dbg.cand_quality) A.dbg.cand_quality[row * NT + k] = ty_ok ? Q : -2.0f;
      /* accepted if Q < T_Q (and the t_y cut holds); lowest Q wins, ties -> lower (side, k) */
      if (ty_ok && (Q < C.T_Q)) {
        key = ((unsigned long long)__float_as_uint(Q) << 32) | (unsigned)((side << F::KB) | k);
        atomicMin(best + slot, key);
      }
    }
    __syncthreads();
    if (key != ~0ull && best[slot] == key) {
      /* the seed's track: its global hit indices (-1 = none; the window row is read again here, by the winner only, rather
       * than kept in 12 registers across the fit), q/p (Eq. 9) and the state at z_state */
      const uint4* wp = reinterpret_cast<const uint4*>(A.win + ((size_t)seed * sides + side) * WIN_ROW);
      const uint4 w0 = __ldg(wp), w1 = __ldg(wp + 1), w2 = __ldg(wp + 2);
      uint32_t wf[NL] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w, w2.x, w2.y, w2.z, w2.w};
#pragma unroll
      for (int l = 0; l < NL; ++l) wf[l] = ((mask >> l) & 1u) ? (E.h0 + (wf[l] >> F::WB) + code_of(h, l)) : 0xFFFFFFFFu;
      const int n = __popc(mask);
      const float a = a0 + da, tt = t0 + dt, c = c0 + dc;
      const float t_ref = tt * 0.001f;
      const float dslope = t_ref - tx;
      float cq[5];
      eq9_coefficients(C, tx, ty, cq);
      const float F = cq[0] + dslope * (cq[1] + dslope * (cq[2] + dslope * (cq[3] + dslope * cq[4])));
      int4* r4 = reinterpret_cast<int4*>(A.ws_rec + (size_t)seed * REC_WORDS);
      r4[0] = make_int4((int)wf[0], (int)wf[1], (int)wf[2], (int)wf[3]);
      r4[1] = make_int4((int)wf[4], (int)wf[5], (int)wf[6], (int)wf[7]);
      r4[2] = make_int4((int)wf[8], (int)wf[9], (int)wf[10], (int)wf[11]);
      r4[3] = make_int4((int32_t)seed, n, __float_as_int((a + tt * C.ds) + c * C.ws),
                        __float_as_int((y + ty * C.dz_state) + (dy0 + dtym * C.ds)));
      r4[4] = make_int4(__float_as_int((tt + c * C.dws) * 0.001f), __float_as_int(ty + dtym * 0.001f),
                        __float_as_int(dslope / F), __float_as_int(Q));
      A.ws_nh[seed] = 1;
    }
    b = min(T.next_b[parity], b + FIT_THREADS); /* next pass: the first record left over, else the next FIT_THREADS */
  }
  __syncthreads(); /* the track flags of this CTA's seeds are visible to all its threads */
  if (tid == 0) T.next_b[0] = T.next_b[1] = 0x7FFFFFFF;
  /* ---- the event's track list: its seeds that have a track, in seed order (a7, first half) */
  int ev_tracks = 0;
  for (int cb = 0; cb < ns; cb += FIT_THREADS) {
    const bool in = cb + tid < ns;
    const uint32_t seed = s0 + (uint32_t)(cb + tid);
    const bool found = in && A.ws_nh[seed] != 0;
    const unsigned m = __ballot_sync(FULL, found);
    if (lane == 0) H.warp_tot[warp] = __popc(m);
    __syncthreads();
    int off = 0, tot = 0;
#pragma unroll
    for (int wq = 0; wq < FIT_THREADS / 32; ++wq) {
      const int tq = H.warp_tot[wq];
      off += (wq < warp) ? tq : 0;
      tot += tq;
    }
    if (found) {
      const int pos = ev_tracks + off + __popc(m & ((1u << lane) - 1u));
      A.ws_rank[s0 + (uint32_t)pos] = (int32_t)seed;
      if (pos < LIST_CAP) T.list[T.misc[TM_SLOT] * LIST_CAP + pos] = seed;
    }
    ev_tracks += tot;
    __syncthreads();
  }
  if (tid == 0) A.ev_count[E.ev] = (uint32_t)ev_tracks;
  return ev_tracks;
}

template <bool DEBUG, bool WIDE>
__global__ void __launch_bounds__(FIT_THREADS, 4) lf_fit_kernel(const __grid_constant__ Consts C,
                                                                const __grid_constant__ EventArgs A,
                                                                const __grid_constant__ TrackOut O) {
  CtaHeader& H = *reinterpret_cast<CtaHeader*>(lf_smem);
  unsigned char* tb = lf_smem + HDR_BYTES + (size_t)A.stage_cap * sizeof(float);
  FitTables T;
  T.best = reinterpret_cast<unsigned long long*>(tb);
  T.next_b = reinterpret_cast<int*>(tb + 2 * FIT_THREADS * 8);
  T.wcnt = T.next_b + 4;
  T.misc = reinterpret_cast<uint32_t*>(T.wcnt + 16);
  T.list = T.misc + TM_WORDS;
  const int tid = threadIdx.x;
  if (tid == 0) {
    mbar_init(&H.mbar, 1);
    T.next_b[0] = T.next_b[1] = 0x7FFFFFFF;
  }
  if (tid < TM_WORDS) T.misc[tid] = 0u; /* published by fetch_event's barriers */
  /* Resolves the event in the TM_OLD_* words: look-back by warp 1, which neither issues nor polls the bulk copy.  Called
   * inside fetch_event (the words it reads were written before fetch_event's first barrier). */
  EventCtx E = {};
  auto resolve = [&](bool taken = true) {
    if (taken && threadIdx.x >= 64) {
      /* the other warps, while the event's hits are on their way: its records, window rows and seed parameters -> L2 */
      const int t = threadIdx.x - 64, nthr = FIT_THREADS - 64;
      const uint32_t s0 = A.seed_off[E.ev], s1 = A.seed_off[E.ev + 1];
      const int sides = WIDE ? C.sides : 1;
      const size_t row0 = (size_t)s0 * sides, n_rows = (size_t)(s1 - s0) * sides;
      const char* recs = reinterpret_cast<const char*>(A.acc_rec + row0 * C.n_triplets);
      const size_t rbytes = (size_t)A.ev_acc[E.ev] * sizeof(uint4);
      for (size_t o = (size_t)t * 128; o < rbytes; o += (size_t)nthr * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(recs + o));
      const char* rows = reinterpret_cast<const char*>(A.win + row0 * WIN_ROW);
      for (size_t o = (size_t)t * 128; o < n_rows * WIN_ROW * 4; o += (size_t)nthr * 128)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(rows + o));
      if (t < 4 * 8) {
        const int a = t >> 3;
        const size_t o = (size_t)(t & 7) * 32;
        const void* base = (a == 0) ? (const void*)(A.sy + s0 + o) : ((a == 1) ? (const void*)(A.stx + s0 + o)
                           : ((a == 2) ? (const void*)(A.sty + s0 + o) : (const void*)(A.ws_nh + s0 + o)));
        if (o < (size_t)(s1 - s0)) asm volatile("prefetch.global.L2 [%0];" ::"l"(base));
      }
    }
    if ((threadIdx.x >> 5) == 1 && T.misc[TM_OLD_EV] != 0u) {
      const int ev = (int)T.misc[TM_OLD_EV] - 1;
      const uint32_t n = T.misc[TM_OLD_N];
      const uint32_t excl = lookback_publish(O.ev_state, ev, n, threadIdx.x & 31);
      if ((threadIdx.x & 31) == 0) {
        T.misc[TM_EXCL] = excl;
        O.event_offsets[ev] = excl;
        if (ev == (int)A.n_events - 1) {
          O.event_offsets[ev + 1] = excl + n;
          *O.n_tracks = excl + n;
        }
      }
    }
  };
  /* after the barrier that follows resolve(): copies the resolved event out and shifts the queue of finished events */
  auto retire = [&]() {
    if (T.misc[TM_OLD_EV] != 0u) {
      const int n = (int)T.misc[TM_OLD_N];
      copy_out_event(A, O, n <= LIST_CAP ? T.list + T.misc[TM_OLD_SLOT] * LIST_CAP : nullptr, T.misc[TM_OLD_S0], n, T.misc[TM_EXCL]);
    }
    __syncthreads();
    if (threadIdx.x < 4) {
      T.misc[TM_OLD_EV + threadIdx.x] = T.misc[TM_NEW_EV + threadIdx.x];
      T.misc[TM_NEW_EV + threadIdx.x] = 0u;
    }
  };
  uint32_t phase = 0;
  while (fetch_event(A, phase, E, resolve)) {
    retire();
    int n;
    if (E.staged) n = fit_event<DEBUG, WIDE, true>(C, A, H, E, HitView<true>(E.skew), T);
    else n = fit_event<DEBUG, WIDE, false>(C, A, H, E, HitView<false>(E.gview), T);
    if (tid == 0) { /* the event is done: publish its count; fetch_event's first barrier publishes the TM_NEW_* words */
      st_state(O.ev_state + E.ev, (1ull << 32) | (unsigned long long)(uint32_t)n);
      T.misc[TM_NEW_EV] = E.ev + 1u;
      T.misc[TM_NEW_S0] = A.seed_off[E.ev];
      T.misc[TM_NEW_N] = (uint32_t)n;
      const uint32_t slot = T.misc[TM_SLOT];
      T.misc[TM_NEW_SLOT] = slot;
      T.misc[TM_SLOT] = (slot == 2u) ? 0u : slot + 1u; /* three lists in turn: the current event's and the two pending ones' */
    }
  }
  /* the batch is exhausted: resolve what this CTA still holds, in event order */
#pragma unroll 1
  for (int r = 0; r < 2; ++r) {
    resolve(false);
    __syncthreads();
    retire();
    __syncthreads();
  }
  /* the last CTA out re-arms the tickets of all event kernels for the next lf_run */
  if (tid == 0) {
    __threadfence();
    if (atomicAdd(O.tickets + N_TICKETS, 1u) == gridDim.x - 1u) {
#pragma unroll
      for (int i = 0; i <= N_TICKETS; ++i) O.tickets[i] = 0u;
    }
  }
}

/* hit_storage = 1 (BASELINE.json configs[2]; "store hit data in fp16 in addition to fp32"):
 * writes the fp16 copy of the hits.  Block-offset encoding: inside every (event, layer, zone) segment,
 * consecutive hits form blocks of 2^H16_SHIFT = 8; a block's origin is the fp32 coordinate of its 5th hit (or its
 * last one if shorter); each hit stores half(x - origin), so |offset| stays within half a block's x span.  The origin
 * slot of block b of global segment g starting at hit S is (S >> H16_SHIFT) + g + b: slots of different segments never
 * overlap, so the index alone locates the origin. */
__global__ void __launch_bounds__(256) lf_pack_hits_kernel(const float* __restrict__ hx, const uint32_t* __restrict__ seg_off,
                                                           uint32_t n_events, uint32_t event_base,
                                                           __half* __restrict__ hx16, float* __restrict__ origin16) {
  for (uint32_t ev = blockIdx.x; ev < n_events; ev += gridDim.x) {
    const uint32_t* so = seg_off + (size_t)ev * NSEG;
    for (int sg = 0; sg < NSEG; ++sg) {
      const uint32_t S = so[sg];
      const int len = (int)(so[sg + 1] - S);
      const uint32_t slot0 = (S >> H16_SHIFT) + ((event_base + ev) * NSEG + (uint32_t)sg);
      constexpr int BL = 1 << H16_SHIFT;
      for (int i = threadIdx.x; i < len; i += blockDim.x) {
        const int b0 = i & ~(BL - 1);
        const float o = hx[S + b0 + min(BL / 2, len - b0 - 1)];
        hx16[S + i] = __float2half_rn(hx[S + i] - o);
        if ((i & (BL - 1)) == 0) origin16[slot0 + (uint32_t)(i >> H16_SHIFT)] = o;
      }
    }
  }
}

/* lf_validate_inputs: the preconditions lf_run does not check (include/lf.h "Conventions").  One warp per
 * (event, layer, zone) segment, grid-stride; result[0] = OR of the violation bits, result[1..3] = smallest index of
 * a violation of each kind (segment / hit / event-or-seed), preset to 0xFFFFFFFF by the caller. */
constexpr uint32_t BAD_SEG_OFFSETS = 1u, BAD_HIT_ORDER = 2u, BAD_SEED_OFFSETS = 4u, BAD_SEED_VALUE = 8u, BAD_HIT_VALUE = 16u;
__global__ void __launch_bounds__(256) lf_validate_kernel(const float* __restrict__ hx, const __half* __restrict__ hx16,
                                                          const float* __restrict__ origin16, const uint32_t* __restrict__ seg_off,
                                                          uint32_t n_events, uint32_t n_hits, const uint32_t* __restrict__ seed_off,
                                                          uint32_t n_seeds, const float* __restrict__ sx, const float* __restrict__ sy,
                                                          const float* __restrict__ stx, const float* __restrict__ sty,
                                                          const float* __restrict__ sqop, uint32_t* __restrict__ result) {
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
  const uint32_t n_seg = n_events * NSEG;
  for (uint32_t sg = warp; sg < n_seg; sg += n_warps) {
    const uint32_t a = seg_off[sg], e = seg_off[sg + 1];
    if (a > e || e > n_hits) {
      if (lane == 0) { atomicOr(result, BAD_SEG_OFFSETS); atomicMin(result + 1, sg); }
      continue;
    }
    if (hx != nullptr) {
      for (uint32_t i = a + lane; i < e; i += 32u) {
        const float v = hx[i];
        if (!isfinite(v)) { atomicOr(result, BAD_HIT_VALUE); atomicMin(result + 2, i); }
        if (i + 1 < e && !(v <= hx[i + 1])) { atomicOr(result, BAD_HIT_ORDER); atomicMin(result + 2, i); }
      }
    } else {
      /* fp16-only input (lf_hits.x == NULL): the hits as the kernels decode them, origin of the block of 8 + half offset.
       * Rounding is monotone under one origin, so ascending fp32 hits stay ascending inside a block; neighbouring blocks
       * have different origins and may overlap by a rounding error, which the lossy mode accepts: the order is checked
       * inside blocks only. */
      const uint32_t slot0 = (a >> H16_SHIFT) + sg;
      for (uint32_t i = a + lane; i < e; i += 32u) {
        const uint32_t k = i - a;
        const float v = origin16[slot0 + (k >> H16_SHIFT)] + __half2float(hx16[i]);
        if (!isfinite(v)) { atomicOr(result, BAD_HIT_VALUE); atomicMin(result + 2, i); }
        if (i + 1 < e && ((k + 1u) >> H16_SHIFT) == (k >> H16_SHIFT) && !(__half2float(hx16[i]) <= __half2float(hx16[i + 1]))) {
          atomicOr(result, BAD_HIT_ORDER);
          atomicMin(result + 2, i);
        }
      }
    }
  }
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, n_thr = gridDim.x * blockDim.x;
  if (tid == 0 && (seg_off[0] != 0u || seg_off[n_seg] != n_hits)) { atomicOr(result, BAD_SEG_OFFSETS); atomicMin(result + 1, n_seg); }
  if (tid == 0 && (seed_off[0] != 0u || seed_off[n_events] != n_seeds)) { atomicOr(result, BAD_SEED_OFFSETS); atomicMin(result + 3, n_events); }
  for (uint32_t ev = tid; ev < n_events; ev += n_thr)
    if (seed_off[ev] > seed_off[ev + 1]) { atomicOr(result, BAD_SEED_OFFSETS); atomicMin(result + 3, ev); }
  for (uint32_t s = tid; s < n_seeds; s += n_thr) {
    bool ok = isfinite(sx[s]) && isfinite(sy[s]) && isfinite(stx[s]) && isfinite(sty[s]);
    if (sqop != nullptr) ok = ok && isfinite(sqop[s]);
    if (!ok) { atomicOr(result, BAD_SEED_VALUE); atomicMin(result + 3, s); }
  }
}

} // namespace lf
