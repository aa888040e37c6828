/*
 * lf.h -- C ABI of the B200-native Looking Forward hot path (arxiv 2402.14670, section VI).
 *
 * One library, three calls on the hot path: lf_create / lf_run / lf_destroy (BASELINE.json
 * north_star (a)).  For every upstream (VELO-UT) seed of every event in a
 * batch the library follows the track through the magnet into the 12 SciFi layers:
 *
 *   a1 extrapolation with the pT-kick
 *   a2 search windows per layer and zone          PAPER.md:165, 181-204 (Eq. 3, n_window cap)
 *   a3 x-layer triplet seeding
 *   a4 extension to the other three x layers      PAPER.md:227-232 (Eq. 4)
 *   a5 u/v stereo matching + hit-count rule
 *   a6 fit, quality factor Q, best per seed, q/p  PAPER.md:238-279 (Eq. 5, 6), 327-338 (Eq. 9)
 *   a7 stream compaction into dense track lists   north_star (c)
 *
 * params.mode = 1 selects the "no-UT" tuning of the same path (section VI.E): the seeds are
 * VELO tracks without momentum or charge; a1/a2 become a straight-line extrapolation with the double-sided
 * windows of Eq. (7)/(8) and Table 5; each window side (charge assumption) is followed separately through
 * a3..a6 and the lowest Q over both sides is kept (readings N1..N9).
 *
 * All of it runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  The readings of
 * the points the paper leaves open are listed in DESIGN.md ("Readings", C1..C22).
 *
 * Conventions
 *   - Plain C99 types only.  No exceptions cross the ABI; every call returns an lf_status.
 *   - Unless a function says HOST, every data pointer is a DEVICE pointer (cudaMalloc'd or a
 *     torch CUDA tensor's data_ptr) owned by the caller; the library never frees or reallocates
 *     caller memory.  The library owns only its workspace (allocated in lf_create, never on the
 *     hot path) and its constant tables.
 *   - Lengths in mm, momenta in GeV, q/p in 1/GeV.
 *   - Layout (north_star (b)): hits are event-major, then layer 0..11, then zone 0 (y < 0) /
 *     zone 1 (y >= 0); the 24 segments of one event are contiguous; inside each segment the stored
 *     coordinate s = x + y*tan_alpha is ASCENDING (precondition, not checked).  Offsets are
 *     monotone.  q/p is finite.
 *   - Output order contract: tracks are ordered by (event, seed index); at most one per seed.
 *   - Limits: n_hits, n_seeds < 2^31 per call; at most 2^25 seeds and 2^25 hits in one event (packed per-event
 *     indices in the library's tables); n_window <= 64, n_triplets <= 32.
 */
#ifndef LF_H
#define LF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LF_ABI_VERSION 7u
#define LF_N_LAYERS 12   /* three T-stations, x-u-v-x each */
#define LF_N_ZONES 2     /* lower / upper half */
#define LF_MAX_WINDOW 32   /* largest params.n_window of the narrow kernels (one warp lane per hit) */
#define LF_MAX_TRIPLETS 16 /* largest params.n_triplets of the narrow kernels */
#define LF_MAX_WINDOW_WIDE 64   /* largest params.n_window at all: beyond LF_MAX_WINDOW / LF_MAX_TRIPLETS, and always */
#define LF_MAX_TRIPLETS_WIDE 32 /* in the no-UT mode, the library runs the wide build of its kernels */

typedef struct lf_handle lf_handle; /* opaque; owned by the library */

typedef enum {
  LF_OK = 0,
  LF_ERR_INVALID_ARG = 1, /* NULL pointer, inconsistent size, value out of the documented range */
  LF_ERR_CUDA = 2,        /* a CUDA runtime call failed (no device, out of memory, launch error) */
  LF_ERR_CAPACITY = 3,    /* batch larger than lf_create's maxima, or out->capacity < n_seeds */
  LF_ERR_UNSUPPORTED = 4  /* valid request this build does not implement */
} lf_status;

/* Detector + field model (section V).  HOST struct, copied at lf_create. */
typedef struct {
  int32_t n_layers;              /* must be LF_N_LAYERS */
  float z[LF_N_LAYERS];          /* layer z positions */
  float tan_alpha[LF_N_LAYERS];  /* stereo: stored s = x + y*tan_alpha; must be 0 for layers 0,3 (mod 4),
                                    non-zero for layers 1,2 (mod 4) */
  float z_seed, z_mag, kick;     /* z of the seed state; magnet centre; delta tx = kick * q/p (Eq. 2) */
  float z_ref, d_ratio;          /* Eq. (1)/(4): dz = z - z_ref (8520 mm); dRatio per mm */
  float k_first, k_last;         /* sagitta factors K_x1 of the two layer sets */
  float qop_poly[5];             /* Eq. (9): q/p = dSlope / sum_i qop_poly[i] * dSlope^i */
  float x_half, y_half;          /* acceptance; used by generators only, ignored by the library */
  float z_state;                 /* z at which the output state is evaluated */
  int32_t polarity;              /* +1 = MU, -1 = MD; selects the asymmetric window edge (Eq. 3) */
  /* Full Eq. (9): the coefficient of dSlope^i is a 2-D polynomial in the seed's slopes,
   * c_i(tx, ty) = sum_j qop_poly2d[i][j] * tx^k * ty^m over the terms the field symmetries allow, k + m <= 6:
   *   even i: (k,m) = (0,0) (2,0) (0,2) (4,0) (2,2) (0,4) (6,0) (4,2) (2,4) (0,6)
   *   odd  i: (k,m) = (1,0) (3,0) (1,2) (5,0) (3,2) (1,4); slots 6..9 are not read.
   * qop_mode = 0: c_i = qop_poly[i] (constants); qop_mode = 1: the table (qop_poly is then not read). */
  int32_t qop_mode;
  float qop_poly2d[5][10];
} lf_geometry;

/* Tunables: Table 3 "Forward" column, Table 4 and the DESIGN.md readings.
 * HOST struct, copied at lf_create. */
typedef struct {
  float T_triplet, T_x, T_uv_slope, T_uv_min, T_ty, T_y, T_Q; /* 8, 2, 50, 0.5, 0.02, 800, 0.5 */
  float C_nhits[4];                                           /* C(n) for n = 9..12: 5, 1, 0.8, 0.5 */
  int32_t n_window, n_triplets, min_hits;                     /* 32, 12, 9 (no-UT: 64, 20, 9);  2 <= n_window <=
                                                                 LF_MAX_WINDOW_WIDE, 1 <= n_triplets <= LF_MAX_TRIPLETS_WIDE */
  float xtol_base, xtol_inv_p, x_asym, uv_half_width;         /* 150, 2000, 100, 800 */
  float p_same_bend, mag_tol_base, mag_tol_inv_p, mag_tol_tx, mag_tol_max; /* 5, 8, 60, 20, 40 */
  int32_t hit_storage;                                        /* 0 = fp32 (bit-exact reference path); 1 = the window and
                                                                 seeding kernels read an fp16 copy of the hits (block-offset
                                                                 encoding, lf_pack_hits; the caller's, or packed by the
                                                                 library at every lf_run); extension and fit stay on the
                                                                 fp32 hits when lf_hits.x is given (BASELINE.json
                                                                 configs[2]); mode 0 with the narrow limits only
                                                                 (LF_ERR_UNSUPPORTED otherwise) */
  /* no-UT tuning; read only when mode == 1 */
  int32_t mode;                  /* 0 = with UT (sections VI.A-D); 1 = no-UT (section VI.E): seeds->qop is not read, the same-bend
                                    filter does not exist, the magnet tolerance uses the assumed 1/p where q/p stood */
  float velo_p_min, velo_pt_min; /* assumed minimum momentum / transverse momentum, GeV: 5, 1; > 0 */
  float xtol_poly[8];            /* c0..c7 of Eq. (7), Table 5 */
  float x_overlap;               /* overlap of the LEFT and RIGHT windows of Eq. (8): 5 mm */
  /* read only when hit_storage == 1 */
  int32_t seed_arith;            /* 1 = one doublet per lane in fp32 on the decoded fp16 hits: the recommended setting and what the
                                    repository's parameter sets (datagen.default_params, bench.py) use, because it is the faster of
                                    the two on B200; 0 = the seeding kernel evaluates PAIRS of doublets in
                                    __half2 ("two combinations at a time"), kept as the measured comparison.  Both
                                    pass configs[2]'s rule */
} lf_params;

/* Input seeds: upstream track states at z_seed, SoA, all events back to back. */
typedef struct {
  const float *x, *y, *tx, *ty, *qop; /* n_seeds each; qop is not read (may be NULL) when params.mode == 1 */
  const uint32_t* event_offsets;      /* n_events + 1; seeds of event e are [off[e], off[e+1]) */
  size_t n_seeds;                     /* == event_offsets[n_events] (caller's knowledge; no device read-back) */
} lf_seeds;

/* Input hits. */
typedef struct {
  const float* x;              /* n_hits stored coordinates (fp32); may be NULL when params.hit_storage == 1 and x16 is given */
  const uint32_t* seg_offsets; /* n_events*24 + 1; segment index = event*24 + layer*2 + zone */
  size_t n_hits;               /* == seg_offsets[n_events*24] */
  /* params.hit_storage == 1 only (ignored otherwise; both NULL = the library packs `x` itself at every lf_run):
   * the fp16 copy of the hits in the block-offset encoding lf_pack_hits writes.  With x == NULL every stage reads
   * this copy (2.125 bytes per hit to move); with x given, extension and fit read the fp32 hits. */
  const uint16_t* x16;         /* n_hits IEEE binary16 offsets */
  const float* origin16;       /* lf_origin_slots(n_events, n_hits) block origins */
} lf_hits;

/* Output tracks (dense, (event, seed) order).  Arrays must hold `capacity` rows;
 * capacity >= seeds->n_seeds is required (at most one track per seed), so no
 * overflow is possible and no host synchronisation is needed to size anything. */
typedef struct {
  int32_t* hit_idx;        /* capacity*12: global hit index used on each layer, or -1; 16-byte aligned (lf_run) */
  int32_t* seed_idx;       /* capacity: global index of the seed the track extends */
  int32_t* n_hits;         /* capacity: number of hits (>= params.min_hits) */
  float* state;            /* capacity*5: x, y, tx, ty, q/p at geometry.z_state */
  float* quality;          /* capacity: Q of Eq. (6) */
  uint32_t* event_offsets; /* n_events + 1: tracks of event e are [off[e], off[e+1]) */
  uint32_t* n_tracks;      /* 1: total number of tracks written */
  size_t capacity;
} lf_tracks;

/* Optional stage-boundary outputs for parity tests (device pointers; any may be NULL).
 * NT = params.n_triplets.  Indices are global hit indices; -1 = none.  Rows are followed tracks: one per seed
 * (row = seed) when mode == 0; one per (seed, window side) when mode == 1, row = 2*seed + side with side 0 =
 * LEFT and 1 = RIGHT window of Eq. (8): read n_seeds below as the number of rows. */
typedef struct {
  int32_t* win_first;   /* n_seeds*12: first hit of the (capped) search window (undefined if empty) */
  int32_t* win_count;   /* n_seeds*12: hits in the window (<= n_window) */
  int32_t* n_triplets;  /* n_seeds: triplets kept, ordered by (chi2, set, h0, h2) */
  int32_t* trip_hits;   /* n_seeds*NT*3: h0, h1, h2 */
  int32_t* trip_set;    /* n_seeds*NT: 0 = first x layers {0,4,8}, 1 = last x layers {3,7,11} */
  float* trip_chi2;     /* n_seeds*NT */
  int32_t* cand_hits;   /* n_seeds*NT*12: hit per layer after extension */
  float* cand_quality;  /* n_seeds*NT: Q; -1 = failed the hit-count rule; -2 = failed the t_y cut */
} lf_debug;

/* What the library launches, for benchmarks and occupancy reports (HOST struct, filled by lf_get_info).
 * Per-kernel arrays are indexed LF_K_WINDOW .. LF_K_FIT (the four event kernels). */
#define LF_K_WINDOW 0  /* a1, a2 */
#define LF_K_SEED 1    /* a3 */
#define LF_K_EXTEND 2  /* a4, a5 */
#define LF_K_FIT 3     /* a6, a7: fit, best candidate per seed, and the stream compaction (look-back scan of the events'
                          track counts + copy of the tracks to their dense position) */
#define LF_N_EVENT_KERNELS 4
#define LF_N_KERNELS 4 /* kernels one lf_run enqueues = entries of lf_kernel_times */
typedef struct {
  int32_t kernels_per_run;       /* kernel launches the most recent lf_run / lf_run_debug on the handle enqueued (lf_run_host: its
                                    last chunk): 4; 5 with hit_storage = 1 when the library packed the hits itself (no x16 / origin16
                                    from the caller); 0 for an empty batch.  Before the first run: the upper bound, 4 + hit_storage */
  int32_t regs[LF_N_EVENT_KERNELS], block[LF_N_EVENT_KERNELS], grid[LF_N_EVENT_KERNELS], ctas_per_sm[LF_N_EVENT_KERNELS];
  int32_t smem_bytes[LF_N_EVENT_KERNELS]; /* dynamic shared memory per CTA */
  int32_t staged_hits_per_event; /* events with more hits than this read hits from global memory */
  int32_t sm_count;
  size_t workspace_bytes;
} lf_info;

/* Creates a context for batches of at most max_events / max_seeds / max_hits.  Validates geometry
 * and params (finite, tolerances >= 0, kick != 0), uploads constants, allocates the workspace (about
 * max_seeds*(153 + 18*n_triplets) + max_events*20 bytes, roughly twice that in the no-UT mode; with hit_storage = 1
 * another 6.5 bytes per hit) on the current CUDA device, sized for 180 GB parts.  The shared-memory stage for one event's
 * hits is sized from the maxima: 1.25 * max_hits / max_events + 512 hits, clamped to [2048, 16384] (the seeding kernel
 * stages the x layers only, half of that); larger events are still processed correctly, reading their hits from global
 * memory.  Handles of different sizes may be alive at the same time.  *out is set only on LF_OK.  HOST pointers. */
lf_status lf_create(const lf_geometry* geometry, const lf_params* params, size_t max_events,
                    size_t max_seeds, size_t max_hits, lf_handle** out);

/* Enqueues the whole hot path (a1..a7) for n_events events on `cuda_stream` (a cudaStream_t; NULL =
 * the legacy default stream).  Asynchronous: performs no host synchronisation and returns after the
 * launches; results are valid once the caller has synchronised the stream.  `seeds`, `hits`, `out`
 * are HOST structs holding DEVICE pointers.  Safe to call repeatedly; calls on one handle must not
 * overlap in time (they share the workspace).  n_events == 0 is valid (writes n_tracks = 0).
 * The call only enqueues kernels, so it may be captured into a CUDA graph and replayed (tests/test_gpu_parity.py).
 * Errors are detected before any launch: LF_ERR_INVALID_ARG (NULL pointer), LF_ERR_CAPACITY. */
lf_status lf_run(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events,
                 lf_tracks* out, void* cuda_stream);

/* lf_run that also writes the stage-boundary tables of `debug` (slower; for tests). */
lf_status lf_run_debug(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events,
                       lf_tracks* out, const lf_debug* debug, void* cuda_stream);

/* End-to-end variant: every pointer inside `seeds`, `hits`, `out` is a HOST pointer (pinned memory
 * makes the copies asynchronous and lets them overlap the kernels).  The batch is pipelined in chunks of
 * events (the seeds of the whole batch first; then the hits in at most 13 equal chunks of at least 2048 events, see
 * lf_set_host_chunk_events, the last of them cut into four shrinking pieces to shorten the pipeline's tail): the host->device copy
 * of chunk c+1, the kernels of chunk c (on `cuda_stream`) and the device->host copy of the tracks of chunk
 * c-1 (library-owned copy streams, ordered after the work already queued on `cuda_stream`) run
 * concurrently; device buffers are library-owned, allocated on first use and sized by lf_create's maxima.
 * The call reads the two HOST offset tables to place the chunks (LF_ERR_INVALID_ARG if
 * event_offsets[0] != 0, event_offsets[n_events] != n_seeds or seg_offsets[n_events*24] != n_hits) and
 * returns after all copies have completed: on LF_OK the host arrays hold exactly what lf_run would have
 * produced for the whole batch (dense, (event, seed) order). */
lf_status lf_run_host(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events,
                      lf_tracks* out, void* cuda_stream);

/* The same in two halves, for a stream of batches: lf_host_submit enqueues everything that needs no answer from the
 * device (the host->device copies of the whole batch, the kernels of every chunk on `cuda_stream`, the read-back of the
 * chunks' track counts) and returns at once; lf_host_collect then places the tracks in the caller's arrays as the chunks
 * finish and returns when the batch's last byte has arrived (it does not wait for anything queued behind the batch).
 * LF_HOST_SLOTS batches can be in flight on one handle, each in its own slot (its own device staging, allocated on first
 * use), so that
 *     submit(batch 0, slot 0); for (i = 1; i < n; ++i) { submit(batch i, slot i % 2); collect(slot (i - 1) % 2); } collect(last)
 * copies batch i + 1 to the device while batch i is still being computed and copied back: the stream of batches then runs
 * at the speed of the host->device link.  lf_run_host(..) == lf_host_submit(.., slot 0) + lf_host_collect(slot 0), except that
 * lf_host_submit starts its copies at once (the caller's host arrays must be complete when it is called) instead of after the
 * work already queued on `cuda_stream`.  The host arrays of `seeds`, `hits` and `out` must stay valid and untouched until the
 * batch has been collected (the structs themselves are copied).  Batches in flight share the handle's workspace, so they must
 * all use the same `cuda_stream` (LF_ERR_INVALID_ARG otherwise); a slot takes a new batch only after its previous one has been
 * collected; lf_run and lf_run_host must not be called while a batch is in flight.  An LF_ERR_CUDA from lf_host_submit or
 * any error from lf_host_collect ABORTS EVERY BATCH IN FLIGHT on the handle: the library waits for its own copy streams and
 * for the stream each pending batch was submitted on, marks all slots idle (their batches can no longer be collected; the
 * host output arrays hold unspecified data) and leaves the handle ready for the next lf_run / lf_host_submit. */
#define LF_HOST_SLOTS 2
lf_status lf_host_submit(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events,
                         lf_tracks* out, void* cuda_stream, int slot);
lf_status lf_host_collect(lf_handle* h, int slot);

/* Smallest number of events lf_run_host puts in one equal pipeline chunk (default 2048; >= 1).  The number of
 * equal chunks is min(13, max(1, n_events / min_events_per_chunk)); the last one is cut into four pieces. */
lf_status lf_set_host_chunk_events(lf_handle* h, size_t min_events_per_chunk);

/* fp16 hit storage (params.hit_storage == 1; "store hit data in fp16 in addition to fp32"; BASELINE.json
 * configs[2]).  Encoding: inside every (event, layer, zone) segment consecutive hits form blocks of 8; a block's origin
 * is the fp32 coordinate of its 5th hit (its last one if shorter); every hit stores binary16(x - origin), so the offset
 * stays within half a block's span (rounding error below 0.25 mm at Run-3 occupancy, median 0.006 mm).  The origin of block
 * b of global segment g that starts at hit S sits in slot (S >> 3) + g + b: lf_origin_slots(n_events, n_hits) =
 * (n_hits >> 3) + 24 * n_events + 2 slots hold them all.  lf_pack_hits writes both arrays from fp32 hits (DEVICE pointers,
 * asynchronous on `cuda_stream`; `hits->x` and `hits->seg_offsets` are read); the result can be kept, copied to the host
 * and handed to lf_run / lf_run_host in lf_hits.x16 / origin16 of later calls with the same offsets. */
size_t lf_origin_slots(size_t n_events, size_t n_hits);
lf_status lf_pack_hits(lf_handle* h, const lf_hits* hits, size_t n_events, uint16_t* x16_out, float* origin16_out,
                       void* cuda_stream);

/* Checks, on the device, the input preconditions lf_run relies on but does not check (see "Conventions"): segment
 * offsets monotone, starting at 0 and ending at n_hits; stored coordinates finite and ascending inside every
 * segment; seed offsets monotone, starting at 0 and ending at n_seeds; seed states finite (q/p only when params.mode
 * == 0).  With the fp16 copy as the only hit input (hits->x == NULL, hit_storage = 1, x16 + origin16 given) the decoded
 * coordinates are checked instead: finite, and ascending inside every block of 8 hits (across blocks the encoding may
 * overlap by a rounding error, which that lossy mode accepts).
 * Arguments as for lf_run (HOST structs holding DEVICE pointers); `out` is not needed.  SYNCHRONOUS: waits
 * for `cuda_stream`.  Returns LF_OK, or LF_ERR_INVALID_ARG with lf_last_error naming the kind of violation and the
 * index of one offending segment / hit / event / seed.  A debugging aid: not part of the hot path. */
lf_status lf_validate_inputs(lf_handle* h, const lf_seeds* seeds, const lf_hits* hits, size_t n_events, void* cuda_stream);

/* Frees the workspace and the handle.  NULL is allowed. */
lf_status lf_destroy(lf_handle* h);

/* Message of the last error on this handle ("" if none); valid until the next call on the handle.
 * With h == NULL: message of the last failed lf_create in this thread. */
const char* lf_last_error(const lf_handle* h);

lf_status lf_get_info(const lf_handle* h, lf_info* out);

/* Per-kernel device timing for benchmarks.  With profiling enabled, lf_run / lf_run_debug record CUDA
 * events on `cuda_stream` around each of their kernels (no synchronisation added).  After the caller
 * has synchronised the stream, lf_kernel_times writes the mean durations in milliseconds over the runs
 * recorded since profiling was enabled (the last 256 at most): ms[0] window kernel (a1, a2), ms[1] seeding
 * kernel (a3), ms[2] extension kernel (a4, a5), ms[3] fit kernel (a6 and the stream compaction a7).
 * LF_ERR_INVALID_ARG if profiling is off or no run was recorded. */
lf_status lf_set_profiling(lf_handle* h, int enabled);
lf_status lf_kernel_times(lf_handle* h, float ms[LF_N_KERNELS]);

/* Work counters of the most recent lf_run / lf_run_debug on this handle (for lf_run_host: of its last chunk), for
 * benchmarks and for the algorithmic work model of DESIGN.md section 7:
 *   [0] candidates that passed the hit-count rule (16-byte records handed from the extension kernel to the fit kernel)
 *   [1] events holding two equal neighbouring hits
 * and, counted only by lf_run_debug (0 after a plain lf_run; any or all pointers of lf_debug may be NULL):
 *   [2] hits inside the search windows, summed over followed tracks and layers (a2)
 *   [3] candidate doublets the seeding kernel evaluated (its bracket of the magnet-opening cut; implementation-specific)
 *   [4] doublets that passed both filters of PAPER.md:210-211 (a3)
 *   [5] triplets that passed the chi2 cut, before the top-n selection (a3)
 *   [6] triplets kept = candidates extended (a4, a5)
 *   [7] tracks written (a6, a7)
 * SYNCHRONOUS: waits for the device, then reads the tables back. */
#define LF_N_COUNTERS 8
lf_status lf_run_counters(lf_handle* h, uint64_t counters[LF_N_COUNTERS]);

/* Search windows (a1 + a2, no-UT: Eq. 7/8) without any allocation and without a handle.
 *
 * Who this is for.  Everything else in this header goes through lf_create, which calls cudaMalloc.  Some hosts cannot
 * afford or are not allowed that call: a trigger application whose framework grabs the whole GPU at start-up and hands
 * out slices itself (a later cudaMalloc then simply fails for lack of memory), an event loop with a latency budget
 * (cudaMalloc and cudaFree stall the whole device and take unbounded time), a plug-in that lives inside somebody else's
 * memory pool, or code that runs where the CUDA allocator must not be entered at all.  Such a caller can still ask this
 * one function which hits each seed would look at: it brings its own input and output buffers, and the kernel's scratch
 * memory is a fixed array compiled into the library (`static __device__`, LF_STATIC_SCRATCH_BYTES = 1 097 984 bytes).
 * The price: every GPU whose context loads this library holds that array from load time until the process exits, whether
 * or not this function is ever called, and the batch size is bounded:
 *     n_events <= LF_STATIC_MAX_EVENTS, followed tracks = seeds->n_seeds * (params->mode == 1 ? 2 : 1) <= LF_STATIC_MAX_ROWS;
 * anything larger is refused with LF_ERR_CAPACITY (split the batch, or use lf_create + lf_run_debug).
 *
 * Arguments: `geometry`, `params` HOST structs as for lf_create (validated the same way; params->hit_storage must be 0,
 * LF_ERR_UNSUPPORTED otherwise); `seeds`, `hits` HOST structs holding DEVICE pointers as for lf_run; `win_first`,
 * `win_count` DEVICE arrays of (followed tracks) * 12 int32, caller-owned, with the meaning and row order of
 * lf_debug.win_first / win_count (global index of the window's first hit -- undefined where the count is 0 -- and the
 * number of hits, <= params->n_window).  The result is what lf_run_debug writes into those two tables, bit for bit.
 * Asynchronous on `cuda_stream` (one 4-byte memset + one kernel); results are valid once the stream has been synchronised.
 * The function calls no cudaMalloc, cudaMallocAsync, cudaFree or other routine that allocates device memory.
 *
 * First call on a device: looks up, once per device and with that device current, where the array lives there
 * (cudaGetSymbolAddress), reads two device attributes and makes sure the window kernel may use the 33 KB of shared
 * memory it is launched with (a function attribute; an lf_create for small events may have set it lower).  The lookup can
 * make the CUDA runtime load the library's code onto the device, so make the first call per device early, during
 * set-up, and before any stream capture begins.
 *
 * Sharing: all calls on a device use the same array, and the array keeps whatever the previous call left in it.  The
 * function clears the one word that has to start at zero (the event counter its thread blocks draw from) at the head of
 * its own work on `cuda_stream`; everything else is overwritten before it is read.  Two calls whose GPU work overlaps in
 * time (different streams, or different host threads on different streams) race on the array and give garbage: keep
 * calls on one device in stream order, or order them with events.  lf_create handles do not touch the array.
 * Errors: status code; the message is lf_last_error(NULL) in the calling thread.  Size and argument errors are found
 * before the first CUDA call. */
#define LF_STATIC_MAX_EVENTS 4096
#define LF_STATIC_MAX_ROWS 16384
#define LF_STATIC_SCRATCH_BYTES (LF_STATIC_MAX_ROWS * 64 + LF_STATIC_MAX_EVENTS * 12 + 256)
lf_status lf_windows_static(const lf_geometry* geometry, const lf_params* params, const lf_seeds* seeds,
                            const lf_hits* hits, size_t n_events, int32_t* win_first, int32_t* win_count,
                            void* cuda_stream);

/* ABI self-description for bindings: version and struct sizes
 * (which: 0 geometry, 1 params, 2 seeds, 3 hits, 4 tracks, 5 debug, 6 info). */
uint32_t lf_abi_version(void);
size_t lf_sizeof(int which);

#ifdef __cplusplus
}
#endif
#endif /* LF_H */
