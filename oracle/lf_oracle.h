/*
 * lf_oracle.h -- C interface of the CPU ORACLE for the Looking Forward hot path (arxiv 2402.14670).
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, single-threaded restatement of the algorithm
 * as PAPER.md defines it (readings of the silent/garbled points: DESIGN.md "Readings", C1..C22).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code, header, table or helper with the CUDA path
 * (paper_2402_14670_b200/csrc, include/lf.h); the struct definitions below are deliberately its
 * own.  All pointers are HOST pointers.
 *
 * Parity pins (tests/test_oracle_pins.py, all -m "not gpu"):
 *   - brute-force twin (oracle/brute_twin.py): no sortedness, no binary search, full sorts;
 *   - generator truth: noise-free single tracks found with exactly their hits, closed forms for
 *     the triplet parabola, K_x1 and q/p;
 *   - invariants on every config; LSQ fits vs numpy.linalg.lstsq in float64; windows vs
 *     numpy.searchsorted; fp32 build vs fp64 build of this same file.
 * Parity-unpinned BY THE PAPER (pinned only by DESIGN.md's reading): the magnet-tolerance formula
 * (C6), the T_uv floor (C12), which chi^2 enters Q (C13); in the no-UT mode: whether the triplet cap
 * is per charge assumption or per track (N6).
 */
#ifndef LF_ORACLE_H
#define LF_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LFO_N_LAYERS 12

typedef struct {
  int32_t n_layers;               /* must be 12: three stations x-u-v-x */
  float z[LFO_N_LAYERS];          /* layer z, mm */
  float tan_alpha[LFO_N_LAYERS];  /* stored coordinate s = x + y*tan_alpha; 0 for x layers */
  float z_seed, z_mag, kick;      /* seed-state z; magnet centre; dtx = kick*q/p */
  float z_ref, d_ratio;           /* Eq. (1)/(4): dz = z - z_ref, dRatio per mm */
  float k_first, k_last;          /* K_x1 per layer set */
  float qop_poly[5];              /* Eq. (9): F(dSlope) = sum c_i dSlope^i */
  float x_half, y_half;           /* acceptance (generator only; unused here) */
  float z_state;                  /* z of the output state */
  int32_t polarity;               /* +1 = MU, -1 = MD (Eq. 3) */
  /* Full Eq. (9): c_i(tx, ty) = sum_j qop_poly2d[i][j] tx^k ty^m over the terms allowed by the
   * field symmetries, k + m <= 6.  Even i: (k,m) = (0,0) (2,0) (0,2) (4,0) (2,2) (0,4) (6,0) (4,2) (2,4) (0,6);
   * odd i: (1,0) (3,0) (1,2) (5,0) (3,2) (1,4), slots 6..9 unused.  qop_mode 0: c_i = qop_poly[i] (constants). */
  int32_t qop_mode;
  float qop_poly2d[5][10];
} lfo_geometry;

typedef struct {
  float T_triplet, T_x, T_uv_slope, T_uv_min, T_ty, T_y, T_Q;   /* Table 3 */
  float C_nhits[4];                                             /* Table 4, n = 9..12 */
  int32_t n_window, n_triplets, min_hits;                       /* 32, 12 (Table 3); 9 */
  float xtol_base, xtol_inv_p, x_asym, uv_half_width;
  float p_same_bend, mag_tol_base, mag_tol_inv_p, mag_tol_tx, mag_tol_max;
  int32_t hit_storage;                                          /* ignored: the oracle is always fp32 storage */
  /* "no-UT" tuning: VELO seeds without momentum, double-sided windows. */
  int32_t mode;                 /* 0 = with UT (sections VI.A-D), 1 = no-UT (section VI.E) */
  float velo_p_min, velo_pt_min; /* assumed minimum momentum / transverse momentum, GeV: 5, 1 */
  float xtol_poly[8];           /* c0..c7 of Eq. (7), Table 5 */
  float x_overlap;              /* overlap of the two windows of Eq. (8): 5 mm */
} lfo_params;

typedef struct {
  const float *x, *y, *tx, *ty, *qop;  /* SoA, n_seeds each */
  const uint32_t* event_offsets;       /* n_events + 1 */
} lfo_seeds;

typedef struct {
  const float* x;                /* stored coordinate, ascending inside each segment */
  const uint32_t* seg_offsets;   /* n_events*24 + 1; segment = (event, layer, zone) */
} lfo_hits;

typedef struct {
  int32_t* hit_idx;        /* capacity*12: global hit index per layer or -1 */
  int32_t* seed_idx;       /* capacity: global seed index */
  int32_t* n_hits;         /* capacity */
  float* state;            /* capacity*5: x, y, tx, ty, q/p at z_state */
  float* quality;          /* capacity: Q of Eq. (6) */
  uint32_t* event_offsets; /* n_events + 1 */
  uint32_t* n_tracks;      /* 1 */
  size_t capacity;         /* rows available in the arrays above */
} lfo_tracks;

/* Optional stage-boundary outputs (any pointer may be NULL).  NT = params.n_triplets.
 * Rows are "followed tracks": mode 0 one per seed (row = seed); mode 1 one per (seed, window side),
 * row = 2*seed + side, side 0 = LEFT, 1 = RIGHT of Eq. (8); read n_seeds below as the number of rows. */
typedef struct {
  int32_t* win_first;     /* n_seeds*12: global index of the first hit of the (capped) window */
  int32_t* win_count;     /* n_seeds*12 */
  int32_t* n_triplets;    /* n_seeds: triplets kept (<= NT), in C9 order */
  int32_t* trip_hits;     /* n_seeds*NT*3: global hit indices h0,h1,h2 */
  int32_t* trip_set;      /* n_seeds*NT: 0 = first layers, 1 = last layers */
  float* trip_chi2;       /* n_seeds*NT */
  int32_t* cand_hits;     /* n_seeds*NT*12: hits after extension (global index or -1) */
  float* cand_quality;    /* n_seeds*NT: Q; -1 = failed hit-count rule; -2 = failed ty cut */
} lfo_debug;

/* Runs stages O1..O7 for every seed of every event.  Returns 0 ok, 1 invalid argument,
 * 3 out->capacity too small. */
int lf_oracle_run(const lfo_geometry* geometry, const lfo_params* params, const lfo_seeds* seeds,
                  const lfo_hits* hits, size_t n_events, lfo_tracks* out, lfo_debug* debug);

/* sizeof(real type) this build computes in: 4 (reference) or 8 (pin build, -DLF_ORACLE_REAL=double). */
int lf_oracle_real_bytes(void);

#ifdef __cplusplus
}
#endif
#endif
