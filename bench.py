#!/usr/bin/env python
"""Benchmark of the Looking Forward hot path on B200 (contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--events E] [--tuning with-ut|no-ut]

A "step" is one pass of the whole hot path (a1..a7: one lf_run = window, seed, extend, fit kernels; the fit kernel also compacts)
over one batch of synthetic events.  Default workload: BASELINE.json configs[3] (20,000 events at
Run-3-like occupancy, fp32, a single lf_run on one stream).  Prints ONE JSON line (rank 0).

  value        events/s with inputs resident in HBM (CUDA events around the K steps, max over ranks)
  e2e          the same metric through the host path (lf_host_submit / lf_host_collect, two batches in flight; the one-call
               lf_run_host figure beside it): pinned HOST buffers, H2D + D2H inside the timing
  roofline     the HBM roofline BASELINE.json's metric names, for the dominant kernel (the slowest event kernel, timed
               live with CUDA events on the launching stream): algorithmic bytes per launch / duration vs the measured
               copy bandwidth of MEASURED_PEAKS.json; "traffic" = DRAM bytes per launch from the committed ncu capture
               when that capture was taken on this very source (sha256 stamp), else null
  alu_algorithmic_frac  ALGORITHMIC lane-operations per step (the committed model of DESIGN.md section 7, evaluated on this
               batch's own work counters) / step time / (148 SMs x 128 lanes x sm_max_mhz)
  issue_utilisation     EXECUTED warp-instructions of the dominant kernel (ncu capture, same sha256 stamp) / its live time /
               (148 SMs x 4 schedulers x sm_max_mhz): how busy the issue slots are, not a roofline fraction
  cpu_baseline the oracle, as it stands, on the box's host cores on a bounded sample (rank 0, N=1)

--impl reference times the oracle (all host cores via the harness's event sharding) on a bounded
sample of the same workload; under torchrun only rank 0 works.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0   # BASELINE.json north_star: "over 8 TB/s"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region (NVML; nvidia-smi as a fallback)."""

    def __init__(self, index: int, period_s: float = 0.02):
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nvml = None

    def _reason_names(self, mask: int):
        n = self._nvml
        table = (("hw_slowdown", "nvmlClocksEventReasonHwSlowdown", 0x8), ("hw_thermal_slowdown", "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 ("sw_thermal_slowdown", "nvmlClocksEventReasonSwThermalSlowdown", 0x20), ("sw_power_cap", "nvmlClocksEventReasonSwPowerCap", 0x4),
                 ("hw_power_brake", "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80))
        return [name for name, attr, default in table if mask & getattr(n, attr, default)]

    def _loop(self):
        n = self._nvml
        while not self._stop.is_set():
            try:
                self.samples.append(int(n.nvmlDeviceGetClockInfo(self._h, n.NVML_CLOCK_SM)))
                try:
                    mask = int(n.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    mask = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                self.reasons.update(self._reason_names(mask))
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self._nvml is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        if self._nvml is None or not self.samples:
            return self._smi_once()
        return {"sm_mhz": float(statistics.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples), "source": "nvml during timed region"}

    def _smi_once(self):
        import subprocess
        try:
            out = subprocess.run(["nvidia-smi", f"--id={self.index}", "--query-gpu=clocks.sm,clocks.max.sm,clocks_event_reasons.active",
                                  "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=20).stdout.strip().split(",")
            return {"sm_mhz": float(out[0]), "sm_max_mhz": float(out[1]), "reasons": [out[2].strip()], "samples": 1,
                    "source": "nvidia-smi after timed region (NVML unavailable)"}
        except Exception as e:  # pragma: no cover
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [f"unavailable: {e}"], "samples": 0}


def source_sha256() -> str:
    """Stamp of the kernel sources a committed ncu capture must carry to describe this build."""
    import hashlib
    h = hashlib.sha256()
    for rel in ("paper_2402_14670_b200/csrc/lf_kernels.cuh", "paper_2402_14670_b200/csrc/lf_api.cu"):
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


# Algorithmic work model ("Algorithmic lane-operations"): lane-operations (one fp32 / int32 add,
# multiply, divide, abs, min / max, compare or select on one lane) that the canonical arithmetic of DESIGN.md section 3 needs
# per work item in the interval-search formulation of the method, at 100 % lane use.  Every coefficient is the sum of the
# terms below, one per expression of section 3; DESIGN.md carries the same table and tests/test_bench_contract.py pins the
# two to each other.  Loads, address arithmetic, packing of the library's tables and the work of mapping items to lanes
# are not counted: they belong to an implementation, not to the method.
LANE_OPS_TERMS = {
    "per_row": {                        # a1, once per followed track
        "aq = max(|qop|, 1e-6); p = 1/aq": 3,
        "x_mag = x + tx*(z_mag - z_seed)": 2,
        "txp = tx + kick*qop": 2,
        "xc_l = x_mag + txp*dzm_l on 12 layers": 24,
        "y_l = y + ty*dzs_l on the 6 u/v layers": 12,
        "yt_l = y_l*tan(alpha_l) on the 6 u/v layers": 6,
        "zone = (ty >= 0)": 1,
        "x_tol = xtol_base + xtol_inv_p*aq": 2,
        "a_left, a_right from sign(q) = polarity": 3,
    },
    "per_row_layer_fixed": {            # a2, once per (followed track, layer), besides the searches
        "lo = (xc - x_tol) - a_left; hi = (xc + x_tol) + a_right": 4,
        "mid = (lo + hi)*0.5": 2,
        "last - first > n_window": 2,
        "first = max(first, c - n/2); last = min(last, c + n/2)": 4,
    },
    "per_search_step": {                # every binary search
        "compare the probed hit": 1,
        "select the new position": 1,
    },
    "per_h0_hit": {                     # a3, once per hit of the first layer's window: the h2 interval filter 2 allows
        "d = x_mag - x0": 1,
        "largest |t| a doublet of this h0 can have": 2,
        "tol = min(mag_tol_max, c_seed + mag_tol_tx*|t|)": 3,
        "lo2 = x0 + (d - tol)*inv_r": 3,
        "hi2 = x0 + (d + tol)*inv_r": 3,
    },
    "per_doublet": {                    # a3, once per doublet that passes both filters
        "t = (x2 - x0)*inv_dz": 2,
        "filter 1: (t - tx)*(kick*qop) > 0": 3,
        "filter 2: |x0 + t*zmag_a - x_mag|": 4,
        "filter 2: < min(mag_tol_max, c_seed + mag_tol_tx*|t|)": 5,
        "x1e = z_b*t + (x0 - t*z_a)*K": 5,
        "(x1 - x1e)^2 < T_triplet": 3,
    },
    "closest_fixed": {                  # every closest-hit search, after its binary search
        "pred - x_left; x_right - pred": 2,
        "compare (ties -> lower index)": 1,
        "select hit and distance": 2,
        "index of the hit": 1,
    },
    "per_triplet_passing": {            # a3, once per triplet below the chi2 cut
        "key (chi2, set, h0, h2)": 4,
        "position among the n smallest: ceil(log2(12 + 1)) = 4 steps": 8,
    },
    "per_triplet_kept": {               # a4, once per triplet extended
        "X10 = x1 - x0; X20 = x2 - x0": 2,
        "c0 = (X20*D10 - X10*D20)*inv_det": 4,
        "t0 = (X10 - c0*W10)*inv_D10": 3,
        "a0 = (x0 - t0*d_a) - c0*w_a": 4,
    },
    "per_prediction": {                 # a4 / a5, once per (candidate, other layer)
        "pred = (a0 + t0*d_l) + c0*w_l": 4,
        "+ yt_l (u/v layers)": 1,
        "dist^2 < T_x or T_uv": 2,
    },
    "per_accepted": {                   # a6, once per candidate that passed the hit-count rule (12 hits, 6 of them u/v)
        "r_l = (s_l - yt_l) - ((a0 + t0*d_l) + c0*w_l): 6 u/v x 6 + 6 x x 5": 66,
        "Sr, Sdr, Swr over 12 hits (the geometry sums come from the per-mask table)": 60,
        "da, dt, dc = ((C.0*Sr + C.1*Sdr) + C.2*Swr)*inv_det": 18,
        "e_l = r_l - ((da + dt*d_l) + dc*w_l) on 12 hits": 60,
        "Q_x += e_l^2 * (1/T) on 12 hits": 36,
        "rho_l = e_l*inv_tan_l on 6 u/v hits": 6,
        "S_rho, S_d_rho over 6 u/v hits": 18,
        "dy0, dty from the 2x2 system": 8,
        "|dty*0.001| < T_ty": 3,
        "Q_y += (rho - (dy0 + dty*d))^2 * (1/T_y) on 6 u/v hits": 36,
        "Q = (Q_x/(n - 3) + Q_y/(n_uv - 2))*C(n); Q < T_Q; lowest Q of the seed": 12,
    },
    "per_track": {                      # a6 / a7, once per output track
        "dSlope = t*0.001 - tx; q/p = dSlope / F(dSlope), F of degree 4 by Horner": 11,
        "state x, tx, y, ty at z_state": 13,
        "20-word record moved to its dense position": 20,
    },
    "per_seed": {                       # a7
        "has-track flag": 1,
        "scan": 1,
    },
}
LANE_OPS = {k: sum(v.values()) for k, v in LANE_OPS_TERMS.items()}


def algorithmic_lane_ops(counters: dict, batch, n_window: int, sides: int) -> dict:
    """Evaluates the model on the batch's own counters (lf_run_counters after a counting run)."""
    import math
    L = LANE_OPS
    rows = batch.n_seeds * sides
    seg_len = batch.n_hits / max(batch.n_events * 24, 1)
    seg_steps = math.ceil(math.log2(seg_len + 1)) if seg_len > 0 else 0
    win_steps = math.ceil(math.log2(n_window + 1))
    closest = win_steps * L["per_search_step"] + L["closest_fixed"]
    h0_hits = counters["window_hits"] / 6.0  # two of the twelve layers open the two layer sets
    parts = {
        "a1_a2": rows * (L["per_row"] + 12 * (L["per_row_layer_fixed"] + 2 * seg_steps * L["per_search_step"])),
        "a3": h0_hits * (L["per_h0_hit"] + 2 * win_steps * L["per_search_step"])
              + counters["doublets_passing"] * (L["per_doublet"] + closest)
              + counters["triplets_passing"] * L["per_triplet_passing"],
        "a4_a5": counters["triplets_kept"] * (L["per_triplet_kept"] + 9 * (L["per_prediction"] + closest)),
        "a6": counters["accepted_candidates"] * L["per_accepted"] + counters["tracks"] * L["per_track"],
        "a7": batch.n_seeds * L["per_seed"],
    }
    parts["total"] = float(sum(parts.values()))
    return parts


def algorithmic_bytes(batch, n_tracks: int) -> int:
    """Unique HBM bytes the method must move: inputs read once, tracks written once."""
    return int(4 * batch.n_hits + batch.seg_offsets.nbytes + 20 * batch.n_seeds + batch.seed_offsets.nbytes
               + 80 * n_tracks + 4 * (batch.n_events + 1) + 4)


def kernel_bytes(batch, n_tracks: int, n_triplets: int, n_acc: int = 0, sides: int = 1, wide: bool = False) -> dict:
    """Algorithmic HBM bytes per launch of each event kernel: every kernel stages the hits it needs
    once (all twelve layers; the seeding kernel only the six x layers) and reads / writes its own tables once.  Tables are
    per followed track (row): one per seed, or one per (seed, window side) in the no-UT tuning (64-byte window rows; the
    wide kernels store 4-byte triplet codes)."""
    H, S, E = batch.n_hits, batch.n_seeds, batch.n_events
    R, cb = S * sides, (4 if wide else 2)
    so = np.asarray(batch.seg_offsets).astype(np.int64)
    seg_len = np.diff(so).reshape(-1, 12, 2).sum(2)          # hits per (event, layer)
    Hx = int(seg_len[:, [0, 3, 4, 7, 8, 11]].sum())          # hits of the six x layers
    offs = batch.seg_offsets.nbytes + batch.seed_offsets.nbytes
    trip = (cb * n_triplets + 1) * R
    acc = 16 * n_acc  # one 16-byte record per candidate that passed the hit-count rule
    # fit (a6 + a7): records, per record its window row and seed parameters, the per-seed track flags; the winners' 80-byte
    # records and the 4-byte track list written and read back by the same CTA (L2-resident in practice), the dense outputs,
    # per event its look-back word (zeroed by the window kernel, written twice, read by later events) and its offset
    return {"window": 4 * H + offs + (16 if sides == 2 else 20) * S + 64 * R + (4 + 8) * E,
            "seed": 4 * Hx + offs + 64 * R + trip + 4 * E,
            "extend": 4 * H + offs + 12 * S + 64 * R + trip + acc + 4 * S + 4 * E,
            "fit": 4 * H + offs + 4 * E + acc + n_acc * (64 + 12) + 4 * S + 2 * 84 * n_tracks + 80 * n_tracks + (8 * 3 + 4) * E}


def tuning_params(args, datagen, cfg):
    """--tuning with-ut: Table 3 "Forward" column (BASELINE.json configs); no-ut: section VI.E."""
    if args.tuning == "no-ut":
        return datagen.no_ut_params()
    return dict(datagen.default_params(), hit_storage=cfg.hit_storage, seed_arith=1 if args.seed_arith == "fp32" else 0)


def oracle_rate(batch, threads: int, geometry, params):
    from oracle import lf_oracle
    t0 = time.perf_counter()
    r = lf_oracle.run(geometry, params, batch, threads=threads)
    dt = time.perf_counter() - t0
    return batch.n_events / dt, dt, r


def run_reference(args):
    """--impl reference: the oracle on the host cores, bounded sample per step."""
    from paper_2402_14670_b200 import datagen, sharding
    rank, _, world = sharding.dist_env()
    if rank != 0:
        return 0
    cfg = datagen.CONFIGS[args.config]
    G, P = datagen.toy_geometry(), tuning_params(args, datagen, cfg)
    cores = os.cpu_count() or 1
    probe = datagen.generate(cfg, n_events=min(200, args.events or cfg.n_events))
    rate, _, _ = oracle_rate(probe, cores, G, P)
    budget = min(0.5, 150.0 / max(args.steps + args.warmup, 1))
    n_sample = int(min(max(rate * budget, 50), 2000, args.events or cfg.n_events))
    batch = datagen.generate(cfg, n_events=n_sample)
    for _ in range(args.warmup):
        oracle_rate(batch, cores, G, P)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_rate(batch, cores, G, P)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = f"first {n_sample} events of {cfg.name} per step (seed {cfg.seed}); oracle sharded over {cores} threads by the harness"
    line = {
        "impl": "reference", "metric": "events_per_s", "value": value, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: Run-3-like occupancy, fp32, {args.tuning} tuning (bounded sample)", "events_per_step": n_sample,
                   "seeds_per_step": batch.n_seeds, "hits_per_step": batch.n_hits},
        "seeds_per_s": batch.n_seeds * args.steps / dt,
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    from paper_2402_14670_b200 import binding, datagen, sharding
    rank, local_rank, world = sharding.dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    # under torchrun (any world size, 1 included) the job runs through torch.distributed: NCCL process group, barrier,
    # max over ranks of the device time
    distributed = world > 1 or ("RANK" in os.environ and "MASTER_ADDR" in os.environ)
    if distributed:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = datagen.CONFIGS[args.config]
    if world > 1:  # weak scaling: every rank gets its own batch of the same recipe
        cfg = datagen.with_overrides(cfg, seed=cfg.seed + 7919 * rank)
    G = datagen.toy_geometry()
    P = tuning_params(args, datagen, cfg)
    no_ut = int(P["mode"]) == 1
    wide = no_ut or int(P["n_window"]) > 32 or int(P["n_triplets"]) > 16
    t_gen = time.perf_counter()
    batch = datagen.generate(cfg, n_events=args.events)
    t_gen = time.perf_counter() - t_gen

    lf = binding.LookingForward(G, P, batch.n_events, batch.n_seeds, batch.n_hits)
    info = lf.info()
    db = binding.DeviceBatch(batch, dev)
    fp16_mode = args.fp16_input if int(P.get("hit_storage", 0)) == 1 else None
    if fp16_mode in ("caller", "only"):
        lf.pack_hits(db)
        if fp16_mode == "only":
            db.drop_fp32()
    out = binding.TrackBuffers(batch.n_seeds, batch.n_events, dev)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if distributed:
            torch.distributed.barrier()

    for _ in range(max(args.warmup, 3)):
        lf.run(db, out, stream)
    barrier()
    n_tracks = int(out.n_tracks.cpu()[0])
    # one counting run (debug build of the kernels, untimed): the work items of every stage, for the algorithmic model
    lf.run_counting(db, out, stream)
    counters = lf.run_counters()
    assert counters["tracks"] == n_tracks, "counting run and plain run disagree on the track count"
    n_acc, n_dup_events = counters["accepted_candidates"], counters["events_with_equal_hits"]
    lf.run(db, out, stream)
    barrier()

    # ---- timed region: K steps, inputs resident in HBM, per-kernel CUDA events recorded by the library
    lf.set_profiling(True)
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # timing rule: the inputs of a step must not be served from L2 left warm by the previous step.  The headline batches are
    # several times the 126 MB L2; a batch that is not (configs 0, 1, 2) is timed step by step with a 256 MB write between steps
    flush_l2 = batch.input_bytes() < 2 * 126e6
    barrier()
    sampler.start()
    if flush_l2:
        scrub = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for a, b in evs:
            scrub.zero_()
            a.record(stream)
            lf.run(db, out, stream)
            b.record(stream)
        barrier()
        clocks = sampler.stop()
        local_ms = sum(a.elapsed_time(b) for a, b in evs)
    else:
        e0.record(stream)
        for _ in range(args.steps):
            lf.run(db, out, stream)
        e1.record(stream)
        barrier()
        clocks = sampler.stop()
        local_ms = e0.elapsed_time(e1)
    ktimes = dict(zip(binding.KERNEL_NAMES, lf.kernel_times()))
    lf.set_profiling(False)
    kernels_per_run = lf.info().kernels_per_run  # what the last timed lf_run enqueued: 4, or 5 when the library packed the fp16 copy
    total_ms, (tot_events, tot_seeds, tot_tracks) = sharding.reduce_job(
        local_ms, [batch.n_events, batch.n_seeds, n_tracks], dev)
    ms_per_step = total_ms / args.steps
    value = tot_events / (ms_per_step * 1e-3)

    # ---- end to end through lf_run_host (pinned host buffers; H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        hb = binding.HostBatch(batch)
        if fp16_mode in ("caller", "only"):
            hb.use_packed(db, keep_fp32=(fp16_mode == "caller"))
        ht = binding.HostTracks(batch.n_seeds, batch.n_events)
        for _ in range(2):
            lf.run_host(hb, ht, stream)
        k_e2e = max(3, min(args.steps, 10))  # the host path is PCIe-bound and steady: ten steps are enough (e2e.steps says so)
        barrier()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            n_host = lf.run_host(hb, ht, stream)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) * 1e3
        assert n_host == n_tracks, "host path and device path disagree on the track count"
        sync_ms, _ = sharding.reduce_job(dt, [0], dev)
        # the same batches as a stream, two in flight (lf_host_submit / lf_host_collect): step i + 1 is copied to the device
        # while step i is computed and copied back.  Every step still moves its inputs from pinned host memory and its
        # tracks back; the timed window runs from the moment step 0 is complete to the moment step k is: k steps, steady state.
        hts = [ht, binding.HostTracks(batch.n_seeds, batch.n_events)]
        barrier()
        lf.host_submit(hb, hts[0], 0, stream)
        t0 = None
        for i in range(1, k_e2e + 2):
            lf.host_submit(hb, hts[i % 2], i % 2, stream)
            lf.host_collect((i - 1) % 2)
            assert int(hts[(i - 1) % 2].n_tracks[0]) == n_tracks, "streamed host path and device path disagree on the track count"
            if i == 1:
                t0 = time.perf_counter()
        dt = (time.perf_counter() - t0) * 1e3
        lf.host_collect((k_e2e + 1) % 2)
        torch.cuda.synchronize()
        e2e_ms, _ = sharding.reduce_job(dt, [0], dev)
        e2e = {"value": tot_events / (e2e_ms / k_e2e * 1e-3), "unit": "events/s", "h2d_bytes_per_step": hb.h2d_bytes(),
               "d2h_bytes_per_step": ht.d2h_bytes(n_tracks), "ms_per_step": e2e_ms / k_e2e, "steps": k_e2e,
               "api": "lf_host_submit / lf_host_collect: a stream of batches from pinned host buffers, two in flight, steady state",
               "one_call_at_a_time": {"value": tot_events / (sync_ms / k_e2e * 1e-3), "ms_per_step": sync_ms / k_e2e,
                                      "api": "lf_run_host (pinned host buffers, synchronous; nothing overlaps between calls)"}}
        del hb, ht, hts

    if rank != 0:
        lf.close()
        if distributed:
            torch.distributed.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (the slowest of the four event kernels): the HBM roofline BASELINE.json's metric
    # names.  The path is bound by instruction issue, not by HBM, so two ALU figures sit beside it
    # as flat keys: alu_algorithmic_frac (a roofline fraction: algorithmic lane-operations of the committed model) and
    # issue_utilisation (how busy the issue slots are with whatever the kernel executes: not a roofline fraction).
    peak, peak_src = measured_peaks()
    sides = 2 if no_ut else 1
    kb = kernel_bytes(batch, n_tracks, int(P["n_triplets"]), n_acc, sides=sides, wide=wide)
    dom = max(binding.EVENT_KERNELS, key=lambda k: ktimes[k])
    # achieved = ALGORITHMIC bytes (inputs read once + tracks written once: ~34.9 KB per event) of the
    # units one launch processes (the whole batch: every kernel is launched once per step on all of it) over the dominant
    # kernel's live duration.  The library's own tables (window rows, triplet codes, candidate records) are not algorithmic
    # bytes; the figure that counts them for the one kernel sits beside it as kernel_table_* (all keys flat).
    path_bytes = algorithmic_bytes(batch, n_tracks)
    achieved = path_bytes / (ktimes[dom] * 1e-3) / 1e9
    step_gbs = path_bytes / (local_ms / args.steps * 1e-3) / 1e9
    table_gbs = kb[dom] / (ktimes[dom] * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": None, "kernel": f"lf_{dom}_kernel", "kernel_ms": ktimes[dom],
                "algorithmic_bytes_per_launch": path_bytes, "algorithmic_bytes_per_event": path_bytes / max(batch.n_events, 1),
                "peak_source": peak_src,
                # the same bytes over the whole step (all four kernels): what the driver-timed ms_per_step implies
                "step_achieved": step_gbs, "step_frac": step_gbs / peak, "step_frac_of_nominal_8TBs": step_gbs / NOMINAL_HBM_GBS,
                # bytes the dominant kernel itself has to touch, its tables included
                "kernel_table_bytes": kb[dom], "kernel_table_achieved": table_gbs, "kernel_table_frac": table_gbs / peak,
                "note": "the path is not HBM-bound (DESIGN.md section 7); frac = SURVEY 8(d) algorithmic bytes of the batch / dominant "
                        "kernel time / measured peak; step_frac = the same bytes / ms_per_step"}
    sm_mhz = float(clocks.get("sm_max_mhz") or 1965.0)
    lane_peak = 148 * 128 * sm_mhz * 1e6
    model = algorithmic_lane_ops(counters, batch, int(P["n_window"]), sides)
    alu_frac = model["total"] / (local_ms / args.steps * 1e-3) / lane_peak
    alu_model = {"lane_ops_per_step": model, "lane_ops_per_seed": model["total"] / max(batch.n_seeds, 1),
                 "peak_lane_ops_per_s": lane_peak, "peak_source": "148 SMs x 128 fp32/int32 lanes x sm_max_mhz",
                 "counters": counters, "coefficients": LANE_OPS,
                 "note": "algorithmic work of the interval-search formulation at 100 % lane use (DESIGN.md section 7), not executed instructions"}
    issue_util, issue_detail = None, None
    tag = ("_noUT" if no_ut else "") + (f"_cfg{args.config}" if args.config != 3 else "")
    traffic_file = os.path.join(ROOT, "profiles", f"dominant_kernel_traffic{tag}.txt")
    if os.path.exists(traffic_file):
        try:
            tr = json.load(open(traffic_file))
            # the ncu counts describe this run only if they were taken on this source and on this batch
            same = (tr.get("source_sha256") == source_sha256() and tr.get("kernel") == roofline["kernel"]
                    and int(tr.get("n_seeds", -1)) == batch.n_seeds)
            if same:
                roofline["traffic"] = tr.get("dram_bytes_per_launch")
                roofline["traffic_source"] = tr.get("source")
                wi = tr.get("all_kernels_warp_inst_per_launch", {})
                if dom in wi:
                    peak_issue = 148 * 4 * sm_mhz * 1e6
                    issue_util = wi[dom] / (ktimes[dom] * 1e-3) / peak_issue
                    ev_k = [k for k in binding.EVENT_KERNELS if k in wi]
                    issue_detail = {"kernel": roofline["kernel"], "warp_inst_per_launch": wi[dom],
                                    "warp_inst_per_seed": wi[dom] / batch.n_seeds,
                                    "all_kernels_warp_inst_per_seed": {k: wi[k] / batch.n_seeds for k in ev_k},
                                    "event_kernels_utilisation": sum(wi[k] for k in ev_k) / (sum(ktimes[k] for k in ev_k) * 1e-3) / peak_issue,
                                    "peak_warp_inst_per_s": peak_issue, "count_source": tr.get("source")}
            else:
                roofline["traffic_note"] = "committed ncu capture was taken on another source or batch (sha256 / n_seeds stamp differs)"
        except Exception:
            pass

    # ---- CPU baseline: the oracle as it stands (single thread), bounded sample; plus an all-cores figure
    cpu = None
    extra = {}
    if world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n1 = min(batch.n_events, args.cpu_events)
        sub = batch.slice_events(0, n1)
        rate1, dt1, ref = oracle_rate(sub, 1, G, P)
        cpu = {"value": rate1, "unit": "events/s", "cores": 1, "kind": "oracle",
               "sample": f"first {n1} events of the same batch, single thread, {dt1:.1f} s"}
        got_prefix = int(out.event_offsets[n1].item())
        extra["oracle_check"] = {"events": n1, "gpu_tracks": got_prefix, "oracle_tracks": int(ref.n_tracks),
                                 "equal": got_prefix == int(ref.n_tracks)}
        nall = min(batch.n_events, args.cpu_events * min(cores, 8))
        rate_all, dt_all, _ = oracle_rate(batch.slice_events(0, nall), cores, G, P)
        extra["cpu_baseline_all_cores"] = {"value": rate_all, "unit": "events/s", "cores": cores, "kind": "oracle",
                                           "sample": f"first {nall} events, harness shards events over {cores} threads, {dt_all:.1f} s"}

    in_bytes = batch.input_bytes()
    line = {
        "metric": "events_per_s", "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: {batch.n_events} events per GPU, {'high' if args.config == 4 else 'Run-3-like'} occupancy, fp32"
                               + ((" with fp16 hit storage, " + args.seed_arith + " seeding") if int(P.get("hit_storage", 0)) == 1 else "")
                               + ", one lf_run on one stream"
                               + (", no-UT tuning (PAPER.md:285-325)" if no_ut else ""),
                   "tuning": args.tuning, "fp16_input": fp16_mode,
                   "events_per_gpu": batch.n_events, "seeds_per_gpu": batch.n_seeds, "hits_per_gpu": batch.n_hits,
                   "tracks_per_step_per_gpu": n_tracks, "accepted_candidates_per_step": n_acc, "events_with_equal_hits": n_dup_events,
                   "l2": (f"flushed: inputs are {in_bytes / 1e6:.0f} MB, so every step is timed on its own after a 256 MB write"
                          if flush_l2 else f"no flush: inputs ({in_bytes / 1e6:.0f} MB) + outputs exceed the 126 MB L2"),
                   "sharding": "events, no data-path collective"},
        "seeds_per_s": tot_seeds / (ms_per_step * 1e-3),
        "tracks_per_s": tot_tracks / (ms_per_step * 1e-3),
        "e2e": e2e, "gpu_launches": kernels_per_run * args.steps,
        "clocks": clocks, "roofline": roofline,
        "alu_algorithmic_frac": alu_frac, "issue_utilisation": issue_util, "alu_model": alu_model, "issue_detail": issue_detail,
        "cpu_baseline": cpu,
        "kernels": {"ms": ktimes, "algorithmic_bytes": kb,
                    "launch": {n: {"regs": info.regs[i], "block": info.block[i], "grid": info.grid[i],
                                   "ctas_per_sm": info.ctas_per_sm[i], "smem_bytes": info.smem_bytes[i]}
                               for i, n in enumerate(binding.EVENT_KERNELS)},
                    "staged_hits_per_event": info.staged_hits_per_event},
        "context": {"paper_hlt1_sequence_khz_a5000": 130, "paper_lf_share": 0.20,
                    "note": "paper numbers are whole-HLT1 on RTX A5000 (PAPER.md:342): context, not a target"},
        "generation_s": t_gen,
    }
    line.update(extra)
    print(json.dumps(line))
    lf.close()
    if distributed:
        torch.distributed.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--tuning", choices=["with-ut", "no-ut"], default="with-ut",
                    help="with-ut: BASELINE.json's headline (default); no-ut: the no-UT tuning of PAPER.md:285-325 on the same events")
    ap.add_argument("--seed-arith", choices=["half2", "fp32"], default="fp32",
                    help="config 2 (fp16 hit storage) only: fp32 = one doublet per lane on the decoded fp16 hits (default, the faster "
                         "one), half2 = pairs of doublets in __half2 (PAPER.md:366; the measured comparison)")
    ap.add_argument("--fp16-input", choices=["library", "caller", "only"], default="library",
                    help="config 2 only: library = lf_run packs the fp32 hits itself (default); caller = the caller hands the packed "
                         "copy next to the fp32 hits; only = the packed copy alone (every stage on fp16: lossy, outside configs[2]'s rule)")
    ap.add_argument("--events", type=int, default=None, help="override the number of events (default: the config's)")
    ap.add_argument("--cpu-events", type=int, default=6000, help="events of the single-thread oracle sample")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":
        return run_reference(args)  # the oracle on the host cores: rank 0 alone works, whatever N is
    if "WORLD_SIZE" in os.environ:   # launched by torchrun: its world size is the number of GPUs
        if int(os.environ["WORLD_SIZE"]) != args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} under a launcher with WORLD_SIZE={os.environ['WORLD_SIZE']}")
        return run_ours(args)
    if args.gpus > 1:
        return launch_ranks(args.gpus)
    return run_ours(args)


def launch_ranks(n: int) -> int:
    """`python bench.py --gpus N` without a launcher: start N ranks (one per GPU) of this same command under
    torch.distributed.run on 127.0.0.1; rank 0 prints the one JSON line with n_gpus = N (each GPU
    its own events, no data-path collective).  Refuses when fewer than N devices are visible instead of timing fewer GPUs
    than the line would claim."""
    import socket
    import subprocess
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < n:
        raise SystemExit(f"bench.py --gpus {n}: only {have} CUDA device(s) visible; one rank per GPU is needed "
                         "(there is no CPU fallback and no oversubscription)")
    with socket.socket(socket.AF_INET, socket.SOCK_STREAM) as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd).returncode


if __name__ == "__main__":
    sys.exit(main())
