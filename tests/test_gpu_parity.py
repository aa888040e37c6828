"""GPU parity: the CUDA path through the C ABI vs the CPU oracle, element by element (-m gpu)."""
import os

import numpy as np
import pytest

from paper_2402_14670_b200 import datagen as dg

from parity import assert_debug_equal, assert_tracks_equal

pytestmark = pytest.mark.gpu
NTHREADS = max(1, (os.cpu_count() or 1))


@pytest.fixture(scope="module")
def lfmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2402_14670_b200 import build as cuda_build
    cuda_build.build()
    from paper_2402_14670_b200 import binding
    binding.load_library()
    return binding


def _gpu_run(binding, G, P, b, debug=False):
    import torch
    lf = binding.LookingForward(G, P, max(b.n_events, 1), max(b.n_seeds, 1), max(b.n_hits, 1))
    out = lf.run(binding.DeviceBatch(b), debug=debug)
    torch.cuda.synchronize()
    got = out.to_numpy()
    if debug:
        got.debug = {k: v.cpu().numpy() for k, v in vars(out.debug_tensors).items()}
    lf.close()
    return got


def test_config0_tracks_and_stage_boundaries(lfmod, oracle, geometry, params):
    b = dg.generate_config(0)
    ref = oracle.run(geometry, params, b, debug=True)
    got = _gpu_run(lfmod, geometry, params, b, debug=True)
    assert_debug_equal(got.debug, ref.debug)
    info = assert_tracks_equal(got, ref, "config 0")
    assert ref.n_tracks > 150
    # the non-debug kernel gives the same result
    got2 = _gpu_run(lfmod, geometry, params, b)
    assert_tracks_equal(got2, ref, "config 0 (release kernel)")
    print("config0", info)


def test_dense_events_stage_boundaries(lfmod, oracle, geometry, params):
    """Window cap and top-n cut bind; both polarities; non-default tunables."""
    cfg = dg.GenConfig("dense", 6, 77, true_fixed=40, fake_mean=8.0, noise_fixed=600, p_min=1.5, smear=0.2)
    b = dg.generate(cfg)
    for G, P in ((geometry, params), (dict(geometry, polarity=-1), params),
                 (dict(geometry, d_ratio=-2.0e-5), dict(params, n_window=9, n_triplets=5, T_x=1.0, T_triplet=4.0)),
                 (geometry, dict(params, n_window=32, n_triplets=16, T_triplet=30.0, min_hits=8))):
        ref = oracle.run(G, P, b, debug=True)
        got = _gpu_run(lfmod, G, P, b, debug=True)
        assert_debug_equal(got.debug, ref.debug)
        assert_tracks_equal(got, ref, "dense")
    assert (ref.debug.n_triplets == 16).sum() > 10


def test_config1_full(lfmod, oracle, geometry, params):
    b = dg.generate_config(1)
    ref = oracle.run(geometry, params, b, threads=NTHREADS)
    got = _gpu_run(lfmod, geometry, params, b)
    print("config1", assert_tracks_equal(got, ref, "config 1"), ref.n_tracks)


def test_config1_stage_boundaries_subset(lfmod, oracle, geometry, params):
    b = dg.generate_config(1, n_events=100)
    ref = oracle.run(geometry, params, b, debug=True, threads=NTHREADS)
    got = _gpu_run(lfmod, geometry, params, b, debug=True)
    assert_debug_equal(got.debug, ref.debug)
    assert_tracks_equal(got, ref, "config 1 subset")


def test_config4_full(lfmod, oracle, geometry, params):
    b = dg.generate_config(4)
    ref = oracle.run(geometry, params, b, threads=NTHREADS)
    got = _gpu_run(lfmod, geometry, params, b)
    print("config4", assert_tracks_equal(got, ref, "config 4"), ref.n_tracks)


def test_config3_full_size(lfmod, oracle, geometry, params):
    """BASELINE.json configs[3]: 20,000 events in one lf_run, the launch configuration bench.py times."""
    b = dg.generate_config(3)
    got = _gpu_run(lfmod, geometry, params, b)
    ref = oracle.run(geometry, params, b, threads=NTHREADS)
    print("config3", assert_tracks_equal(got, ref, "config 3"), ref.n_tracks)


def test_deterministic(lfmod, geometry, params):
    b = dg.generate_config(1, n_events=300)
    a = _gpu_run(lfmod, geometry, params, b)
    c = _gpu_run(lfmod, geometry, params, b)
    for k in ("hit_idx", "seed_idx", "n_hits", "event_offsets"):
        assert np.array_equal(getattr(a, k), getattr(c, k))
    assert np.array_equal(a.state.view(np.uint32), c.state.view(np.uint32))
    assert np.array_equal(a.quality.view(np.uint32), c.quality.view(np.uint32))


def test_edge_cases(lfmod, oracle, geometry, params):
    import torch
    # zero events
    empty = dg.generate(dg.GenConfig("e", 0, 1))
    got = _gpu_run(lfmod, geometry, params, empty)
    assert got.n_tracks == 0 and got.event_offsets.tolist() == [0]
    # events without seeds; events without hits; a mix of empty and full events
    noseed = dg.generate(dg.GenConfig("ns", 3, 2, true_fixed=0, noise_fixed=50))
    got = _gpu_run(lfmod, geometry, params, noseed)
    assert got.n_tracks == 0 and got.event_offsets.tolist() == [0, 0, 0, 0]
    b = dg.generate_config(0)
    nohits = dg.Batch(**{**b.__dict__, "hit_x": np.zeros(0, np.float32),
                        "seg_offsets": np.zeros(b.n_events * 24 + 1, np.uint32), "hit_track": np.zeros(0, np.int32)})
    got = _gpu_run(lfmod, geometry, params, nohits)
    assert got.n_tracks == 0
    # one hit per segment, duplicates of one x value in every segment
    one = dg.Batch(**{**b.__dict__})
    one.hit_x = np.full(b.n_events * 24 * 3, 12.5, np.float32)
    one.seg_offsets = (np.arange(b.n_events * 24 + 1) * 3).astype(np.uint32)
    one.hit_track = np.full(one.hit_x.shape[0], -1, np.int32)
    ref = oracle.run(geometry, params, one, debug=True)
    got = _gpu_run(lfmod, geometry, params, one, debug=True)
    assert_debug_equal(got.debug, ref.debug)
    assert_tracks_equal(got, ref, "duplicates")


def test_unaligned_event_starts_and_misaligned_base(lfmod, oracle, geometry, params):
    """Event hit blocks start at arbitrary 4-byte offsets; also a hit array whose base is not 16-byte aligned."""
    import torch
    b = dg.generate_config(1, n_events=40)
    ref = oracle.run(geometry, params, b)
    lf = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, b.n_hits + 8)
    for shift in (0, 1, 2, 3):
        db = lfmod.DeviceBatch(b)
        big = torch.zeros(b.n_hits + 8, dtype=torch.float32, device=db.device)
        big[shift:shift + b.n_hits] = db.hit_x
        db.hit_x = big[shift:shift + b.n_hits]
        out = lf.run(db)
        torch.cuda.synchronize()
        assert_tracks_equal(out.to_numpy(), ref, f"base shift {shift}")
    lf.close()


def test_event_larger_than_stage_buffer(lfmod, oracle, geometry, params):
    """An event with more hits than the shared-memory stage holds takes the global-memory path."""
    cfg = dg.GenConfig("huge", 3, 9, true_fixed=60, fake_mean=5.0, noise_fixed=1700)
    b = dg.generate(cfg)
    import torch
    lf = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, b.n_hits)
    assert b.n_hits / b.n_events > lf.info().staged_hits_per_event
    out = lf.run(lfmod.DeviceBatch(b), debug=True)
    torch.cuda.synchronize()
    got = out.to_numpy()
    got.debug = {k: v.cpu().numpy() for k, v in vars(out.debug_tensors).items()}
    ref = oracle.run(geometry, params, b, debug=True)
    assert_debug_equal(got.debug, ref.debug)
    assert_tracks_equal(got, ref, "huge events")
    lf.close()


def test_run_host_matches_device_path(lfmod, oracle, geometry, params):
    b = dg.generate_config(1, n_events=200)
    ref = oracle.run(geometry, params, b, threads=NTHREADS)
    lf = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, b.n_hits)
    hb = lfmod.HostBatch(b)
    ht = lfmod.HostTracks(b.n_seeds, b.n_events)
    for _ in range(2):
        n = lf.run_host(hb, ht)
        assert n == ref.n_tracks
        assert_tracks_equal(ht.to_numpy(), ref, "host path")
    # the chunked pipeline (H2D / kernels / D2H overlapped) gives the same dense output for any chunking,
    # with pinned and with pageable host memory
    for chunk, pin in ((7, True), (16, True), (64, False), (199, True)):
        lf.set_host_chunk_events(chunk)
        hb2, ht2 = lfmod.HostBatch(b, pin=pin), lfmod.HostTracks(b.n_seeds, b.n_events, pin=pin)
        assert lf.run_host(hb2, ht2) == ref.n_tracks
        assert_tracks_equal(ht2.to_numpy(), ref, f"host path, chunks of >= {chunk} events")
    lf.close()
    # fp16 hit storage goes through the same pipeline: chunked == unchunked
    P16 = dict(params, hit_storage=1)
    lf = lfmod.LookingForward(geometry, P16, b.n_events, b.n_seeds, b.n_hits)
    ht_a, ht_b = lfmod.HostTracks(b.n_seeds, b.n_events), lfmod.HostTracks(b.n_seeds, b.n_events)
    lf.run_host(hb, ht_a)
    lf.set_host_chunk_events(13)
    lf.run_host(hb, ht_b)
    a, c = ht_a.to_numpy(), ht_b.to_numpy()
    assert a.n_tracks == c.n_tracks and np.array_equal(a.hit_idx, c.hit_idx) and np.array_equal(a.event_offsets, c.event_offsets)
    assert np.array_equal(a.state.view(np.uint32), c.state.view(np.uint32))
    lf.close()


def test_repeated_runs_and_capacity_errors(lfmod, geometry, params):
    import torch
    b = dg.generate_config(1, n_events=50)
    lf = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, b.n_hits)
    db = lfmod.DeviceBatch(b)
    out = lfmod.TrackBuffers(b.n_seeds, b.n_events, db.device)
    first = None
    for _ in range(5):
        lf.run(db, out)
        torch.cuda.synchronize()
        r = out.to_numpy()
        if first is None:
            first = r
        assert r.n_tracks == first.n_tracks and np.array_equal(r.hit_idx, first.hit_idx)
    small = lfmod.TrackBuffers(b.n_seeds - 1, b.n_events, db.device)
    with pytest.raises(lfmod.LfError) as ei:
        lf.run(db, small)
    assert ei.value.status == lfmod.LF_ERR_CAPACITY
    lf.close()
    lf2 = lfmod.LookingForward(geometry, params, 10, 10, 10)
    with pytest.raises(lfmod.LfError) as ei:
        lf2.run(db, out)
    assert ei.value.status == lfmod.LF_ERR_CAPACITY
    lf2.close()


@pytest.mark.parametrize("seed_arith", [0, 1])
def test_config2_fp16_hit_storage(lfmod, oracle, geometry, params, seed_arith):
    """BASELINE.json configs[2]: fp16 storage of the hits for windows + seeding, fp32 extension and fit.  seed_arith 0 is
    the half2 seeding kernel (pairs of doublets in __half2), 1 the fp32 arithmetic on the decoded fp16 hits.
    Rule: >= 99.5 % of the fp32 oracle's tracks reproduced with identical hit lists, and the truth-matched
    efficiency within 0.2 % absolute."""
    from paper_2402_14670_b200 import truth
    b = dg.generate_config(2)
    assert dg.CONFIGS[2].hit_storage == 1
    P16 = dict(params, hit_storage=1, seed_arith=seed_arith)
    ref = oracle.run(geometry, params, b, threads=NTHREADS)
    got = _gpu_run(lfmod, geometry, P16, b)
    common, ig, ir = np.intersect1d(got.seed_idx, ref.seed_idx, return_indices=True)
    same = (got.hit_idx[ig] == ref.hit_idx[ir]).all(1)
    frac = same.sum() / ref.n_tracks
    e_got = truth.evaluate(b, got.hit_idx, got.n_hits)
    e_ref = truth.evaluate(b, ref.hit_idx, ref.n_hits)
    print(f"config2 fp16 (seed_arith {seed_arith}): identical hit lists {frac:.5f} of {ref.n_tracks}; tracks {got.n_tracks}; "
          f"eff {e_got.efficiency:.5f} vs {e_ref.efficiency:.5f}; ghost {e_got.ghost_rate:.5f} vs {e_ref.ghost_rate:.5f}")
    assert frac >= 0.995
    assert abs(e_got.efficiency - e_ref.efficiency) <= 0.002
    # identical hit lists went through the fp32 fit; the winning triplet (the fit's expansion point) may
    # differ, so states agree to fp32 rounding noise (cf. test_f32_build_matches_f64_build), not bitwise
    d = np.abs(got.state[ig][same].astype(np.float64) - ref.state[ir][same].astype(np.float64))
    assert d[:, 0].max() <= 2e-3 and d[:, 1].max() <= 2e-2 and d[:, 2].max() <= 3e-6 and d[:, 3].max() <= 3e-5
    # the fp16 path is deterministic too
    got2 = _gpu_run(lfmod, geometry, P16, b)
    assert np.array_equal(got.hit_idx, got2.hit_idx) and np.array_equal(got.state.view(np.uint32), got2.state.view(np.uint32))
    # the stage-boundary tables of the seeding kernel stay consistent in the half2 build: kept triplets are ordered by
    # chi2, below the cut, and made of hits inside the seed's windows
    dbg = _gpu_run(lfmod, geometry, P16, dg.generate_config(2, n_events=40), debug=True).debug
    nt, c = dbg["n_triplets"], dbg["trip_chi2"]
    for k in range(params["n_triplets"] - 1):
        both = nt > k + 1
        assert np.all(c[both, k] <= c[both, k + 1])
    assert np.all(c[c >= 0] < params["T_triplet"]) and np.all(nt <= params["n_triplets"])
    for i, l in ((0, (0, 3)), (1, (4, 7)), (2, (8, 11))):
        h = dbg["trip_hits"][:, :, i]
        st = dbg["trip_set"]
        for s_, layer in enumerate(l):
            m = (st == s_) & (h >= 0)
            wf = np.broadcast_to(dbg["win_first"][:, layer][:, None], h.shape)[m]
            wc = np.broadcast_to(dbg["win_count"][:, layer][:, None], h.shape)[m]
            assert np.all(h[m] >= wf) and np.all(h[m] < wf + wc)


def test_validate_inputs(lfmod, geometry, params):
    """lf_validate_inputs: the preconditions lf_run relies on, checked on the device."""
    import torch
    b = dg.generate_config(1, n_events=20)
    lf = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, b.n_hits)
    lf.validate_inputs(lfmod.DeviceBatch(b))                                   # a generated batch is valid
    lf.validate_inputs(lfmod.DeviceBatch(dg.generate(dg.GenConfig("e", 0, 1))))  # so is an empty one

    def expect(batch, word, handle=lf):
        with pytest.raises(lfmod.LfError) as ei:
            handle.validate_inputs(lfmod.DeviceBatch(batch))
        assert ei.value.status == lfmod.LF_ERR_INVALID_ARG and word in str(ei.value), str(ei.value)

    hx = b.hit_x.copy()
    s0 = int(b.seg_offsets[5])
    hx[s0], hx[s0 + 1] = hx[s0 + 1] + 1.0, hx[s0]
    expect(dg.Batch(**{**b.__dict__, "hit_x": hx}), "not ascending")
    hx = b.hit_x.copy()
    hx[7] = np.inf
    expect(dg.Batch(**{**b.__dict__, "hit_x": hx}), "non-finite hit")
    so = b.seg_offsets.copy()
    so[10], so[11] = so[11], so[10] + (1 if so[10] == so[11] else 0)
    expect(dg.Batch(**{**b.__dict__, "seg_offsets": so}), "seg_offsets")
    eo = b.seed_offsets.copy()
    eo[3] = eo[4] + 1
    expect(dg.Batch(**{**b.__dict__, "seed_offsets": eo}), "seed event_offsets")
    q = b.seed_qop.copy()
    q[11] = np.nan
    bad_q = dg.Batch(**{**b.__dict__, "seed_qop": q})
    expect(bad_q, "non-finite seed")
    lf.close()
    # q/p is not an input of the no-UT mode
    lf1 = lfmod.LookingForward(geometry, dg.no_ut_params(), b.n_events, b.n_seeds, b.n_hits)
    lf1.validate_inputs(lfmod.DeviceBatch(bad_q))
    tx = b.seed_tx.copy()
    tx[0] = np.nan
    expect(dg.Batch(**{**b.__dict__, "seed_tx": tx}), "non-finite seed", lf1)
    lf1.close()


def test_lf_run_is_graph_capturable(lfmod, oracle, geometry, params):
    """lf_run only enqueues kernels on the caller's stream (no sync, no allocation): it can be captured into a CUDA
    graph and replayed, e.g. for small launch-bound batches."""
    import torch
    b = dg.generate_config(1, n_events=64)
    ref = oracle.run(geometry, params, b, threads=NTHREADS)
    lf = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, b.n_hits)
    db = lfmod.DeviceBatch(b)
    out = lfmod.TrackBuffers(b.n_seeds, b.n_events, db.device)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        lf.run(db, out, side)            # warm-up outside the capture
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            lf.run(db, out, side)
    for _ in range(3):
        out.hit_idx.fill_(-7)
        out.n_tracks.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert_tracks_equal(out.to_numpy(), ref, "graph replay")
    # launch-bound regime: replaying the graph is not slower than four separate launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    st = torch.cuda.current_stream()
    for _ in range(5):
        g.replay()
    e0.record(st)
    for _ in range(50):
        g.replay()
    e1.record(st)
    torch.cuda.synchronize()
    t_graph = e0.elapsed_time(e1) / 50
    e0.record(st)
    for _ in range(50):
        lf.run(db, out, st)
    e1.record(st)
    torch.cuda.synchronize()
    t_plain = e0.elapsed_time(e1) / 50
    print(f"64 events: graph replay {t_graph * 1e3:.1f} us, plain launches {t_plain * 1e3:.1f} us")
    lf.close()


def test_garbage_inputs_are_memory_safe(lfmod, geometry, params):
    """Unsorted hits, NaN / inf / huge values in hits and seeds: the preconditions are violated, so the result is
    unspecified - but every index stays in range, the offsets are consistent and nothing hangs (searches are bounded
    by the segment and window limits whatever the comparisons return)."""
    import torch
    rng = np.random.default_rng(5)
    for P in (params, dg.no_ut_params(), dict(params, n_window=64, n_triplets=32)):
        b = dg.generate_config(1, n_events=30)
        hx = rng.uniform(-4000, 4000, b.n_hits).astype(np.float32)
        hx[rng.integers(0, b.n_hits, 200)] = np.nan
        hx[rng.integers(0, b.n_hits, 200)] = np.inf

        def junk(a):
            a = a.copy()
            idx = rng.integers(0, a.shape[0], a.shape[0] // 5)
            a[idx] = rng.choice([np.nan, np.inf, -np.inf, 1e30, -1e30, 0.0], idx.shape[0]).astype(np.float32)
            return a
        bb = dg.Batch(**{**b.__dict__, "hit_x": hx, "seed_x": junk(b.seed_x), "seed_y": junk(b.seed_y),
                         "seed_tx": junk(b.seed_tx), "seed_ty": junk(b.seed_ty), "seed_qop": junk(b.seed_qop)})
        lf = lfmod.LookingForward(geometry, P, bb.n_events, bb.n_seeds, bb.n_hits)
        with pytest.raises(lfmod.LfError):
            lf.validate_inputs(lfmod.DeviceBatch(bb))
        for debug in (False, True):
            out = lf.run(lfmod.DeviceBatch(bb), debug=debug)
            torch.cuda.synchronize()
            r = out.to_numpy()
            assert 0 <= r.n_tracks <= bb.n_seeds
            assert np.all(np.diff(r.event_offsets.astype(np.int64)) >= 0) and r.event_offsets[-1] == r.n_tracks
            if r.n_tracks:
                assert r.hit_idx.min() >= -1 and r.hit_idx.max() < bb.n_hits
                assert r.seed_idx.min() >= 0 and r.seed_idx.max() < bb.n_seeds
        lf.close()


def test_two_live_handles_of_different_size(lfmod, oracle, geometry, params):
    """The dynamic shared-memory limit is an attribute of the kernel function, not of a handle: creating a handle with a
    smaller stage (or fewer triplets) after a large one must not break the large one."""
    import torch
    big = dg.generate_config(4, n_events=12)        # ~12 000 hits per event: the largest stage
    small = dg.generate_config(0)
    lf_big = lfmod.LookingForward(geometry, params, big.n_events, big.n_seeds, big.n_hits)
    assert max(lf_big.info().smem_bytes) > 48 * 1024
    lf_small = lfmod.LookingForward(geometry, dict(params, n_triplets=4), small.n_events, small.n_seeds, small.n_hits)
    assert max(lf_small.info().smem_bytes) < max(lf_big.info().smem_bytes)
    out_small = lf_small.run(lfmod.DeviceBatch(small))
    out_big = lf_big.run(lfmod.DeviceBatch(big))    # needs the larger limit that lf_small's creation must not have lowered
    torch.cuda.synchronize()
    assert_tracks_equal(out_big.to_numpy(), oracle.run(geometry, params, big), "big handle after a small lf_create")
    assert_tracks_equal(out_small.to_numpy(), oracle.run(geometry, dict(params, n_triplets=4), small), "small handle")
    lf_small.close()
    lf_big.close()


def test_reversed_field(lfmod, oracle, params):
    """kick < 0 with polarity -1 (C7): the same-bend filter follows the sign of kick * q/p."""
    G = dg.toy_geometry(polarity=-1, kick_sign=-1.0)
    cfg = dg.with_overrides(dg.CONFIGS[1], kick_sign=-1.0, p_min=1.5)
    b = dg.generate(cfg, n_events=40)
    ref = oracle.run(G, params, b, debug=True)
    assert ref.n_tracks > 0.7 * (b.seed_track >= 0).sum()
    got = _gpu_run(lfmod, G, params, b, debug=True)
    assert_tracks_equal(got, ref, "reversed field")
    assert_debug_equal(got.debug, ref.debug)


def _rule_config2(b, got, ref, what, min_same=0.995):
    """BASELINE.json configs[2] rule: >= 99.5 % identical hit lists, truth-matched efficiency within 0.2 % absolute."""
    from paper_2402_14670_b200 import truth
    common, ig, ir = np.intersect1d(got.seed_idx, ref.seed_idx, return_indices=True)
    same = (got.hit_idx[ig] == ref.hit_idx[ir]).all(1)
    frac = same.sum() / ref.n_tracks
    e_got, e_ref = truth.evaluate(b, got.hit_idx, got.n_hits), truth.evaluate(b, ref.hit_idx, ref.n_hits)
    print(f"{what}: identical hit lists {frac:.5f} of {ref.n_tracks}; eff {e_got.efficiency:.5f} vs {e_ref.efficiency:.5f}")
    assert frac >= min_same and abs(e_got.efficiency - e_ref.efficiency) <= 0.002
    return frac


def test_config2_packed_input_and_fp16_only(lfmod, oracle, geometry, params):
    """hit_storage = 1 with the caller's packed copy (lf_pack_hits): identical to the library packing it, and within the
    configs[2] rule.  With the fp32 hits dropped every stage reads the fp16 copy (2.5 bytes per hit instead of 4; only the
    packed copy crosses PCIe in lf_run_host): a LOSSY mode outside the configs[2] rule, because extension and fit then
    see the fp16 rounding (<= 0.03 mm typically) next to a 0.08 mm resolution: the efficiency is unchanged but only about
    98.5 % of the hit lists stay identical."""
    import torch
    b = dg.generate_config(2)
    P16 = dict(params, hit_storage=1)
    ref = oracle.run(geometry, params, b, threads=NTHREADS)
    lf = lfmod.LookingForward(geometry, P16, b.n_events, b.n_seeds, b.n_hits)
    db = lfmod.DeviceBatch(b)
    a = lf.run(db)
    torch.cuda.synchronize()
    a = a.to_numpy()
    assert lf.info().kernels_per_run == 5       # the library packed the fp16 copy itself: one more kernel
    lf.pack_hits(db)
    # the packed copy follows the documented encoding: hit = origin(block) + half; the error is half an fp16 ulp of the
    # offset to the block origin (<= 0.125 mm for offsets below 512 mm, <= 0.25 mm below 1024 mm)
    x16, org = db.hit_x16.cpu().numpy().astype(np.float32), db.origin16.cpu().numpy()
    S = np.repeat(b.seg_offsets[:-1].astype(np.int64), np.diff(b.seg_offsets.astype(np.int64)))
    g = np.repeat(np.arange(b.n_events * 24), np.diff(b.seg_offsets.astype(np.int64)))
    i = np.arange(b.n_hits) - S
    dec = org[(S >> 3) + g + (i >> 3)] + x16
    err = np.abs(dec - b.hit_x)
    assert err.max() <= 1.0 and np.percentile(err, 99) <= 0.26 and np.median(err) <= 0.07
    c = lf.run(db)          # x and x16 given: windows + seeding on the caller's copy, extension + fit on fp32
    torch.cuda.synchronize()
    c = c.to_numpy()
    assert lf.info().kernels_per_run == 4       # the caller's copy: nothing to pack (lf_get_info reports the last launch)
    assert c.n_tracks == a.n_tracks and np.array_equal(c.hit_idx, a.hit_idx) and np.array_equal(c.state.view(np.uint32), a.state.view(np.uint32))
    _rule_config2(b, c, ref, "fp16 windows+seeding, fp32 extension+fit")
    db.drop_fp32()          # fp16 only
    # lf_validate_inputs checks the fp16-only input as the kernels decode it: finite, ascending inside every block of 8
    lf.validate_inputs(db)
    s0 = int(b.seg_offsets[7])
    assert int(b.seg_offsets[8]) - s0 >= 8
    keep16, keep_org = db.hit_x16.clone(), db.origin16.clone()
    db.hit_x16[s0 + 1], db.hit_x16[s0 + 2] = keep16[s0 + 2] + 1.0, keep16[s0 + 1]
    with pytest.raises(lfmod.LfError) as ei:
        lf.validate_inputs(db)
    assert "not ascending" in str(ei.value) and f"hit {s0 + 1})" in str(ei.value), str(ei.value)
    db.hit_x16.copy_(keep16)
    db.origin16[(s0 >> 3) + 7] = float("inf")
    with pytest.raises(lfmod.LfError) as ei:
        lf.validate_inputs(db)
    assert "non-finite hit" in str(ei.value), str(ei.value)
    db.origin16.copy_(keep_org)
    lf.validate_inputs(db)
    d = lf.run(db)
    torch.cuda.synchronize()
    d = d.to_numpy()
    _rule_config2(b, d, ref, "fp16 everywhere (lossy, outside the rule)", min_same=0.98)
    hb = lfmod.HostBatch(b).use_packed(db)
    assert hb.hit_x is None and hb.h2d_bytes() < 0.75 * lfmod.HostBatch(b, pin=False).h2d_bytes()
    ht = lfmod.HostTracks(b.n_seeds, b.n_events)
    lf.set_host_chunk_events(64)
    assert lf.run_host(hb, ht) == d.n_tracks
    e = ht.to_numpy()
    assert np.array_equal(e.hit_idx, d.hit_idx) and np.array_equal(e.state.view(np.uint32), d.state.view(np.uint32))
    lf.close()


def test_fp16_only_events_larger_than_the_stage(lfmod, oracle, geometry, params):
    """fp16-only input with events that do not fit the shared-memory stage: the window kernel decodes them once into the
    library's fp32 scratch image; the result equals the staged decoding of the same packed hits."""
    import torch
    cfg = dg.GenConfig("huge16", 6, 19, true_fixed=60, fake_mean=5.0, noise_fixed=1000)
    b = dg.generate(cfg)
    P16 = dict(params, hit_storage=1)
    small = lfmod.LookingForward(geometry, P16, b.n_events, b.n_seeds, b.n_hits)              # stage sized for these events
    tiny = lfmod.LookingForward(geometry, P16, 100 * b.n_events, b.n_seeds, b.n_hits)         # 2 048-hit stage: all oversize
    assert b.n_hits / b.n_events <= small.info().staged_hits_per_event
    assert np.diff(b.seg_offsets[::24].astype(np.int64)).min() > tiny.info().staged_hits_per_event
    db = lfmod.DeviceBatch(b)
    small.pack_hits(db)
    db.drop_fp32()
    r1 = small.run(db)
    r2 = tiny.run(db)
    torch.cuda.synchronize()
    r1, r2 = r1.to_numpy(), r2.to_numpy()
    assert r1.n_tracks == r2.n_tracks > 100 and np.array_equal(r1.hit_idx, r2.hit_idx)
    assert np.array_equal(r1.state.view(np.uint32), r2.state.view(np.uint32))
    ref = oracle.run(geometry, params, b)
    common, ig, ir = np.intersect1d(r2.seed_idx, ref.seed_idx, return_indices=True)
    assert ((r2.hit_idx[ig] == ref.hit_idx[ir]).all(1).sum() / ref.n_tracks) > 0.95  # fp16 everywhere is lossy
    small.close()
    tiny.close()


def _thin_uv_layers(b, keep=0.12, seed=5):
    """The same batch with most noise hits of the u/v layers dropped (true hits stay), so that the x layers hold well over
    half of an event's hits: the seeding kernel's half-size x-layer stage overflows while the full-event stage of the other
    kernels does not."""
    from dataclasses import replace
    rng = np.random.default_rng(seed)
    so = b.seg_offsets.astype(np.int64)
    seg_of_hit = np.repeat(np.arange(so.size - 1), np.diff(so))
    layer = (seg_of_hit % 24) // 2
    uv = ((layer % 4) == 1) | ((layer % 4) == 2)
    keep_mask = ~uv | (b.hit_track >= 0) | (rng.uniform(size=b.n_hits) < keep)
    new_so = np.concatenate([[0], np.cumsum(np.bincount(seg_of_hit[keep_mask], minlength=so.size - 1))]).astype(np.uint32)
    return replace(b, hit_x=b.hit_x[keep_mask], hit_track=b.hit_track[keep_mask], seg_offsets=new_so)


def test_x_layer_stage_overflow(lfmod, oracle, geometry, params):
    """Events that fit the full-event stage of the window, extension and fit kernels but whose x layers overflow the seeding
    kernel's half-size stage: fp32 hits are then read from global memory by that kernel alone (bit-identical to the oracle),
    fp16-only hits from the scratch image the window kernel decodes for exactly these events (identical to the staged
    decoding of the same packed hits)."""
    import torch
    b = _thin_uv_layers(dg.generate(dg.GenConfig("xheavy", 8, 23, true_fixed=40, fake_mean=4.0, noise_fixed=500)))
    nx = [int(sum(b.seg_offsets[e * 24 + 2 * l + 2] - b.seg_offsets[e * 24 + 2 * l] for l in (0, 3, 4, 7, 8, 11))) for e in range(b.n_events)]
    nh = np.diff(b.seg_offsets[::24].astype(np.int64))
    assert min(nx) > 0.7 * nh.max()
    roomy = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, 3 * b.n_hits)      # both stages hold the events
    tight = lfmod.LookingForward(geometry, params, b.n_events, b.n_seeds, b.n_hits)          # only the full-event stage does
    cap = tight.info().staged_hits_per_event
    assert nh.max() <= cap and min(nx) + 28 > cap // 2 + 256 + 256, (nh.max(), min(nx), cap)
    ref = oracle.run(geometry, params, b, debug=True)
    for lf in (roomy, tight):
        out = lf.run(lfmod.DeviceBatch(b), debug=True)
        torch.cuda.synchronize()
        got = out.to_numpy()
        got.debug = {k: v.cpu().numpy() for k, v in vars(out.debug_tensors).items()}
        assert_debug_equal(got.debug, ref.debug)
        assert_tracks_equal(got, ref, "x-heavy events")
        lf.close()
    P16 = dict(params, hit_storage=1, seed_arith=1)
    roomy = lfmod.LookingForward(geometry, P16, b.n_events, b.n_seeds, 3 * b.n_hits)
    tight = lfmod.LookingForward(geometry, P16, b.n_events, b.n_seeds, b.n_hits)
    db = lfmod.DeviceBatch(b)
    roomy.pack_hits(db)
    db.drop_fp32()
    r1, r2 = roomy.run(db), tight.run(db)
    torch.cuda.synchronize()
    r1, r2 = r1.to_numpy(), r2.to_numpy()
    assert r1.n_tracks == r2.n_tracks > 50 and np.array_equal(r1.hit_idx, r2.hit_idx)
    assert np.array_equal(r1.state.view(np.uint32), r2.state.view(np.uint32))
    roomy.close()
    tight.close()


def _drop_seeds(b, keep_event):
    """The same hits, but only the events with keep_event[e] keep their seeds."""
    counts = np.diff(b.seed_offsets.astype(np.int64))
    ev_of_seed = np.repeat(np.arange(b.n_events), counts)
    sel = keep_event[ev_of_seed]
    new_counts = np.where(keep_event, counts, 0)
    off = np.zeros(b.n_events + 1, np.uint32)
    off[1:] = np.cumsum(new_counts).astype(np.uint32)
    return dg.Batch(**{**b.__dict__, "seed_x": b.seed_x[sel], "seed_y": b.seed_y[sel], "seed_tx": b.seed_tx[sel],
                       "seed_ty": b.seed_ty[sel], "seed_qop": b.seed_qop[sel], "seed_track": b.seed_track[sel],
                       "seed_offsets": off})


def test_stream_compaction_lookback_stress(lfmod, oracle, geometry, params):
    """a7 inside the fit kernel (decoupled look-back over the events' track counts): batches that
    stress the scan rather than the arithmetic.  (1) 40 000 tiny events, most of them without a track, far more events than
    resident CTAs; (2) full events alternating with seedless ones in runs of irregular length, so that CTAs finish their
    events in an order far from the event order; (3) two handles running on two streams at the same time; (4) events with
    more tracks than the shared-memory track list holds; (5) the tiny events through lf_run_host, whose chunks are separate
    launches."""
    import torch
    tiny = dg.generate(dg.GenConfig("tiny_events", 40000, 77, true_mean=1.2, fake_mean=0.3, noise_mean=6.0))
    ref = oracle.run(geometry, params, tiny, threads=NTHREADS)
    assert 0 < ref.n_tracks and (np.diff(ref.event_offsets) == 0).mean() > 0.2
    for rep in range(2):
        assert_tracks_equal(_gpu_run(lfmod, geometry, params, tiny), ref, "40 000 tiny events")
    b = dg.generate_config(1, n_events=600)
    rng = np.random.default_rng(5)
    keep = np.zeros(b.n_events, bool)
    e = 0
    while e < b.n_events:  # runs of 1..40 kept events, then 1..120 seedless ones
        n_keep = int(rng.integers(1, 41))
        keep[e:e + n_keep] = True
        e += n_keep + int(rng.integers(1, 121))
    mixed = _drop_seeds(b, keep)
    ref_m = oracle.run(geometry, params, mixed, threads=NTHREADS)
    assert ref_m.n_tracks > 1000
    assert_tracks_equal(_gpu_run(lfmod, geometry, params, mixed), ref_m, "full and seedless events mixed")
    # two handles, two streams, in flight together; repeated so that the launches really overlap
    lf1 = lfmod.LookingForward(geometry, params, tiny.n_events, tiny.n_seeds, tiny.n_hits)
    lf2 = lfmod.LookingForward(geometry, params, mixed.n_events, mixed.n_seeds, mixed.n_hits)
    d1, d2 = lfmod.DeviceBatch(tiny), lfmod.DeviceBatch(mixed)
    o1 = lfmod.TrackBuffers(tiny.n_seeds, tiny.n_events, d1.device)
    o2 = lfmod.TrackBuffers(mixed.n_seeds, mixed.n_events, d2.device)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(5):
        lf1.run(d1, o1, s1)
        lf2.run(d2, o2, s2)
    torch.cuda.synchronize()
    assert_tracks_equal(o1.to_numpy(), ref, "two handles in flight (tiny events)")
    assert_tracks_equal(o2.to_numpy(), ref_m, "two handles in flight (mixed events)")
    lf1.close()
    lf2.close()
    # events with more tracks than the shared-memory track list holds (384): the copy-out reads the global list
    big = dg.generate(dg.GenConfig("big_events", 24, 78, true_mean=700.0, fake_mean=50.0, noise_mean=100.0))
    ref_b = oracle.run(geometry, params, big, threads=NTHREADS)
    assert np.diff(ref_b.event_offsets).min() > 384
    assert_tracks_equal(_gpu_run(lfmod, geometry, params, big), ref_b, "events with more than 384 tracks")
    # the host path: chunks are separate launches, each with its own look-back
    lf = lfmod.LookingForward(geometry, params, tiny.n_events, tiny.n_seeds, tiny.n_hits)
    lf.set_host_chunk_events(1500)
    ht = lfmod.HostTracks(tiny.n_seeds, tiny.n_events)
    lf.run_host(lfmod.HostBatch(tiny), ht)
    assert_tracks_equal(ht.to_numpy(), ref, "tiny events through lf_run_host")
    lf.close()


def test_host_submit_collect_pipeline(lfmod, oracle, geometry, params):
    """lf_host_submit / lf_host_collect (include/lf.h): a stream of different batches, two in flight, gives for every batch
    exactly what lf_run_host gives (= the oracle's tracks); misuse is refused before anything is enqueued."""
    import torch
    whole = dg.generate_config(1, n_events=900)
    cuts = [0, 260, 300, 610, 611, 900]  # batches of different sizes, one of them a single event
    batches = [whole.slice_events(a, b) for a, b in zip(cuts[:-1], cuts[1:])] + [dg.generate(dg.GenConfig("e", 0, 1))]
    refs = [oracle.run(geometry, params, b, threads=NTHREADS) for b in batches]
    lf = lfmod.LookingForward(geometry, params, max(b.n_events for b in batches), max(b.n_seeds for b in batches),
                              max(b.n_hits for b in batches))
    lf.set_host_chunk_events(64)
    hbs = [lfmod.HostBatch(b) for b in batches]
    hts = [lfmod.HostTracks(max(b.n_seeds, 1), b.n_events) for b in batches]
    st = torch.cuda.Stream()
    for rep in range(2):
        for t in hts:
            t.hit_idx.fill_(-7)
            t.n_tracks.zero_()
        lf.host_submit(hbs[0], hts[0], 0, st)
        for i in range(1, len(batches)):
            lf.host_submit(hbs[i], hts[i], i % 2, st)
            lf.host_collect((i - 1) % 2)
            assert_tracks_equal(hts[i - 1].to_numpy(), refs[i - 1], f"pipelined batch {i - 1}")
        lf.host_collect((len(batches) - 1) % 2)
        assert_tracks_equal(hts[-1].to_numpy(), refs[-1], "pipelined last batch")
    # the one-call path still works afterwards and agrees
    lf.run_host(hbs[2], hts[2], st)
    assert_tracks_equal(hts[2].to_numpy(), refs[2], "lf_run_host after the pipeline")
    # misuse
    lf.host_submit(hbs[0], hts[0], 0, st)
    with pytest.raises(lfmod.LfError):
        lf.host_submit(hbs[1], hts[1], 0, st)                      # slot not collected
    with pytest.raises(lfmod.LfError):
        lf.host_submit(hbs[1], hts[1], 1, torch.cuda.Stream())     # another stream while a batch is in flight
    with pytest.raises(lfmod.LfError):
        lf.run_host(hbs[1], hts[1], st)                            # one-call path while a batch is in flight
    with pytest.raises(lfmod.LfError):
        lf.run(lfmod.DeviceBatch(batches[1]))                      # device path while a batch is in flight
    with pytest.raises(lfmod.LfError):
        lf.host_collect(1)                                         # nothing submitted there
    with pytest.raises(lfmod.LfError):
        lf.host_submit(hbs[1], hts[1], 2, st)                      # no such slot
    lf.host_collect(0)
    assert_tracks_equal(hts[0].to_numpy(), refs[0], "batch collected after refused calls")
    lf.host_submit(hbs[0], hts[0], 1, st)
    lf.close()  # lf_destroy with a batch in flight waits for it
    torch.cuda.synchronize()
