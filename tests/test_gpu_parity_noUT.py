"""GPU parity of the wide kernels (-m gpu): the no-UT tuning and the with-UT tuning with caps
beyond the narrow limits, through the C ABI, vs the CPU oracle element by element."""
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


@pytest.fixture(scope="module")
def nparams():
    return dg.no_ut_params()


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


def _both(lfmod, oracle, G, P, b, what, debug=True):
    ref = oracle.run(G, P, b, debug=debug, threads=NTHREADS)
    got = _gpu_run(lfmod, G, P, b, debug=debug)
    if debug:
        assert_debug_equal(got.debug, ref.debug)
    return assert_tracks_equal(got, ref, what), ref


def test_noUT_config0_tracks_and_stage_boundaries(lfmod, oracle, geometry, nparams):
    b = dg.generate_config(0)
    info, ref = _both(lfmod, oracle, geometry, nparams, b, "no-UT config 0")
    assert ref.n_tracks > 100 and ref.debug.win_count.shape[0] == 2 * b.n_seeds
    got2 = _gpu_run(lfmod, geometry, nparams, b)
    assert_tracks_equal(got2, ref, "no-UT config 0 (release kernel)")
    print("noUT config0", info, ref.n_tracks)


def test_noUT_dense_events_stage_boundaries(lfmod, oracle, geometry, nparams):
    """Window cap (64 and smaller) and top-n cut bind on both sides; loose cuts; non-zero dRatio; both polarities."""
    cfg = dg.GenConfig("dense", 6, 77, true_fixed=40, fake_mean=8.0, noise_fixed=900, p_min=3.0)
    b = dg.generate(cfg)
    loose = dict(nparams, T_triplet=8.0, T_x=2.0, T_uv_slope=50.0, T_ty=0.02, mag_tol_base=30.0, mag_tol_max=30.0, x_overlap=60.0)
    for G, P in ((geometry, nparams), (dict(geometry, polarity=-1), loose),
                 (dict(geometry, d_ratio=-2.0e-5), dict(loose, n_window=17, n_triplets=3)),
                 (geometry, dict(loose, n_window=64, n_triplets=32, min_hits=8, velo_p_min=3.0, velo_pt_min=0.6))):
        info, ref = _both(lfmod, oracle, G, P, b, "no-UT dense")
    assert (ref.debug.win_count == 64).mean() > 0.2
    assert (ref.debug.n_triplets == 32).sum() > 10


def test_noUT_config1_full(lfmod, oracle, geometry, nparams):
    b = dg.generate_config(1)
    info, ref = _both(lfmod, oracle, geometry, nparams, b, "no-UT config 1", debug=False)
    print("noUT config1", info, ref.n_tracks)


def test_noUT_config1_stage_boundaries_subset(lfmod, oracle, geometry, nparams):
    _both(lfmod, oracle, geometry, nparams, dg.generate_config(1, n_events=100), "no-UT config 1 subset")


def test_noUT_config4_full_size(lfmod, oracle, geometry, nparams):
    """High occupancy (about 500 hits per segment): the 64-hit cap binds often.  All 5 000 events of BASELINE.json
    configs[4] in one lf_run, element by element: the workload whose no-UT time DESIGN.md section 7.1 quotes; the stage
    boundaries on a 40-event subset."""
    b = dg.generate_config(4)
    assert b.n_events == 5000
    info, ref = _both(lfmod, oracle, geometry, nparams, b, "no-UT config 4", debug=False)
    b2 = dg.generate_config(4, n_events=40)
    info2, ref2 = _both(lfmod, oracle, geometry, nparams, b2, "no-UT config 4 subset")
    assert (ref2.debug.win_count == 64).mean() > 0.3
    print("noUT config4", info, ref.n_tracks)


def test_noUT_config3_full_size(lfmod, oracle, geometry, nparams):
    """The launch configuration `bench.py --config 5` times: 20,000 events in one lf_run."""
    b = dg.generate_config(3)
    got = _gpu_run(lfmod, geometry, nparams, b)
    ref = oracle.run(geometry, nparams, b, threads=NTHREADS)
    print("noUT config3", assert_tracks_equal(got, ref, "no-UT config 3"), ref.n_tracks)


def test_withUT_wide_caps(lfmod, oracle, geometry, params):
    """mode 0 beyond the narrow limits (n_window > 32 or n_triplets > 16) runs the wide kernels."""
    b = dg.generate_config(4, n_events=60)
    for P in (dict(params, n_window=64, n_triplets=20), dict(params, n_window=47, n_triplets=32, T_triplet=20.0),
              dict(params, n_window=32, n_triplets=17)):
        info, ref = _both(lfmod, oracle, geometry, P, b, "with-UT wide")
    b1 = dg.generate_config(1, n_events=300)
    _both(lfmod, oracle, geometry, dict(params, n_window=64, n_triplets=20), b1, "with-UT wide config 1", debug=False)


def test_noUT_edge_cases(lfmod, oracle, geometry, nparams):
    import torch
    empty = dg.generate(dg.GenConfig("e", 0, 1))
    got = _gpu_run(lfmod, geometry, nparams, empty)
    assert got.n_tracks == 0 and got.event_offsets.tolist() == [0]
    noseed = dg.generate(dg.GenConfig("ns", 3, 2, true_fixed=0, noise_fixed=50))
    got = _gpu_run(lfmod, geometry, nparams, noseed)
    assert got.n_tracks == 0 and got.event_offsets.tolist() == [0, 0, 0, 0]
    b = dg.generate_config(0)
    # q/p is never read in the no-UT mode: NaN seeds give the same answer
    ref = oracle.run(geometry, nparams, b, debug=True)
    bn = dg.Batch(**{**b.__dict__, "seed_qop": np.full_like(b.seed_qop, np.nan)})
    got = _gpu_run(lfmod, geometry, nparams, bn, debug=True)
    assert_debug_equal(got.debug, ref.debug)
    assert_tracks_equal(got, ref, "NaN q/p")
    # duplicates of one x value in every segment; zero slopes (x_tol = 0: only the overlap)
    one = dg.Batch(**{**b.__dict__})
    one.hit_x = np.full(b.n_events * 24 * 3, 12.5, np.float32)
    one.seg_offsets = (np.arange(b.n_events * 24 + 1) * 3).astype(np.uint32)
    one.hit_track = np.full(one.hit_x.shape[0], -1, np.int32)
    _both(lfmod, oracle, geometry, nparams, one, "duplicates")
    flat = dg.Batch(**{**b.__dict__, "seed_tx": np.zeros_like(b.seed_tx), "seed_ty": np.zeros_like(b.seed_ty)})
    _both(lfmod, oracle, geometry, nparams, flat, "zero slopes")


def test_noUT_event_larger_than_stage_buffer(lfmod, oracle, geometry, nparams):
    cfg = dg.GenConfig("huge", 3, 9, true_fixed=60, fake_mean=5.0, noise_fixed=1700, p_min=4.0)
    b = dg.generate(cfg)
    import torch
    lf = lfmod.LookingForward(geometry, nparams, b.n_events, b.n_seeds, b.n_hits)
    assert b.n_hits / b.n_events > lf.info().staged_hits_per_event
    out = lf.run(lfmod.DeviceBatch(b), debug=True)
    torch.cuda.synchronize()
    got = out.to_numpy()
    got.debug = {k: v.cpu().numpy() for k, v in vars(out.debug_tensors).items()}
    ref = oracle.run(geometry, nparams, b, debug=True)
    assert_debug_equal(got.debug, ref.debug)
    assert_tracks_equal(got, ref, "no-UT huge events")
    lf.close()


def test_noUT_run_host_and_determinism(lfmod, oracle, geometry, nparams):
    b = dg.generate_config(1, n_events=200)
    ref = oracle.run(geometry, nparams, b, threads=NTHREADS)
    lf = lfmod.LookingForward(geometry, nparams, b.n_events, b.n_seeds, b.n_hits)
    hb = lfmod.HostBatch(b)
    for chunk in (1024, 13):
        lf.set_host_chunk_events(chunk)
        ht = lfmod.HostTracks(b.n_seeds, b.n_events)
        assert lf.run_host(hb, ht) == ref.n_tracks
        assert_tracks_equal(ht.to_numpy(), ref, f"no-UT host path, chunks of >= {chunk} events")
    lf.close()
    a = _gpu_run(lfmod, geometry, nparams, b)
    c = _gpu_run(lfmod, geometry, nparams, b)
    assert np.array_equal(a.hit_idx, c.hit_idx) and np.array_equal(a.state.view(np.uint32), c.state.view(np.uint32))
    assert np.array_equal(a.quality.view(np.uint32), c.quality.view(np.uint32))


def test_noUT_stream_of_batches(lfmod, oracle, geometry, nparams):
    """lf_host_submit / lf_host_collect in the no-UT tuning (two rows per seed, seeds without q/p): a stream of unequal
    batches, two in flight, against the oracle."""
    import torch
    whole = dg.generate_config(1, n_events=240)
    cuts = [0, 100, 101, 170, 240]
    batches = [whole.slice_events(a, b) for a, b in zip(cuts[:-1], cuts[1:])]
    refs = [oracle.run(geometry, nparams, b, threads=NTHREADS) for b in batches]
    lf = lfmod.LookingForward(geometry, nparams, max(b.n_events for b in batches), max(b.n_seeds for b in batches),
                              max(b.n_hits for b in batches))
    lf.set_host_chunk_events(16)
    hbs = [lfmod.HostBatch(b) for b in batches]
    hts = [lfmod.HostTracks(b.n_seeds, b.n_events) for b in batches]
    st = torch.cuda.Stream()
    lf.host_submit(hbs[0], hts[0], 0, st)
    for i in range(1, len(batches)):
        lf.host_submit(hbs[i], hts[i], i % 2, st)
        lf.host_collect((i - 1) % 2)
        assert_tracks_equal(hts[i - 1].to_numpy(), refs[i - 1], f"no-UT stream, batch {i - 1}")
    lf.host_collect((len(batches) - 1) % 2)
    assert_tracks_equal(hts[-1].to_numpy(), refs[-1], "no-UT stream, last batch")
    lf.close()


def test_full_eq9_table_both_tunings(lfmod, oracle, geometry, params, nparams):
    """geometry.qop_mode = 1: q/p from the 2-D polynomial table, in a non-uniform toy field,
    narrow kernels (with UT) and wide kernels (no-UT); also the mirrored event (negated stereo angles, polarity)."""
    from paper_2402_14670_b200 import momentum_fit as mf
    table = mf.fit_qop_poly2d(0.8, 1.5)
    G1 = dict(geometry, qop_mode=1, qop_poly2d=table)
    b = dg.generate(dg.with_overrides(dg.CONFIGS[1], field_ax=0.8, field_ay=1.5, seed=3001), n_events=300)
    for P, what in ((params, "Eq. 9 table, with UT"), (nparams, "Eq. 9 table, no-UT")):
        info, ref = _both(lfmod, oracle, G1, P, b, what, debug=False)
        assert ref.n_tracks > 10000
        # the table changes q/p and nothing else
        ref0 = oracle.run(geometry, P, b, threads=NTHREADS)
        assert np.array_equal(ref.hit_idx, ref0.hit_idx) and np.array_equal(ref.state[:, :4], ref0.state[:, :4])
        assert np.max(np.abs(ref.state[:, 4] / ref0.state[:, 4] - 1.0)) > 0.02
    Gm = dict(G1, polarity=-1, tan_alpha=[-t for t in geometry["tan_alpha"]])
    _both(lfmod, oracle, Gm, params, b, "Eq. 9 table, mirrored geometry", debug=False)


def test_scan_script_runs(lfmod, tmp_path):
    """`python -m paper_2402_14670_b200.scan` (the Fig. 10-12 analogue) on a small batch: report written, rates positive."""
    from paper_2402_14670_b200 import scan
    out = tmp_path / "scan.md"
    assert scan.main(["--events", "150", "--steps", "1", "--sections", "window,streams", "--out", str(out)]) == 0
    text = out.read_text()
    assert "n_window scan" in text and "concurrent streams" in text
    rows = [l for l in text.splitlines() if l.startswith("| 32 |")]
    assert rows and float(rows[0].split("|")[5].strip().rstrip(" %")) > 95.0   # efficiency (p > 5, pT > 1) at n_window = 32
