"""Randomised parameter sweep (-m gpu): narrow and wide kernels, both tunings, against the oracle at every stage boundary.

Seeded draws of the tunables (window cap 2..64, triplet cap 1..32, hit-count rule, tolerances, window overlap incl. a
negative one, polarity, dRatio, Eq. 9 table on/off) on small dense and sparse batches.  Everything must equal the oracle:
windows, kept triplets, extension hit lists, candidate Q, tracks; every third set also through the release build of the
kernels, every fifth through the host path as a stream of two batches."""
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


def _draw(rng, geometry, table):
    mode = int(rng.integers(0, 2))
    P = dg.no_ut_params() if mode == 1 else dg.default_params()
    P = dict(P)
    P["n_window"] = int(rng.choice([2, 3, 7, 16, 31, 32, 33, 47, 63, 64]))
    P["n_triplets"] = int(rng.choice([1, 2, 5, 12, 16, 17, 20, 31, 32]))
    P["min_hits"] = int(rng.integers(6, 13))
    P["T_triplet"] = float(rng.choice([0.5, 2.0, 8.0, 40.0]))
    P["T_x"] = float(rng.choice([0.3, 0.5, 2.0, 9.0]))
    P["T_uv_slope"] = float(rng.choice([5.0, 15.0, 50.0, 200.0]))
    P["T_uv_min"] = float(rng.choice([0.1, 0.5, 4.0]))
    P["T_ty"] = float(rng.choice([0.001, 0.003, 0.02, 0.2]))
    P["T_Q"] = float(rng.choice([0.05, 0.5, 5.0]))
    P["uv_half_width"] = float(rng.choice([100.0, 800.0, 1200.0]))
    if mode == 0:
        P["xtol_base"] = float(rng.choice([20.0, 150.0, 400.0]))
        P["x_asym"] = float(rng.choice([0.0, 100.0, 300.0]))
        P["p_same_bend"] = float(rng.choice([0.0, 5.0, 50.0]))
        P["mag_tol_tx"] = float(rng.choice([0.0, 20.0, 100.0]))
        P["mag_tol_max"] = float(rng.choice([10.0, 40.0, 120.0]))
    else:
        P["velo_p_min"] = float(rng.choice([2.0, 5.0, 20.0]))
        P["velo_pt_min"] = float(rng.choice([0.3, 1.0]))
        P["x_overlap"] = float(rng.choice([-3.0, 0.0, 5.0, 80.0]))
        P["mag_tol_base"] = P["mag_tol_max"] = float(rng.choice([3.0, 10.0, 35.0]))
    G = dict(geometry, polarity=int(rng.choice([-1, 1])), d_ratio=float(rng.choice([0.0, -2.0e-5, 1.5e-5])))
    if rng.integers(0, 2):
        G = dict(G, qop_mode=1, qop_poly2d=table)
    return G, P


def test_random_parameter_sets(lfmod, oracle, geometry):
    import torch
    from paper_2402_14670_b200 import momentum_fit as mf
    table = mf.fit_qop_poly2d(0.8, 1.5, n_toys=20000)
    batches = [dg.generate(dg.GenConfig("fz_dense", 5, 501, true_fixed=35, fake_mean=6.0, noise_fixed=700, p_min=1.5, smear=0.2)),
               dg.generate(dg.GenConfig("fz_sparse", 12, 502, true_fixed=15, fake_mean=3.0, noise_fixed=60)),
               dg.generate(dg.with_overrides(dg.CONFIGS[1], seed=503, field_ax=0.8, field_ay=1.5), n_events=25)]
    rng = np.random.Generator(np.random.PCG64(20240601))
    n_wide = n_tracks = 0
    for it in range(60):
        G, P = _draw(rng, geometry, table)
        b = batches[it % len(batches)]
        ref = oracle.run(G, P, b, debug=True, threads=NTHREADS)
        lf = lfmod.LookingForward(G, P, b.n_events, b.n_seeds, b.n_hits)
        out = lf.run(lfmod.DeviceBatch(b), debug=True)
        torch.cuda.synchronize()
        got = out.to_numpy()
        got.debug = {k: v.cpu().numpy() for k, v in vars(out.debug_tensors).items()}
        what = f"fuzz {it}: mode {P['mode']}, n_window {P['n_window']}, n_triplets {P['n_triplets']}, min_hits {P['min_hits']}"
        try:
            assert_debug_equal(got.debug, ref.debug)
            assert_tracks_equal(got, ref, what)
            if it % 3 == 0:  # the release build of the kernels
                out2 = lf.run(lfmod.DeviceBatch(b))
                torch.cuda.synchronize()
                assert_tracks_equal(out2.to_numpy(), ref, what + " (release kernels)")
            if it % 5 == 0:  # the host path as a stream: the same batch in both slots, small chunks
                lf.set_host_chunk_events(int(rng.integers(1, 9)))
                hb = lfmod.HostBatch(b)
                hts = [lfmod.HostTracks(max(b.n_seeds, 1), b.n_events) for _ in range(2)]
                lf.host_submit(hb, hts[0], 0)
                lf.host_submit(hb, hts[1], 1)
                for slot in range(2):
                    lf.host_collect(slot)
                    assert_tracks_equal(hts[slot].to_numpy(), ref, what + f" (stream, slot {slot})")
        except AssertionError as e:
            raise AssertionError(f"{what}: {e}\nparams: {P}") from e
        lf.close()
        n_wide += int(P["mode"] == 1 or P["n_window"] > 32 or P["n_triplets"] > 16)
        n_tracks += ref.n_tracks
    assert 20 <= n_wide <= 58 and n_tracks > 3000
