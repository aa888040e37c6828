"""``lf_windows_static``: the entry point for callers that cannot allocate device memory.

Why it exists: every other call of include/lf.h needs a handle from ``lf_create``, and ``lf_create`` calls ``cudaMalloc``.
A host that has handed all of the GPU's memory to its own pool at start-up, or that sits in an event loop where the
device-wide stall of ``cudaMalloc`` / ``cudaFree`` is not acceptable, cannot make that call.  For such a host the library
offers the search-window stage (a1 + a2) with its scratch memory in a fixed array inside the library image: no handle,
no allocation, but a bounded batch size and one shared array per GPU.

What is checked here:
  * (CPU) batches beyond the fixed array are refused with LF_ERR_CAPACITY and a message naming the limits, and bad
    arguments are refused, all before the first CUDA call;
  * (GPU) two calls in a row on one stream, with different batches and no synchronisation in between, each give the
    window tables that the existing path (``lf_create`` + ``lf_run_debug``) gives for the same batch.  The tables are
    integers, so "within the tests' tolerance" means equal: counts everywhere, first-hit indices wherever the count is
    non-zero (include/lf.h leaves the index of an empty window undefined).  The second call finds the array as the first
    one left it, which is the situation the entry point must cope with;
  * (GPU) the device's free memory is the same before and after a call once the first call on the device is behind us.

The file name sorts last on purpose: ``pytest -x`` stops at the first failure, and a failure here should not hide any
other test.  The GPU tests build and load the library themselves, so they pass alone in a fresh process as well as at the
end of the whole suite (where other handles have already run on the device).
"""
import ctypes

import numpy as np
import pytest

from paper_2402_14670_b200 import datagen as dg


@pytest.fixture(scope="module")
def binding():
    from paper_2402_14670_b200 import build as cuda_build
    cuda_build.build()
    from paper_2402_14670_b200 import binding as bd
    bd.load_library()
    return bd


def test_static_limits_are_refused_before_any_cuda_call(binding, geometry, params):
    """Runs without a GPU: sizes and arguments are checked before the first CUDA call."""
    lib = binding.load_library()
    g = binding._fill(binding.lf_geometry(), geometry)
    p = binding._fill(binding.lf_params(), params)
    hits = binding.lf_hits(None, None, 0, None, None)

    def call(pp, n_events, n_seeds):
        seeds = binding.lf_seeds(None, None, None, None, None, None, n_seeds)
        return lib.lf_windows_static(ctypes.byref(g), ctypes.byref(pp), ctypes.byref(seeds), ctypes.byref(hits), n_events,
                                     None, None, None)

    assert call(p, binding.STATIC_MAX_EVENTS + 1, 10) == binding.LF_ERR_CAPACITY
    msg = lib.lf_last_error(None).decode()
    assert "LF_STATIC_MAX_EVENTS = 4096" in msg and "LF_STATIC_MAX_ROWS = 16384" in msg
    assert call(p, 10, binding.STATIC_MAX_ROWS + 1) == binding.LF_ERR_CAPACITY
    # the no-UT tuning follows two window sides per seed: half as many seeds fit
    p_nout = binding._fill(binding.lf_params(), dg.no_ut_params())
    assert call(p_nout, 10, binding.STATIC_MAX_ROWS // 2 + 1) == binding.LF_ERR_CAPACITY
    # at the limit the sizes pass, and the call stops at the next check (NULL offset tables)
    assert call(p, binding.STATIC_MAX_EVENTS, binding.STATIC_MAX_ROWS) == binding.LF_ERR_INVALID_ARG
    assert call(p_nout, 10, binding.STATIC_MAX_ROWS // 2) == binding.LF_ERR_INVALID_ARG
    # fp16 hit storage needs more scratch than the fixed array has; invalid tunables are refused as lf_create refuses them
    assert call(binding._fill(binding.lf_params(), dict(params, hit_storage=1)), 10, 10) == binding.LF_ERR_UNSUPPORTED
    assert call(binding._fill(binding.lf_params(), dict(params, n_window=65)), 10, 10) == binding.LF_ERR_INVALID_ARG
    assert lib.lf_windows_static(None, None, None, None, 0, None, None, None) == binding.LF_ERR_INVALID_ARG
    # an empty batch is valid and writes nothing
    assert call(p, 0, 0) == binding.LF_OK
    # the header's size is the sum of its parts: 64-byte rows, 8 + 4 bytes per event, one 256-byte block
    assert binding.STATIC_MAX_ROWS * 64 + binding.STATIC_MAX_EVENTS * 12 + 256 == 1097984


def _existing_path(binding, G, P, b):
    """Window tables through lf_create + lf_run_debug (library-allocated workspace)."""
    import torch
    lf = binding.LookingForward(G, P, max(b.n_events, 1), max(b.n_seeds, 1), max(b.n_hits, 1))
    out = lf.run(binding.DeviceBatch(b), debug=True)
    torch.cuda.synchronize()
    first, count = out.debug_tensors.win_first.cpu().numpy(), out.debug_tensors.win_count.cpu().numpy()
    lf.close()
    return first, count


def _assert_same_windows(first, count, ref_first, ref_count, what):
    assert count.shape == ref_count.shape
    assert np.array_equal(count, ref_count), f"{what}: window sizes differ from lf_run_debug's"
    m = ref_count > 0
    assert np.array_equal(first[m], ref_first[m]), f"{what}: window starts differ from lf_run_debug's"


@pytest.mark.gpu
@pytest.mark.parametrize("tuning", ["with-ut", "no-ut"])
def test_static_windows_match_existing_path_two_calls_in_a_row(binding, geometry, params, tuning):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    P = dg.no_ut_params() if tuning == "no-ut" else params
    sides = 2 if tuning == "no-ut" else 1
    big = dg.generate_config(1, n_events=40)    # ~7 200 seeds, ~200 000 hits: several events per thread block
    small = dg.generate_config(0)               # 10 events, 200 seeds: fewer events than the first call left state for
    assert big.n_seeds * sides <= binding.STATIC_MAX_ROWS
    refs = [_existing_path(binding, geometry, P, b) for b in (big, small)]

    dbs = [binding.DeviceBatch(b) for b in (big, small)]
    outs = [(torch.full((b.n_seeds * sides, 12), -7, dtype=torch.int32, device="cuda"),
             torch.full((b.n_seeds * sides, 12), -7, dtype=torch.int32, device="cuda")) for b in (big, small)]
    torch.cuda.synchronize()
    # two calls in a row on the same stream, nothing in between: the second starts on the array as the first left it
    for db, (wf, wc) in zip(dbs, outs):
        binding.windows_static(geometry, P, db, wf, wc)
    torch.cuda.synchronize()
    for name, (wf, wc), (rf, rc) in zip(("first call", "second call"), outs, refs):
        wc_h = wc.cpu().numpy()
        assert (wc_h >= 0).all(), f"{name}: rows left unwritten"
        _assert_same_windows(wf.cpu().numpy(), wc_h, rf, rc, f"{tuning}, {name}")
    assert refs[0][1].max() == int(P["n_window"]) and refs[0][1].sum() > 0   # the cap binds somewhere: a real workload

    # and once more the other way round (large batch after the small one), now checking that nothing gets allocated:
    # the set-up of the first call on this device is behind us
    free_before, _ = torch.cuda.mem_get_info()
    wf, wc = outs[0]
    wf.fill_(-7), wc.fill_(-7)
    binding.windows_static(geometry, P, dbs[0], wf, wc)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    _assert_same_windows(wf.cpu().numpy(), wc.cpu().numpy(), refs[0][0], refs[0][1], f"{tuning}, third call")
    assert free_after == free_before, "lf_windows_static changed the device's free memory"


@pytest.mark.gpu
def test_static_windows_oversize_batch_is_refused_on_the_gpu(binding, geometry, params):
    """A real batch beyond the limit comes back as LF_ERR_CAPACITY, and the next valid call still works."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    too_big = dg.generate_config(1, n_events=120)   # ~21 600 seeds > LF_STATIC_MAX_ROWS
    assert too_big.n_seeds > binding.STATIC_MAX_ROWS
    db = binding.DeviceBatch(too_big)
    wf = torch.empty((too_big.n_seeds, 12), dtype=torch.int32, device="cuda")
    wc = torch.empty_like(wf)
    with pytest.raises(binding.LfError) as ei:
        binding.windows_static(geometry, params, db, wf, wc)
    assert ei.value.status == binding.LF_ERR_CAPACITY and "exceed the static scratch" in str(ei.value)
    small = dg.generate_config(0)
    rf, rc = _existing_path(binding, geometry, params, small)
    wf = torch.full((small.n_seeds, 12), -7, dtype=torch.int32, device="cuda")
    wc = torch.full_like(wf, -7)
    binding.windows_static(geometry, params, binding.DeviceBatch(small), wf, wc)
    torch.cuda.synchronize()
    _assert_same_windows(wf.cpu().numpy(), wc.cpu().numpy(), rf, rc, "after a refused call")
