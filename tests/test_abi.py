"""The C-ABI library loads on a CPU-only box and exports every symbol include/lf.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2402_14670_b200 import build as cuda_build
    cuda_build.build()
    from paper_2402_14670_b200 import binding
    return binding.load_library()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "lf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lf_[a-z_]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    names = _declared_functions()
    assert {"lf_create", "lf_run", "lf_run_debug", "lf_run_host", "lf_destroy", "lf_last_error", "lf_get_info",
            "lf_abi_version", "lf_sizeof"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"liblf_b200.so does not export {n}"


def test_struct_sizes_match_binding(lib):
    from paper_2402_14670_b200 import binding
    for i, st in enumerate(binding._STRUCTS):
        assert lib.lf_sizeof(i) == ctypes.sizeof(st)
    assert lib.lf_sizeof(99) == 0 and lib.lf_abi_version() == 7


def test_argument_validation_needs_no_gpu(lib, geometry, params):
    """Invalid arguments are rejected before any CUDA call (so this runs on a CPU-only box)."""
    from paper_2402_14670_b200 import binding as bd
    h = ctypes.c_void_p()
    assert lib.lf_create(None, None, 1, 1, 1, ctypes.byref(h)) == bd.LF_ERR_INVALID_ARG
    g = bd._fill(bd.lf_geometry(), geometry)
    for bad_params, why in ((dict(params, n_window=65), "n_window"), (dict(params, n_triplets=0), "n_triplets"),
                            (dict(params, n_triplets=33), "n_triplets"), (dict(params, mode=2), "mode"),
                            (dict(params, mode=1, velo_pt_min=0.0), "velo_pt_min"),
                            (dict(params, min_hits=2), "min_hits"), (dict(params, T_x=0.0), "positive"),
                            (dict(params, mag_tol_max=float("inf")), "non-finite"), (dict(params, xtol_base=float("nan")), "non-finite"),
                            (dict(params, uv_half_width=-1.0), ">= 0"), (dict(params, C_nhits=[5.0, 0.0, 0.8, 0.5]), "C_nhits")):
        p = bd._fill(bd.lf_params(), bad_params)
        assert lib.lf_create(ctypes.byref(g), ctypes.byref(p), 1, 1, 1, ctypes.byref(h)) == bd.LF_ERR_INVALID_ARG
        assert why in lib.lf_last_error(None).decode()
    # fp16 hit storage exists for the narrow with-UT kernels only
    for unsupported in (dict(params, hit_storage=1, mode=1), dict(params, hit_storage=1, n_window=64)):
        p = bd._fill(bd.lf_params(), unsupported)
        assert lib.lf_create(ctypes.byref(g), ctypes.byref(p), 1, 1, 1, ctypes.byref(h)) == bd.LF_ERR_UNSUPPORTED
    p = bd._fill(bd.lf_params(), params)
    for bad_geo in (dict(geometry, n_layers=8), dict(geometry, polarity=0), dict(geometry, qop_mode=2),
                    dict(geometry, tan_alpha=[0.0] * 12), dict(geometry, z=list(reversed(geometry["z"]))),
                    dict(geometry, kick=0.0), dict(geometry, kick=float("inf")), dict(geometry, z_ref=float("nan"))):
        gg = bd._fill(bd.lf_geometry(), bad_geo)
        assert lib.lf_create(ctypes.byref(gg), ctypes.byref(p), 1, 1, 1, ctypes.byref(h)) == bd.LF_ERR_INVALID_ARG
    assert lib.lf_destroy(None) == bd.LF_OK
    assert lib.lf_run(None, None, None, 0, None, None) == bd.LF_ERR_INVALID_ARG


def test_no_cpu_fallback(lib, geometry, params):
    """Without a CUDA device lf_create fails loudly with LF_ERR_CUDA; nothing routes through the oracle."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    from paper_2402_14670_b200 import binding as bd
    with pytest.raises(bd.LfError) as ei:
        bd.LookingForward(geometry, params, 1, 1, 1)
    assert ei.value.status == bd.LF_ERR_CUDA
    # the product package never imports the oracle
    import subprocess, sys
    code = "import sys; import paper_2402_14670_b200.binding, paper_2402_14670_b200.datagen; assert not any(m.startswith('oracle') for m in sys.modules)"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
