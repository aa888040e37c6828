"""the oracle under AddressSanitizer + UndefinedBehaviorSanitizer.

The oracle is built with ``-fsanitize=address,undefined -fno-sanitize-recover=all`` into a temporary directory and
driven, in a subprocess with the sanitizer runtimes preloaded, over configs 0, 1 and 4 in both tunings (with the
debug tables, the fp32 and the fp64 build).  Any out-of-bounds access, use of an uninitialised index as an array
subscript that leaves its object, signed overflow or misaligned access aborts the subprocess."""
import os
import shutil
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "lf_oracle.cpp")


def _runtime(name):
    path = subprocess.run(["g++", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return path if os.path.isabs(path) and os.path.exists(path) else None


@pytest.mark.skipif(shutil.which("g++") is None, reason="needs g++")
def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if asan is None or ubsan is None:
        pytest.skip("sanitizer runtimes not installed")
    flags = ["-std=c++17", "-O1", "-g", "-ffp-contract=off", "-fno-fast-math", "-fsanitize=address,undefined",
             "-fno-sanitize-recover=all", "-shared", "-fPIC"]
    libs = {"f32": str(tmp_path / "liblf_oracle.so"), "f64": str(tmp_path / "liblf_oracle_f64.so")}
    for kind, lib in libs.items():
        subprocess.run(["g++"] + flags + (["-DLF_ORACLE_REAL=double"] if kind == "f64" else []) + [SRC, "-o", lib], check=True)
    script = textwrap.dedent(f"""
        import sys
        sys.path.insert(0, {ROOT!r})
        from oracle import lf_oracle
        from paper_2402_14670_b200 import datagen as dg
        lf_oracle._LIBS = {libs!r}
        G = dg.toy_geometry()
        total = 0
        for cid, n_ev in ((0, None), (1, 30), (4, 10)):
            b = dg.generate_config(cid, n_events=n_ev)
            for P in (dg.default_params(), dg.no_ut_params()):
                for real in ("f32", "f64"):
                    total += lf_oracle.run(G, P, b, debug=True, real=real).n_tracks
        # edge cases: no events, events without seeds or hits
        import numpy as np
        e = dg.generate(dg.GenConfig("empty", 3, 1, true_fixed=0, noise_fixed=0))
        total += lf_oracle.run(G, dg.default_params(), e, debug=True).n_tracks
        print("SANITIZED_OK", total)
    """)
    env = dict(os.environ, LD_PRELOAD=f"{asan}:{ubsan}", ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    res = subprocess.run([sys.executable, "-c", script], capture_output=True, text=True, env=env, timeout=900)
    assert res.returncode == 0, res.stdout[-2000:] + res.stderr[-4000:]
    assert "SANITIZED_OK" in res.stdout
    assert "runtime error" not in res.stderr and "AddressSanitizer" not in res.stderr
