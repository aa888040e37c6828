"""Writes tests/golden/cfg0_oracle_tracks.txt from the ORACLE only (never from the CUDA path).

Run from the repo root:  python tests/golden/make_golden.py
The file is a regression guard for the oracle (a later change to its arithmetic must name, in its
commit message, the PAPER.md passage or DESIGN.md reading that justifies it), not a pin.
Columns: seed_idx n_hits hit_idx[0..11] quality(float32 hex) state[0..4](float32 hex).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import lf_oracle  # noqa: E402
from paper_2402_14670_b200 import datagen  # noqa: E402  (input generator only)


def main():
    b = datagen.generate_config(0)
    r = lf_oracle.run(datagen.toy_geometry(), datagen.default_params(), b)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle_tracks.txt")
    with open(out, "w") as f:
        f.write("# oracle output for BASELINE.json configs[0] (10 events x 20 tracks, seed 1000); written by make_golden.py\n")
        for i in range(r.n_tracks):
            hx = lambda v: np.float32(v).view(np.uint32).item()
            f.write(" ".join([str(int(r.seed_idx[i])), str(int(r.n_hits[i]))] + [str(int(h)) for h in r.hit_idx[i]]
                             + [f"{hx(r.quality[i]):08x}"] + [f"{hx(v):08x}" for v in r.state[i]]) + "\n")
    print("wrote", out, r.n_tracks, "tracks")


if __name__ == "__main__":
    main()
