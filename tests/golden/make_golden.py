"""Writes tests/golden/synth_values.txt: a few values of the seeded input generators.

Calls only paper_1808_01309_b200.synth (input data, no method arithmetic) -- never the CUDA path.
The values guard the generators against accidental change (a changed input would silently change
every parity case).  Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from paper_1808_01309_b200 import synth  # noqa: E402


def main():
    out = os.path.join(ROOT, "tests", "golden", "synth_values.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py from paper_1808_01309_b200/synth.py only\n")
        x = synth.uniform_field(32, 1, 1234)[0]
        for (k, j, i) in [(0, 0, 0), (1, 2, 3), (31, 31, 31)]:
            f.write(f"uniform64 32 1234 {k} {j} {i} {float(x[k, j, i])!r}\n")
        x = synth.uniform_field(32, 1, 1234, np.float32)[0]
        for (k, j, i) in [(0, 0, 0), (1, 2, 3), (31, 31, 31)]:
            f.write(f"uniform32 32 1234 {k} {j} {i} {float(x[k, j, i])!r}\n")
        u = synth.solenoidal_spectrum(128, 4.0, 32, 1234, 0)
        for (c, r, q, p) in [(0, 1, 2, 3), (1, 127, 5, 0), (2, 3, 126, 7)]:
            v = u[c, r, q, p]
            f.write(f"solenoidal 128 4.0 32 1234 0 {c} {r} {q} {p} {float(v.real)!r} {float(v.imag)!r}\n")
        u = synth.broadband_spectrum(64, seed=1234, tag=0)
        for (c, r, q, p) in [(0, 1, 2, 3), (1, 63, 5, 0), (2, 50, 10, 20)]:
            v = u[c, r, q, p]
            f.write(f"broadband 64 1234 0 {c} {r} {q} {p} {float(v.real)!r} {float(v.imag)!r}\n")
        t = synth.broadband_scalar(64, seed=1234)
        for (r, q, p) in [(1, 2, 3), (63, 5, 0)]:
            v = t[r, q, p]
            f.write(f"broadband_scalar 64 1234 7 {r} {q} {p} {float(v.real)!r} {float(v.imag)!r}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
