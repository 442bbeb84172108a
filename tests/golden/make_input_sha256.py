"""Writes tests/golden/input_sha256.txt: SHA-256 of the seeded coefficient arrays of
paper_2402_01282_b200/inputs.py (random draws only; no transform arithmetic, nothing from the CUDA path)."""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from paper_2402_01282_b200 import inputs as I  # noqa: E402

with open(os.path.join(HERE, "input_sha256.txt"), "w") as fh:
    fh.write("# SHA-256 of inputs.config_coefficients(name) (numpy default_rng streams; DESIGN.md 'Inputs').\n")
    fh.write("# written by tests/golden/make_input_sha256.py\n# columns: config sha256\n")
    for name in ("C1", "C2", "C3", "C4", "C5"):
        fh.write("%s %s\n" % (name, I.sha256(I.config_coefficients(name))))
