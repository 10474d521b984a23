"""Writes tests/golden/charge_codes.txt: inputs and O9 codes (n = 4 for the charge and n = 3 for the
size).  Calls only oracle/ (never the CUDA path).  Run:  python tests/golden/make_charge_codes.py"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import tpc_oracle as orc      # noqa: E402

q = np.array([0, 1, 2, 15, 16, 17, 30, 31, 32, 33, 34, 35, 47, 48, 49, 63, 64, 65, 66, 67, 68, 99, 100, 101, 127, 128, 129,
              131, 132, 255, 256, 257, 264, 511, 512, 1000, 1023, 1024, 4095, 4096, 5000, 32767, 32768, 50000, 63487,
              63488, 64511, 64512, 65535, 0.5, 1.5, 2.5, 20.25, 99.99], np.float32)
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "charge_codes.txt"), "w") as f:
    f.write("# q  code(n=4, charge)  code(n=3, size)   -- PAPER.md L70; written by make_charge_codes.py from oracle/ only\n")
    for v, c4, c3 in zip(q, orc.pack_charge(q, 4), orc.pack_charge(q, 3)):
        f.write(f"{float(v):.2f} {int(c4)} {int(c3)}\n")
