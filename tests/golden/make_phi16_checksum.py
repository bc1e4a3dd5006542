"""Writes tests/golden/phi16_grid_checksum.txt from the CPU oracle only (never the CUDA path).

Grid: i, j = -400..400 (i outer), x = float32((i+0.5)*0.055*1.9),
y = float32((j+0.5)*0.055*1.9) evaluated in double then rounded; FNV-1a-64 over the
little-endian bytes of uint16(phi16).
Run: python tests/golden/make_phi16_checksum.py
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle  # noqa: E402


def grid():
    i = np.arange(-400, 401)
    v = ((i + 0.5) * 0.055 * 1.9).astype(np.float32)
    return np.repeat(v, 801), np.tile(v, 801)


def fnv1a64(data: bytes) -> int:
    h = 0xCBF29CE484222325
    for c in data:
        h = ((h ^ c) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
    return h


if __name__ == "__main__":
    x, y = grid()
    ph = oracle.phi16(x, y)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "phi16_grid_checksum.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_phi16_checksum.py (oracle only); see README.md\n")
        f.write("%016x\n" % fnv1a64(ph.astype(np.uint16).astype("<u2").tobytes()))
    print(open(out).read())
