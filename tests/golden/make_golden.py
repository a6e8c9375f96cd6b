"""Writes tests/golden/offset_crc32.txt: zlib CRC-32 of the little-endian int64 offset array
(n_sticks + 1 entries) of each configuration.  Calls ONLY the oracle (never the CUDA path).

    python tests/golden/make_golden.py
"""
import os
import sys
import zlib

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import oracle  # noqa: E402

CASES = [
    ("cfg1", (32, 32, 32), (8, 8, 8)),
    ("cfg2", (64, 64, 64), (16, 16, 16)),
    ("cfg3", (128, 128, 128), (32, 32, 32)),
    ("cfg4", (96, 96, 192), (24, 24, 48)),
    ("cfg5", (256, 256, 256), (64, 64, 64)),
    ("tiny8", (8, 8, 8), (2, 2, 2)),
    ("tiny468", (4, 6, 8), (1, 1, 2)),
]

with open(os.path.join(HERE, "offset_crc32.txt"), "w") as f:
    f.write("# written by tests/golden/make_golden.py from oracle.stick_map only\n")
    f.write("# name N1 N2 N3 a1 a2 a3 n_points n_sticks crc32(off as <i8)\n")
    for name, n, a in CASES:
        m = oracle.stick_map(n, a)
        crc = zlib.crc32(m["off"].astype("<i8").tobytes()) & 0xFFFFFFFF
        f.write(f"{name} {n[0]} {n[1]} {n[2]} {a[0]} {a[1]} {a[2]} {int(m['off'][-1])} {len(m['k1'])} {crc:08x}\n")
