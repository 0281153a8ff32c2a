"""Rewrites tests/golden/keyed_hash.txt from the oracle alone (never from the CUDA path)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import sgw_oracle as o  # noqa: E402

CASES = [(0, 0, 0), (1, 0, 0), (1, 2, 3), (20260121, 63, 884735)]
with open(os.path.join(os.path.dirname(__file__), "keyed_hash.txt"), "w") as f:
    f.write("# seed vec g hash  -- keyed hash h = sm64(sm64(sm64(seed) ^ vec) ^ g); sign = top bit (SURVEY.md 8(c))\n")
    for s, v, g in CASES:
        f.write(f"{s} {v} {g} 0x{o.keyed_hash(s, v, g):016X}\n")
