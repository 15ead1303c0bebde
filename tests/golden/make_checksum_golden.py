"""Writes tests/golden/checksum.txt.  Calls only oracle/ (never the CUDA path).

The checksum is build-defined (BASELINE.json north_star (d), reading R22), so there is no
printed value in the paper to cite: the literals freeze the definition, and tests/test_oracle_checksum.py checks the
oracle against them AND against a big-int restatement that shares nothing with oracle/.

    python tests/golden/make_checksum_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import rco  # noqa: E402


def main():
    z = np.zeros(4096, np.uint8)
    ramp = (np.arange(4096) & 0xFF).astype(np.uint8)
    zb = np.zeros(4 * 4096, np.uint8)
    dz = rco.block_digest(zb, 4, 0)
    rows = [
        ("mixL(0)", rco.mixL(0)), ("mixL(1)", rco.mixL(1)), ("mixF(1)", rco.mixF(1)),
        ("mum(3,5)", rco.mum(3, 5)), ("mum(2^63,6)", rco.mum(1 << 63, 6)),
        ("mum(C1,C2)", rco.mum(0x9E3779B97F4A7C15, 0x6A09E667F3BCC909)),
        ("page_digest(zero4096).d", rco.page_digest(z, 0)), ("page_digest(zero4096).e", rco.page_digest(z, 1)),
        ("page_digest(ramp4096).d", rco.page_digest(ramp, 0)), ("page_digest(ramp4096).e", rco.page_digest(ramp, 1)),
        ("block_digest(tiny zero block).d", dz), ("block_digest(tiny zero block).e", rco.block_digest(zb, 4, 1)),
        ("chain_seed(1)", rco.chain_of(1, [])), ("chain_of(1,[dz])", rco.chain_of(1, [dz])),
        ("chain_of(1,[dz,dz])", rco.chain_of(1, [dz, dz])),
    ]
    with open(os.path.join(HERE, "checksum.txt"), "w") as f:
        f.write("# Golden checksum values, written by tests/golden/make_checksum_golden.py (calls only oracle/).\n"
                "# The checksum is build-defined (BASELINE.json north_star (d); DESIGN.md \"Checksum\", reading R22):\n"
                "# these literals freeze it.  mixL / mixF / chain seed are unchanged from SURVEY.md 8(c).3; the lane\n"
                "# fold is the mum fold of R22.  tests/test_oracle_checksum.py checks the oracle against them and\n"
                "# against an independent big-int restatement.\n")
        for k, v in rows:
            f.write("%s = 0x%X\n" % (k, v))


if __name__ == "__main__":
    main()
