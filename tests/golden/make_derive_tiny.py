"""Writes tests/golden/derive_tiny.txt: IR, D and B of two chained frames of a tiny configuration, from the CPU oracle.

Imports nothing but `oracle/` (never the CUDA library): the stored bytes are the oracle's, and tests/test_oracle_derivation.py
checks them against a pure-Python binary64 restatement of SURVEY.md 8(c) steps 2-7 and 10 (PAPER.md:35-43 Eq. 1, :55, :59) that
shares no code with the oracle, and tests/test_library_host.py checks the product's host derivation against the same file.
Run from the repository root:   python tests/golden/make_derive_tiny.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle  # noqa: E402

KEY = (3.141592653589793, 2.718281828459045, 1.4142135623730951, 1.7320508075688772)
GAMMA, N, W, H = -1.0, 2, 5, 7
HASHES = [bytes(range(32)), bytes((37 * i + 11) & 255 for i in range(32))]


def main():
    ctx = oracle.lib().ctx(KEY, GAMMA, N, W, H)
    out = [
        "# D, B and the LHCS_m records IR of two CHAINED frames, n = 2, w = 5, h = 7, gamma = -1.0,",
        "# key = (pi, e, sqrt 2, sqrt 3) as binary64; SURVEY.md 8(c) steps 2-7 and 10 (PAPER.md:35-43 Eq. 1, :55, :59).",
        "# Written by tests/golden/make_derive_tiny.py from oracle/ only.  Fields per frame:",
        "#   H <64 hex>   S <4 x 16 hex: base state before the frame, IEEE-754 bit patterns, big-endian digits>",
        "#   IR <2n x 4 x 16 hex>   D <3(h+w) x 4 hex, uint16 values>   B <3wh x 2 hex, HWC byte order>",
    ]
    for Hh in HASHES:
        S = ctx.state
        D, B, IR = ctx.derive(Hh, want_ir=True)
        out.append("H " + Hh.hex())
        out.append("S " + " ".join("%016x" % int(v.view("u8")) for v in S))
        out.append("IR " + " ".join("%016x" % int(v) for v in IR.ravel().view("u8")))
        out.append("D " + " ".join("%04x" % int(v) for v in D))
        out.append("B " + B.tobytes().hex())
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "derive_tiny.txt"), "w") as f:
        f.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
