"""Writes tests/golden/worked_vector.txt from exact rational arithmetic (tests/exact.py).

Calls neither oracle/ nor the CUDA path: every value is Eq. 4 evaluated with
python Fractions and explicit IEEE roundings, so the file is an independent pin for both.
Run from the repo root:  python tests/golden/derive_worked_vector.py
"""
import os
import sys
from fractions import Fraction

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
import exact  # noqa: E402

X = [1.0, -0.5, 0.25, 2.0]
W = [[1, 0, -1, 1], [-1, -1, 0, 1]]
BETA_BITS = 0x3D4CCCCD  # 0.05f


def bf16_bits(v):
    return exact.fraction_to_bf16_bits(Fraction(v))


def f32_from_bits(b):
    e = (b >> 23) & 0xFF
    m = b & 0x7FFFFF
    return (1 + Fraction(m, 1 << 23)) * Fraction(2) ** (e - 127)


def main():
    xb = [bf16_bits(v) for v in X]
    r = exact.linear([xb], W, f32_from_bits(BETA_BITS))
    lines = [
        "# Worked vector for Eq. 4 of arxiv/paper_2606_08094 (PAPER.md lines 75-80, Section III-D).",
        "# The paper prints no numeric example; these values are Eq. 4 evaluated in exact rational",
        "# arithmetic with explicit fp32/bf16 roundings by tests/golden/derive_worked_vector.py",
        "# (independent of oracle/ and of the CUDA path).  63.5 -> 64 is a round-half-to-even case.",
        "# Real-valued x.W^T.beta = [0.1375, 0.075].",
        "x_bf16_bits " + " ".join("0x%04X" % b for b in xb),
        "w_row0 " + " ".join(str(v) for v in W[0]),
        "w_row1 " + " ".join(str(v) for v in W[1]),
        "beta_f32_bits 0x%08X" % BETA_BITS,
        "alpha_f32_bits 0x%08X" % exact.fraction_to_f32_bits(r["alpha"][0]),
        "a " + " ".join(str(v) for v in r["a"][0]),
        "acc " + " ".join(str(v) for v in r["acc"][0]),
        "y_f32_bits " + " ".join("0x%08X" % exact.fraction_to_f32_bits(v) for v in r["y32"][0]),
        "y_bf16_bits " + " ".join("0x%04X" % exact.fraction_to_bf16_bits(v) for v in r["ybf16"][0]),
    ]
    with open(os.path.join(HERE, "worked_vector.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
