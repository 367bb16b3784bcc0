"""Writes tests/golden/appendixA_worked_examples.txt from the closed forms the paper PRINTS for its worked
p_z example: Eq. (A7) and Eq. (A8).  Uses `math` only — neither the oracle
nor the CUDA path is involved, so the fixture is the paper's statement evaluated at a few parameter sets.

    python tests/golden/make_appendixA_golden.py
"""
import math
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def xi_A7(sigma):            # Eq. (A7): xi = (1/2 pi^{3/2} sigma^5)^{-1/2}
    return (0.5 * math.pi ** 1.5 * sigma ** 5) ** -0.5


def N_A8(d0, d1, s0, s1):    # Eq. (A8): N = [d0^2 + d1^2 + 2 d0 d1 (2 s0 s1 / (s0^2 + s1^2))^{5/2}]^{-1/2}
    return (d0 * d0 + d1 * d1 + 2.0 * d0 * d1 * (2.0 * s0 * s1 / (s0 * s0 + s1 * s1)) ** 2.5) ** -0.5


def main():
    lines = ["# Worked p_z normalisation examples of arxiv 2512.18010, Appendix A.",
             "# A7 rows: 'A7 sigma xi'           xi from Eq. (A7), PAPER.md:649",
             "# A8 rows: 'A8 d0 d1 sigma0 sigma1 N'  N from Eq. (A8), PAPER.md:654",
             "# Written by tests/golden/make_appendixA_golden.py (math only; no oracle, no CUDA)."]
    for s in (1.0, 0.5, 2.0, 0.13, 3.7):
        lines.append(f"A7 {s!r} {xi_A7(s)!r}")
    for (d0, d1, s0, s1) in ((1.0, 1.0, 1.0, 1.0), (0.3, 0.9, 0.5, 1.5), (0.7, 0.2, 2.0, 0.25), (1.0, -0.4, 0.8, 1.1)):
        lines.append(f"A8 {d0!r} {d1!r} {s0!r} {s1!r} {N_A8(d0, d1, s0, s1)!r}")
    with open(os.path.join(HERE, "appendixA_worked_examples.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
