"""Writes tests/golden/bb_moments.txt: EXACT coordinate moments for the background block.

With mask = NULL the B-B block of the normal matrix is (SURVEY.md §8(c) pin P4)

    A[B(p,q), B(p',q')] = sum_{x,y} xi(x)^(p+p') eta(y)^(q+q') = mx(p+p'; W) * my(q+q'; H),
    mx(a; W) = sum_{x=0}^{W-1} ((2x+1-W)/W)^a        (xi as in SURVEY §8.0 / DESIGN.md A3)

computed here in exact rational arithmetic (fractions.Fraction); this script calls nothing from
oracle/ or from the CUDA path.  Closed forms it reproduces: mx(0)=W, mx(odd)=0,
mx(2)=(W^2-1)/(3W).  Run:  python tests/golden/make_bb_moments.py
"""
from fractions import Fraction
import os

SIZES = [16, 64, 256, 1024, 2048, 4096]
MAXPOW = 6


def moment(a, n):
    return sum(Fraction(2 * x + 1 - n, n) ** a for x in range(n))


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "bb_moments.txt")
    with open(out, "w") as f:
        f.write("# exact sum_x ((2x+1-n)/n)^a ; columns: n a numerator denominator float_repr\n")
        f.write("# source: closed form / exact rational arithmetic, SURVEY.md 8(c) pin P4\n")
        for n in SIZES:
            for a in range(MAXPOW + 1):
                m = moment(a, n)
                if a == 2:
                    assert m == Fraction(n * n - 1, 3 * n)
                if a % 2 == 1:
                    assert m == 0
                f.write(f"{n} {a} {m.numerator} {m.denominator} {float(m)!r}\n")


if __name__ == "__main__":
    main()
