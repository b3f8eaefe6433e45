"""Writes ns_scalar_sequence.txt rows (exact rationals of Eq. 9's scalar recurrence). Stdlib only."""
from fractions import Fraction as F

if __name__ == "__main__":
    x = F(1, 2)
    for k in range(4):
        print(k, x.numerator, x.denominator)
        x = F(1, 2) * x * (3 - x * x)
