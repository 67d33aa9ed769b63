"""Writes the golden fixtures from the paper's printed formulas with exact / 50-digit arithmetic.
Imports nothing from oracle/ or the CUDA package."""
import os
from decimal import Decimal, getcontext
from fractions import Fraction

HERE = os.path.dirname(os.path.abspath(__file__))


def k_eq10(Y: Fraction) -> Fraction:          # PAPER.md:82-85, Eq. 10 (0 < Y < 1 branch)
    return 10 * Y ** 6 - 15 * Y ** 8 + 6 * Y ** 10


def main():
    with open(os.path.join(HERE, "k_eq10.txt"), "w") as f:
        f.write("# PAPER.md:82-85 Eq. 10: K = 10Y^6 - 15Y^8 + 6Y^10, 0<Y<1.  columns: Y_num Y_den K_num K_den\n")
        for num, den in [(1, 8), (1, 4), (3, 8), (1, 2), (5, 8), (3, 4), (7, 8), (1, 3), (2, 3), (1, 10), (9, 10)]:
            k = k_eq10(Fraction(num, den))
            f.write(f"{num} {den} {k.numerator} {k.denominator}\n")
    getcontext().prec = 50
    with open(os.path.join(HERE, "rb_eq5.txt"), "w") as f:
        f.write("# PAPER.md:59 Eq. 5: r_b = b/2 + sqrt(b^2/4 + sqrt(3 B2/a_err)).  columns: b_max B2 a_err r_b\n")
        for b, B2, aerr in [("1", "1", "0.00390625"), ("0.5", "0.03125", "0.00390625"), ("2", "0", "0.00390625"),
                            ("0", "0", "0.00390625"), ("0.25", "1e-6", "0.001"), ("3", "10", "0.125")]:
            bd, Bd, ad = Decimal(b), Decimal(B2), Decimal(aerr)
            rb = bd / 2 + (bd * bd / 4 + (3 * Bd / ad).sqrt()).sqrt()
            f.write(f"{b} {B2} {aerr} {rb:.30f}\n")


if __name__ == "__main__":
    main()
