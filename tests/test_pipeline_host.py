"""CPU-only checks of the Python-side host logic of the product (no GPU, no library call): the exact rounding helper matches the oracle's
(the pooling order lives in the library, fenc_sum_pool, and is compared with the oracle's on the GPU)."""
from fractions import Fraction

from oracle import ckks as ck
from paper_2606_16359_b200.pipeline import POLY3, _round_half_up


def test_round_half_up_and_coefficients():
    for x in (Fraction(1, 2), Fraction(-1, 2), Fraction(3, 2), Fraction(-7, 3), Fraction(197, 1000) * 2 ** 100):
        assert _round_half_up(x) == ck.round_half_up(x)
    assert _round_half_up(Fraction(1, 2)) == 1 and _round_half_up(Fraction(-1, 2)) == 0
    assert tuple(POLY3) == tuple(ck.POLY3)
