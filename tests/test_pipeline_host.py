"""CPU-only checks of the Python-side host logic of the product (no GPU, no library call): the pooling order used by
pipeline.Pipeline equals the oracle's independent statement of it, and the exact rounding helper matches the oracle's."""
from fractions import Fraction

from oracle import ckks as ck
from oracle import network as nw
from paper_2606_16359_b200.pipeline import POLY3, Pipeline, _round_half_up


def test_pool_order_matches_oracle_statement():
    for n_ct, S in ((16, 4), (96, 4), (24, 2), (64, 2), (128, 8)):
        assert Pipeline.pool_order(n_ct, S) == nw.pool_order(n_ct, S)
        order = Pipeline.pool_order(n_ct, S)
        assert sorted(order) == list(range(n_ct))  # a permutation: every fragment is summed exactly once


def test_round_half_up_and_coefficients():
    for x in (Fraction(1, 2), Fraction(-1, 2), Fraction(3, 2), Fraction(-7, 3), Fraction(197, 1000) * 2 ** 100):
        assert _round_half_up(x) == ck.round_half_up(x)
    assert _round_half_up(Fraction(1, 2)) == 1 and _round_half_up(Fraction(-1, 2)) == 0
    assert tuple(POLY3) == tuple(ck.POLY3)
