"""CPU model of the exact-fp64 arithmetic the CUDA kernels use for moduli below 2^50 (
paper_2606_16359_b200/csrc/fenc_device.cuh: mulmod_dd, reduce_dd, the narrow and wide register rounds; fenc_elem.cu:
20-bit limbs accumulated by DFMA).  IEEE-754 binary64 with a correctly rounded fma is emulated with exact rationals, so
these tests check the REASONING behind the kernels' bit-exactness -- error-free product, quotient estimate within one,
value ranges of a round -- on the host, at the extremes of the admitted ranges.  No CUDA, no oracle import."""
import random
from fractions import Fraction

import pytest

MAGIC = 6755399441055744.0  # 1.5 * 2^52


def rn(x):  # exact rational -> nearest double (ties to even), what one IEEE operation returns
    return float(Fraction(x))


def fma(a, b, c):
    return rn(Fraction(a) * Fraction(b) + Fraction(c))


def mul(a, b):
    return rn(Fraction(a) * Fraction(b))


def add(a, b):
    return rn(Fraction(a) + Fraction(b))


def mulmod_dd(xd, c, cq, q):  # fenc_device.cuh
    h = mul(xd, c)
    l = fma(xd, c, -h)
    k = add(fma(xd, cq, MAGIC), -MAGIC)
    return add(fma(-k, q, h), l)


def reduce_dd(v, q, qinv):
    k = add(fma(v, qinv, MAGIC), -MAGIC)
    return fma(-k, q, v)


def primes_like(bits):  # odd moduli at both ends of a bit size (primality is irrelevant to the arithmetic)
    return [(1 << bits) - 1, (1 << bits) - 3 * (1 << 14) + 1, (1 << (bits - 1)) + 1 + (1 << 15)]


@pytest.mark.parametrize("bits,xmax_log2", [(30, 51), (40, 51), (45, 51), (50, 51)])
def test_twiddle_multiply_is_exact_and_within_q(bits, xmax_log2):
    rnd = random.Random(bits)
    for q in primes_like(bits):
        qd = float(q)
        for trial in range(400):
            c = rnd.randrange(1, q) if trial else q - 1
            cq = rn(Fraction(c) / Fraction(q))  # (double)(c / q), correctly rounded (the host rounds a long double: 1 ulp)
            lim = min(1 << xmax_log2, (1 << 51) * q // max(c, 1))  # the kernels keep |x c / q| below 2^51
            x = rnd.randrange(-lim + 1, lim) if trial > 2 else (lim - 1) * (1 if trial else -1)
            t = mulmod_dd(float(x), float(c), cq, qd)
            assert t == int(t) and abs(t) < q
            assert (int(t) - x * c) % q == 0


@pytest.mark.parametrize("bits", [30, 45, 50])
def test_reduce_is_centred(bits):
    rnd = random.Random(100 + bits)
    for q in primes_like(bits):
        qd, qinv = float(q), rn(Fraction(1) / Fraction(q))
        for _ in range(400):
            v = rnd.randrange(-8 * q + 8, 8 * q - 8)  # the largest magnitude an inverse wide round produces
            r = reduce_dd(float(v), qd, qinv)
            assert r == int(r) and (int(r) - v) % q == 0 and abs(r) <= q // 2 + 1


def _round(vals, tw, q, fwd, wide, first=True, last=True):
    """One radix-8 register round as tile_round_ct<F64, FIRST, LAST> runs it, on exact doubles.  first: the inputs are the
    unsigned words of the fill; otherwise the doubles the previous round of the same transform left in the tile.
    last: returns the unsigned lazy words every consumer reads; otherwise the doubles left for the next round."""
    qd, qinv = float(q), rn(Fraction(1) / Fraction(q))
    if first:
        x = [add(float(v), -qd) if wide else float(v) for v in vals]
    else:
        x = [float(v) for v in vals]
    done = 0
    for ss in range(3):
        s = 2 - ss if fwd else ss
        pre = wide and (done >= 2 if fwd else done >= 1)
        done += 1
        for k in range(8):
            if k & (1 << s):
                continue
            k2 = k | (1 << s)
            c = tw[s][k >> (s + 1)]
            cq = rn(Fraction(c) / Fraction(q))
            if fwd:
                y = reduce_dd(x[k2], qd, qinv) if pre else x[k2]
                assert abs(y) * c < (1 << 51) * q
                t = mulmod_dd(y, float(c), cq, qd)
                x[k], x[k2] = add(x[k], t), add(x[k], -t)
            else:
                d = add(x[k], -x[k2])
                x[k] = add(x[k], x[k2])
                if pre:
                    d = reduce_dd(d, qd, qinv)
                assert abs(d) * c < (1 << 51) * q
                x[k2] = mulmod_dd(d, float(c), cq, qd)
        assert all(abs(v) < 2 ** 53 and v == int(v) for v in x)
    red = wide or not fwd
    if not last:
        return [reduce_dd(v, qd, qinv) if red else v for v in x]
    out = [add(reduce_dd(v, qd, qinv), qd) if red else add(v, 16 * qd) for v in x]
    assert all(0 <= v < 2 ** 52 and v == int(v) for v in out)
    return [int(v) for v in out]


def _round_int(vals, tw, q, fwd):  # the textbook butterflies on integers
    x = list(vals)
    for ss in range(3):
        s = 2 - ss if fwd else ss
        for k in range(8):
            if k & (1 << s):
                continue
            k2 = k | (1 << s)
            c = tw[s][k >> (s + 1)]
            if fwd:
                t = x[k2] * c
                x[k], x[k2] = x[k] + t, x[k] - t
            else:
                x[k], x[k2] = x[k] + x[k2], (x[k] - x[k2]) * c
    return [v % q for v in x]


@pytest.mark.parametrize("bits,wide", [(40, False), (45, False), (50, True), (46, True)])
@pytest.mark.parametrize("fwd", [True, False])
def test_register_round_matches_integer_butterflies_and_keeps_its_ranges(bits, wide, fwd):
    rnd = random.Random(7 * bits + fwd)
    for q in primes_like(bits):
        for trial in range(60):
            tw = {2: [rnd.randrange(1, q)], 1: [rnd.randrange(1, q) for _ in range(2)], 0: [rnd.randrange(1, q) for _ in range(4)]}
            if wide or not fwd:
                hi = 2 * q  # contract at the start of a wide round and of every inverse round: [0, 2q]
            else:
                hi = 30 * q  # narrow forward rounds accept their own lazy outputs (up to 36q after five rounds)
            vals = [rnd.randrange(0, hi) for _ in range(8)] if trial else [hi - 1] * 4 + [0] * 4
            got = _round(vals, tw, q, fwd, wide)
            want = _round_int(vals, tw, q, fwd)
            assert [g % q for g in got] == want
            if wide or not fwd:
                assert all(0 <= g <= 2 * q for g in got)
            else:
                assert all(0 <= g < hi + 19 * q + 1 for g in got)  # moved by less than 3q in the round, then + 16q


@pytest.mark.parametrize("bits,wide", [(40, False), (45, False), (50, True), (46, True)])
@pytest.mark.parametrize("fwd", [True, False])
def test_three_rounds_chained_through_doubles_match_integer_butterflies(bits, wide, fwd):
    """The 8 stages of a pass as three register rounds (3 + 3 + 2 stages share one element group here: the point is the
    FORMAT between rounds): the first round converts from unsigned words, the tile holds doubles between rounds, the last
    round converts back.  Residues equal the integer butterflies', every intermediate stays an exact integer below 2^53,
    every multiplied operand inside the multiply's range (asserted in _round), the final words inside the consumers'
    contract ([0, 2q] where a round reduces, below 2^52 for narrow forward)."""
    rnd = random.Random(11 * bits + fwd)
    for q in primes_like(bits):
        for trial in range(40):
            hi = 2 * q if (wide or not fwd) else (1 << 50)  # narrow forward passes accept lazy inputs below 2^50
            vals = [rnd.randrange(0, hi) for _ in range(8)] if trial else [hi - 1] * 4 + [0] * 4
            tws = [{2: [rnd.randrange(1, q)], 1: [rnd.randrange(1, q) for _ in range(2)], 0: [rnd.randrange(1, q) for _ in range(4)]}
                   for _ in range(3)]
            x, want = list(vals), list(vals)
            for r in range(3):
                x = _round(x, tws[r], q, fwd, wide, first=(r == 0), last=(r == 2))
                want = _round_int(want, tws[r], q, fwd)
            assert [g % q for g in x] == want
            if wide or not fwd:
                assert all(0 <= g <= 2 * q for g in x)


def test_mac_limb_sums_stay_exact():
    """fenc_elem.cu MODE 2: x, w < 2^40 split in 20-bit limbs; 2047 products per partial sum plus a folded residue."""
    m = (1 << 20) - 1
    a0 = (1 << 40) + 2047 * m * m  # folded residue (< q < 2^40) + 2047 maximal products
    a1 = 2047 * 2 * m * m
    assert a0 < 2 ** 53 and a1 < 2 ** 53
    acc = 0.0
    for _ in range(2047):  # worst case accumulates without rounding
        acc = fma(float(m), float(m), acc)
    assert acc == 2047 * m * m
