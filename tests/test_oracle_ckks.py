"""Pins for oracle/ckks.py + oracle/fenc_oracle.c (CPU only).

Each test checks the oracle against something other than itself: the schoolbook definition,
closed forms, exact big-integer characterisations computed here with Python integers, textbook
invariants, and second-implementation hashes (tests/golden/)."""
import decimal
import hashlib
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import ckks as ck

GOLD = os.path.join(os.path.dirname(__file__), "golden")
lib = ck._lib
P_ = ck._p


@pytest.fixture(scope="module")
def toy():
    # N = 64, 4 ciphertext primes of 30 bits, 2 special primes of 31 bits, dlen = 2 (beta = 2)
    return ck.Params(6, 4, 30, 2, 31, 2, 25)


@pytest.fixture(scope="module")
def toy_keys(toy):
    return ck.keygen(toy, 42, [1, 2, 5, toy.n - 5, 17], want_relin=True)


# ------------------------------------------------------------------ parameters
def test_prime_chains_match_second_implementation():
    for line in open(os.path.join(GOLD, "prime_chain_hashes.txt")):
        if line.startswith("#") or not line.strip():
            continue
        logN, nq, qb, npp, pb, sha, q0, p0 = line.split()
        q = ck.find_primes(int(logN), int(qb), int(nq))
        p = ck.find_primes(int(logN), int(pb), int(npp))
        assert q[0] == int(q0) and p[0] == int(p0)
        assert hashlib.sha256(",".join(map(str, q + p)).encode()).hexdigest()[:16] == sha


def test_prime_rule_independent_check():
    # descending, = 1 mod 2N, below the bound, prime by trial division, and nothing skipped in between
    logN, bits = 6, 30
    q = ck.find_primes(logN, bits, 4)
    twoN = 2 << logN

    def trial(n):
        return n > 1 and all(n % d for d in range(2, math.isqrt(n) + 1))
    assert all(x < 2 ** bits and x % twoN == 1 and trial(x) for x in q)
    assert q == sorted(q, reverse=True)
    top = (2 ** bits - 1) // twoN * twoN + 1
    cands = [c for c in range(top, q[-1] - 1, -twoN) if c < 2 ** bits and trial(c)]
    assert cands == q


def test_psi_is_primitive_2N_root(toy):
    for m, psi in zip(toy.mod, toy.psi):
        assert pow(psi, toy.N, m) == m - 1 and pow(psi, 2 * toy.N, m) == 1


# ------------------------------------------------------------------ NTT (R2.1)
@pytest.mark.parametrize("logN", [2, 3, 4, 5, 6])
def test_ntt_product_equals_schoolbook(logN):
    N = 1 << logN
    rng = np.random.default_rng(logN)
    for q in ck.find_primes(logN, 40, 2) + ck.find_primes(logN, 60, 1):
        psi = ck.find_psi(q, N)
        a = rng.integers(0, q, N, dtype=np.uint64)
        b = rng.integers(0, q, N, dtype=np.uint64)
        c1 = np.zeros(N, dtype=np.uint64)
        c2 = np.zeros(N, dtype=np.uint64)
        lib.orc_polymul(N, q, psi, P_(a), P_(b), P_(c1))
        lib.orc_schoolbook(N, q, P_(a), P_(b), P_(c2))
        assert np.array_equal(c1, c2)
        # independent of C: Python-integer schoolbook
        ai, bi = a.tolist(), b.tolist()
        ref = [0] * N
        for i in range(N):
            for j in range(N):
                k = i + j
                if k < N:
                    ref[k] += ai[i] * bi[j]
                else:
                    ref[k - N] -= ai[i] * bi[j]
        assert [x % q for x in ref] == c1.tolist()


def test_ntt_is_evaluation_at_odd_powers():
    # NTT(a)[e] = a(psi^(2e+1)): check on a random polynomial by Horner in Python integers
    N, q = 32, ck.find_primes(5, 40, 1)[0]
    psi = ck.find_psi(q, N)
    a = np.random.default_rng(3).integers(0, q, N, dtype=np.uint64)
    f = a.copy()
    lib.orc_ntt(N, q, psi, P_(f))
    for e in range(N):
        x = pow(psi, 2 * e + 1, q)
        acc = 0
        for c in reversed(a.tolist()):
            acc = (acc * x + c) % q
        assert acc == int(f[e])


def test_ntt_round_trip_full_size():
    N, q = 1 << 13, ck.find_primes(13, 40, 1)[0]
    psi = ck.find_psi(q, N)
    a = np.random.default_rng(5).integers(0, q, N, dtype=np.uint64)
    f = a.copy()
    lib.orc_ntt(N, q, psi, P_(f))
    assert not np.array_equal(f, a)
    lib.orc_intt(N, q, psi, P_(f))
    assert np.array_equal(f, a)


# ------------------------------------------------------------------ automorphism (R2.7)
def test_automorphism_on_unit_vectors_and_inverse():
    N, q = 16, 97
    for g in (5, 25, 3, 31):
        for i in range(N):
            e = np.zeros(N, dtype=np.uint64)
            e[i] = 1
            out = np.zeros(N, dtype=np.uint64)
            lib.orc_automorph(N, q, g, P_(e), P_(out))
            k = i * g % (2 * N)
            exp = np.zeros(N, dtype=np.uint64)
            exp[k % N] = 1 if k < N else q - 1  # sigma_g(X^i) = +-X^(ig mod N)
            assert np.array_equal(out, exp)
        ginv = pow(g, -1, 2 * N)
        a = np.random.default_rng(g).integers(0, q, N, dtype=np.uint64)
        b = np.zeros(N, dtype=np.uint64)
        c = np.zeros(N, dtype=np.uint64)
        lib.orc_automorph(N, q, g, P_(a), P_(b))
        lib.orc_automorph(N, q, ginv, P_(b), P_(c))
        assert np.array_equal(a, c)


# ------------------------------------------------------------------ encode / decode (R2.2)
def test_encode_closed_forms():
    N, s = 64, 2 ** 30
    m = ck.encode_coeffs(np.full(N // 2, 0.75), N, s)
    exp = np.zeros(N, dtype=np.int64)
    exp[0] = round(0.75 * s)
    assert np.array_equal(m, exp)  # constant vector <-> constant polynomial
    mono = np.zeros(N, dtype=np.int64)
    mono[N // 2] = s
    z = ck.decode_coeffs(mono, N, s)  # s X^(N/2) decodes to (i, ..., i)
    assert np.allclose(z, 1j * np.ones(N // 2), atol=1e-12)


@pytest.mark.parametrize("N", [16, 64, 256])
def test_encode_fft_equals_definition_and_round_trip(N):
    rng = np.random.default_rng(N)
    z = rng.uniform(-1, 1, N // 2) + 1j * rng.uniform(-1, 1, N // 2)
    s = 2 ** 40
    a, b = ck.encode_coeffs(z, N, s), ck.encode_coeffs_def(z, N, s)
    assert np.abs(a - b).max() <= 1
    assert np.abs(ck.decode_coeffs(a, N, s) - z).max() < 1e-9


def test_slots_multiply_and_rotate():
    """decode is a ring homomorphism onto slot-wise products, and sigma_{5^r} is a LEFT cyclic shift (A8)."""
    N, q = 64, ck.find_primes(6, 60, 1)[0]
    psi = ck.find_psi(q, N)
    rng = np.random.default_rng(9)
    za, zb = rng.uniform(-1, 1, N // 2), rng.uniform(-1, 1, N // 2)
    s = 2 ** 25
    ma, mb = ck.encode_coeffs(za, N, s), ck.encode_coeffs(zb, N, s)
    ua = np.where(ma >= 0, ma, ma + q).astype(np.uint64)
    ub = np.where(mb >= 0, mb, mb + q).astype(np.uint64)
    c = np.zeros(N, dtype=np.uint64)
    lib.orc_polymul(N, q, psi, P_(ua), P_(ub), P_(c))
    cc = [int(x) - q if int(x) > q // 2 else int(x) for x in c]
    assert np.abs(ck.decode_coeffs(cc, N, s * s) - za * zb).max() < 1e-5
    for r in (1, 3, 7):
        out = np.zeros(N, dtype=np.uint64)
        lib.orc_automorph(N, q, pow(5, r, 2 * N), P_(ua), P_(out))
        oc = [int(x) - q if int(x) > q // 2 else int(x) for x in out]
        assert np.abs(ck.decode_coeffs(oc, N, s) - np.roll(za, -r)).max() < 1e-6


# ------------------------------------------------------------------ randomness (R2.3)
def test_mix64_is_splitmix64():
    # published SplitMix64 test vector: seed 1234567 -> first outputs
    assert int(ck.draws(1234567, [0, 1, 2])[0]) == 6457827717110365317
    assert int(ck.draws(1234567, [0, 1, 2])[1]) == 3203168211198807973
    assert ck.mix64((1234567 + ck._GAMMA) & ck._M64) == 6457827717110365317


def test_gauss_cdt_against_decimal_arithmetic():
    decimal.getcontext().prec = 80
    sig = decimal.Decimal("3.2")
    w = [(-(decimal.Decimal(x * x)) / (2 * sig * sig)).exp() for x in range(20)]
    tot = w[0] + 2 * sum(w[1:])
    acc = decimal.Decimal(0)
    for x in range(19):
        acc += w[x] if x == 0 else 2 * w[x]
        assert int(acc / tot * (1 << 64)) == ck.GAUSS_CDT[x]


def test_sampler_statistics():
    N = 1 << 15
    e = ck.sample_gauss(ck.stream_key(1, ck.PURPOSE_ENC_E), N)
    assert abs(e.mean()) < 0.1 and abs(e.var() - 10.24) < 0.3 and np.abs(e).max() <= 19
    s = ck.sample_ternary(ck.stream_key(1, ck.PURPOSE_SECRET), N)
    assert set(np.unique(s)) == {-1, 0, 1} and abs((s == 0).mean() - 1 / 3) < 0.02
    q = 1099511480321
    u = ck.sample_uniform(ck.stream_key(1, ck.PURPOSE_ENC_A, 0), N, q)
    assert u.max() < q and abs(u.astype(np.float64).mean() / q - 0.5) < 0.01
    # streams differ by purpose / index
    assert ck.stream_key(1, 2, 3, 0, 1) != ck.stream_key(1, 2, 3, 1, 0)


def test_uniform_rejection_path():
    # a prime far below its power of two exercises the redraw path; result must be the first accepted draw
    q, key, N = 769, 99, 512
    u = ck.sample_uniform(key, N, q)
    for i in range(0, N, 37):
        a = 0
        while True:
            x = ck.mix64((key + (i * 64 + a + 1) * ck._GAMMA) & ck._M64) & 1023
            if x < q:
                break
            a += 1
        assert int(u[i]) == x


# ------------------------------------------------------------------ ModUp / ModDown / Rescale (R2.6, R2.8)
def _crt(residues, mods):
    Q = math.prod(mods)
    v = 0
    for r, m in zip(residues, mods):
        Qh = Q // m
        v += int(r) * Qh * pow(Qh, -1, m)
    return v % Q


def test_modup_exact_characterisation(toy):
    P, N, L = toy, toy.N, 3  # L = 3: digit 0 = {q0,q1}, digit 1 = {q2} (short last digit)
    rng = np.random.default_rng(1)
    d = np.stack([rng.integers(0, P.q[t], N, dtype=np.uint64) for t in range(L)])
    for j in range(2):
        up = np.zeros((L + P.np_, N), dtype=np.uint64)
        lib.orc_modup(P._h, L, j, P_(d), P_(up))
        dig = [t for t in P.digit(j) if t < L]
        Qj = math.prod(P.q[t] for t in dig)
        tmods = P.q[:L] + P.p
        for n in range(N):
            x = _crt([d[t, n] for t in dig], [P.q[t] for t in dig])
            # U = sum y_i (Q_j/q_i), y_i = [d (Q_j/q_i)^-1]_{q_i}:  U = d (mod Q_j), 0 <= U < |D_j| Q_j
            U = sum((int(d[t, n]) * pow(Qj // P.q[t], -1, P.q[t]) % P.q[t]) * (Qj // P.q[t]) for t in dig)
            assert U % Qj == x and 0 <= U < len(dig) * Qj
            for row, t in enumerate(tmods):
                assert int(up[row, n]) == U % t
            for t in dig:
                assert up[t, n] == d[t, n]


def test_moddown_exact_characterisation(toy):
    P, N, L = toy, toy.N, 3
    rng = np.random.default_rng(2)
    mods = P.q[:L] + P.p
    acc = np.stack([rng.integers(0, m, N, dtype=np.uint64) for m in mods])
    out = np.zeros((L, N), dtype=np.uint64)
    lib.orc_moddown(P._h, L, P_(acc), P_(out))
    for n in range(N):
        A = _crt([acc[r, n] for r in range(L + P.np_)], mods)  # any integer representing acc
        V = sum((int(acc[L + i, n]) * pow(P.P // P.p[i], -1, P.p[i]) % P.p[i]) * (P.P // P.p[i]) for i in range(P.np_))
        assert (A - V) % P.P == 0 and 0 <= V < P.np_ * P.P
        for t in range(L):
            assert int(out[t, n]) == ((A - V) // P.P) % P.q[t]


def test_rescale_is_exact_floor(toy):
    P, N, L = toy, toy.N, 4
    rng = np.random.default_rng(3)
    c = np.stack([rng.integers(0, P.q[t], N, dtype=np.uint64) for t in range(L)])
    out = np.zeros((L - 1, N), dtype=np.uint64)
    lib.orc_rescale(P._h, L, P_(c), P_(out))
    for n in range(N):
        C = _crt(c[:, n], P.q[:L])
        for t in range(L - 1):
            assert int(out[t, n]) == (C // P.q[L - 1]) % P.q[t]


# ------------------------------------------------------------------ keys, key switch, rotation
def _centre(v, q):
    return [int(x) - q if int(x) > q // 2 else int(x) for x in v]


def test_switching_key_equation(toy, toy_keys):
    """b + a s - f s' = e: small (|e| <= 19), the same e on every limb of a digit."""
    P = toy
    b, a = toy_keys.evk[5]
    g = P.galois(5)
    for j in range(P.beta_max):
        es = []
        for t in range(len(P.mod)):
            q = P.mod[t]
            srot = np.zeros(P.N, dtype=np.uint64)
            lib.orc_automorph(P.N, q, g, P_(toy_keys.s_rns[t].copy()), P_(srot))
            as_ = ck._polymul(P, t, a[j, t], toy_keys.s_rns[t])
            f = P.P % q if t in P.digit(j) else 0
            v = (b[j, t].astype(object) + as_.astype(object) - f * srot.astype(object)) % q
            es.append(_centre(v, q))
        assert all(e == es[0] for e in es) and max(abs(x) for x in es[0]) <= 19


def test_keyswitch_noise_bound(toy, toy_keys):
    P, L = toy, 4
    rng = np.random.default_rng(4)
    d = np.stack([rng.integers(0, P.q[t], P.N, dtype=np.uint64) for t in range(L)])
    k0, k1 = ck.keyswitch(P, L, d, toy_keys.evk[ck.RELIN_KEY_ID])
    # decrypt_s(KS(d)) - d s^2 must be small
    s2 = np.stack([ck._polymul(P, t, toy_keys.s_rns[t], toy_keys.s_rns[t]) for t in range(L)])
    diff = np.zeros((L, P.N), dtype=np.uint64)
    for t in range(L):
        q = np.uint64(P.q[t])
        lhs = (k0[t] + ck._polymul(P, t, k1[t], toy_keys.s_rns[t])) % q
        rhs = ck._polymul(P, t, d[t], s2[t])
        diff[t] = (lhs + q - rhs) % q
    err = ck.crt_centre(P, diff, L)
    Qj = max(math.prod(P.q[t] for t in P.digit(j)) for j in range(P.beta_max))
    bound = 8 * (P.beta_max * math.sqrt(P.N) * 3.2 * Qj / (P.P * math.sqrt(12)) * math.sqrt(P.N) + P.np_ * math.sqrt(P.N) + P.N)
    assert max(abs(e) for e in err) < bound


def test_rotation_is_left_cyclic_shift(toy, toy_keys):
    P = toy
    rng = np.random.default_rng(5)
    z = rng.uniform(-1, 1, P.n)
    ct = ck.encrypt(P, toy_keys, ck.encode(P, z, P.nq), 77)
    assert np.abs(ck.decrypt_decode(P, toy_keys, ct) - z).max() < 1e-5
    for r in (1, 2, 5, 17):
        d = ck.decrypt_decode(P, toy_keys, ck.rotate(P, toy_keys, ct, r))
        assert np.abs(d - np.roll(z, -r)).max() < 1e-4
        assert np.abs(d - np.roll(z, r)).max() > 0.1
    back = ck.rotate(P, toy_keys, ck.rotate(P, toy_keys, ct, 5), P.n - 5)
    assert np.abs(ck.decrypt_decode(P, toy_keys, back) - z).max() < 1e-4
    # at a lower level (short last digit: L = 3, dlen = 2)
    ct3 = ck.encrypt(P, toy_keys, ck.encode(P, z, 3), 78)
    assert np.abs(ck.decrypt_decode(P, toy_keys, ck.rotate(P, toy_keys, ct3, 2)) - np.roll(z, -2)).max() < 1e-4


def test_square_sum_relin_is_sum_of_squares(toy, toy_keys):
    """R2.12c: the tensor products of several ciphertexts added before ONE relinearisation decrypt to the sum of the
    squared slot vectors; with one ciphertext the limbs are square_relin's; with four they are not the sum of four
    square_relin results (one key-switch noise instead of four), but decrypt to the same values."""
    P = toy
    rng = np.random.default_rng(31)
    zs = [rng.uniform(-1, 1, P.n) for _ in range(4)]
    cts = [ck.encrypt(P, toy_keys, ck.encode(P, z, P.nq), 200 + i) for i, z in enumerate(zs)]
    one = ck.square_sum_relin(P, toy_keys, cts[:1])
    assert np.array_equal(one.c, ck.square_relin(P, toy_keys, cts[0]).c) and one.L == P.nq - 1
    four = ck.square_sum_relin(P, toy_keys, cts)
    assert four.L == P.nq - 1 and four.scale == one.scale
    want = sum(z * z for z in zs)
    assert np.abs(ck.decrypt_decode(P, toy_keys, four).real - want).max() < 1e-3
    eager = ck.square_relin(P, toy_keys, cts[0])
    for c in cts[1:]:
        eager = ck.add(P, eager, ck.square_relin(P, toy_keys, c))
    assert not np.array_equal(eager.c, four.c)
    assert np.abs(ck.decrypt_decode(P, toy_keys, eager).real - ck.decrypt_decode(P, toy_keys, four).real).max() < 1e-3
    two = ck.square_sum_relin(P, toy_keys, cts[:2])
    assert np.abs(ck.decrypt_decode(P, toy_keys, two).real - (zs[0] ** 2 + zs[1] ** 2)).max() < 1e-3


def test_hoisted_rotation_decrypts_like_rotation(toy, toy_keys):
    """R2.7b: the hoisted form (ModUp of the unrotated c1, automorphism on the extended digits) is the same LEFT cyclic
    shift with key-switch noise of the same size: the two decryptions differ by a small integer polynomial (the
    ModDown of multiples of Q_j times the key), far below the scale, while the limbs themselves differ."""
    P = toy
    rng = np.random.default_rng(15)
    z = rng.uniform(-1, 1, P.n)
    for L in (P.nq, 3):  # top level, and a short last digit
        ct = ck.encrypt(P, toy_keys, ck.encode(P, z, L), 90 + L)
        for r in (1, 2, 5, 17):
            h, p = ck.rotate_hoisted(P, toy_keys, ct, r), ck.rotate(P, toy_keys, ct, r)
            d = ck.decrypt_decode(P, toy_keys, h)
            assert np.abs(d - np.roll(z, -r)).max() < 1e-4
            assert np.abs(d - np.roll(z, r)).max() > 0.1
            assert not np.array_equal(h.c, p.c)
            mh, mp = ck.decrypt_coeffs(P, toy_keys, h), ck.decrypt_coeffs(P, toy_keys, p)
            diff = max(abs(int(a) - int(b)) for a, b in zip(mh, mp))
            assert diff < 2 ** 10  # measured about 25; both carry rounding + e-terms of a few bits times sqrt(N); the scale is 2^25 and more
    same = ck.rotate_hoisted(P, toy_keys, ct, 0)
    assert np.array_equal(same.c, ct.c)


def test_pmult_rescale_and_square(toy, toy_keys):
    P = toy
    rng = np.random.default_rng(6)
    z, w = rng.uniform(-1, 1, P.n), rng.uniform(-1, 1, P.n)
    ct = ck.encrypt(P, toy_keys, ck.encode(P, z, P.nq), 79)
    pw = ck.encode(P, w, P.nq, P.q[P.nq - 1])
    out = ck.rescale(P, ck.pmult(P, ct, pw))
    assert out.L == P.nq - 1 and out.scale == P.scale  # s_w = q_{L-1} keeps the scale exactly (A14)
    assert np.abs(ck.decrypt_decode(P, toy_keys, out) - z * w).max() < 1e-4
    sq = ck.square_relin(P, toy_keys, ct)
    assert sq.scale == P.scale * P.scale / P.q[P.nq - 1]
    assert np.abs(ck.decrypt_decode(P, toy_keys, sq) - z * z).max() < 1e-4


def test_literal_dnum1_is_numerically_unusable():
    """A1: with one digit (Q_j = Q >> P) the rotation noise swamps the message; dlen = 1 is fine."""
    z = np.random.default_rng(7).uniform(-1, 1, 256)
    errs = []
    for dlen in (3, 1):
        P = ck.Params(9, 3, 40, 1, 60, 1, 40, dlen=dlen)
        keys = ck.keygen(P, 1, [3])
        ct = ck.encrypt(P, keys, ck.encode(P, z, 3), 2)
        errs.append(np.abs(ck.decrypt_decode(P, keys, ck.rotate(P, keys, ct, 3)) - np.roll(z, -3)).max())
    assert errs[0] > 1e3 and errs[1] < 1e-6
