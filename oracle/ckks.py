"""RNS-CKKS oracle (CPU, slow, plain).  TEST INFRASTRUCTURE ONLY -- see oracle/__init__.py.

The paper names the primitives only (Add, PMult, CMult, Rot = automorphism +
key switch (Eq. 1), Rescale); their RNS form is "standard RNS-CKKS with hybrid key switching"
fixed by the readings R2.1-R2.8 of DESIGN.md section 4.  N-length integer work is done by
oracle/fenc_oracle.c (coefficient domain, canonical residues); structure, randomness, encoding
and exact scale bookkeeping are here, in Python integers / numpy / fractions.

Every ciphertext / plaintext / key polynomial is stored in the COEFFICIENT domain.
"""
import ctypes
import math
from fractions import Fraction

import numpy as np

from . import build as _build

_lib = ctypes.CDLL(_build.build())
_u64p = ctypes.POINTER(ctypes.c_uint64)
_i64p = ctypes.POINTER(ctypes.c_int64)


def _p(a):
    assert a.dtype == np.uint64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_u64p)


_lib.orc_params_new.restype = ctypes.c_void_p
_lib.orc_params_new.argtypes = [ctypes.c_size_t, ctypes.c_int, _u64p, _u64p, ctypes.c_int, _u64p, _u64p, ctypes.c_int]
_lib.orc_params_free.argtypes = [ctypes.c_void_p]
for _name, _args in {
    "orc_ntt": [ctypes.c_size_t, ctypes.c_uint64, ctypes.c_uint64, _u64p],
    "orc_intt": [ctypes.c_size_t, ctypes.c_uint64, ctypes.c_uint64, _u64p],
    "orc_polymul": [ctypes.c_size_t, ctypes.c_uint64, ctypes.c_uint64, _u64p, _u64p, _u64p],
    "orc_schoolbook": [ctypes.c_size_t, ctypes.c_uint64, _u64p, _u64p, _u64p],
    "orc_automorph": [ctypes.c_size_t, ctypes.c_uint64, ctypes.c_uint64, _u64p, _u64p],
    "orc_modup": [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, _u64p, _u64p],
    "orc_moddown": [ctypes.c_void_p, ctypes.c_int, _u64p, _u64p],
    "orc_keyswitch": [ctypes.c_void_p, ctypes.c_int, _u64p, _u64p, _u64p, _u64p, _u64p],
    "orc_rotate": [ctypes.c_void_p, ctypes.c_int, ctypes.c_uint64, _u64p, _u64p, _u64p, _u64p],
    "orc_rotate_hoisted": [ctypes.c_void_p, ctypes.c_int, ctypes.c_uint64, _u64p, _u64p, _u64p, _u64p],
    "orc_add": [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, _u64p, _u64p, _u64p],
    "orc_pmult_acc": [ctypes.c_void_p, ctypes.c_int, _u64p, _u64p, _u64p],
    "orc_polymul_rns": [ctypes.c_void_p, ctypes.c_int, _u64p, _u64p, _u64p],
    "orc_rescale": [ctypes.c_void_p, ctypes.c_int, _u64p, _u64p],
    "orc_mul_scalar": [ctypes.c_void_p, ctypes.c_int, _u64p, _u64p, _u64p],
    "orc_reduce_signed": [ctypes.c_void_p, ctypes.c_int, _i64p, _u64p],
}.items():
    getattr(_lib, _name).argtypes = _args
    getattr(_lib, _name).restype = None


# --------------------------------------------------------------------------- primes (R 8(c)-1)
def is_prime(n: int) -> bool:
    """Deterministic Miller-Rabin for n < 2^64 (bases 2..37)."""
    if n < 2:
        return False
    small = (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37)
    for p in small:
        if n % p == 0:
            return n == p
    d, s = n - 1, 0
    while d % 2 == 0:
        d //= 2
        s += 1
    for a in small:
        x = pow(a, d, n)
        if x in (1, n - 1):
            continue
        for _ in range(s - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def find_primes(logN: int, bits: int, count: int):
    """The `count` largest primes p < 2^bits with p = 1 (mod 2N), descending (BASELINE.json configs)."""
    twoN = 2 << logN
    p = ((1 << bits) - 1) // twoN * twoN + 1
    if p >= (1 << bits):
        p -= twoN
    out = []
    while len(out) < count:
        if p < twoN:
            raise ValueError("not enough primes")
        if is_prime(p):
            out.append(p)
        p -= twoN
    return out


def find_psi(q: int, N: int) -> int:
    """A primitive 2N-th root of unity mod q (psi^N = -1).  Which one is implementation private (R2.1)."""
    x = 2
    while True:
        psi = pow(x, (q - 1) // (2 * N), q)
        if pow(psi, N, q) == q - 1:
            return psi
        x += 1


class Params:
    """Parameter set: ring degree, RNS chain, special primes, digit length (R 8(c)-1, R2.4)."""

    def __init__(self, logN, n_q, q_bits, n_p, p_bits, dnum, log2_scale, q_override=None, p_override=None, dlen=None):
        self.logN, self.N, self.n = logN, 1 << logN, 1 << (logN - 1)
        self.q = list(q_override) if q_override else find_primes(logN, q_bits, n_q)
        self.p = list(p_override) if p_override else find_primes(logN, p_bits, n_p)
        self.nq, self.np_ = len(self.q), len(self.p)
        self.dlen = dlen if dlen else -(-self.nq // dnum)
        self.beta_max = -(-self.nq // self.dlen)
        self.mod = self.q + self.p
        self.psi = [find_psi(m, self.N) for m in self.mod]
        self.P = math.prod(self.p)
        self.scale = Fraction(2) ** int(log2_scale)
        qa = np.array(self.q, dtype=np.uint64)
        pa = np.array(self.p, dtype=np.uint64)
        psq = np.array(self.psi[: self.nq], dtype=np.uint64)
        psp = np.array(self.psi[self.nq:], dtype=np.uint64)
        self._h = _lib.orc_params_new(self.N, self.nq, _p(qa), _p(psq), self.np_, _p(pa), _p(psp), self.dlen)
        assert self._h

    def __del__(self):
        if getattr(self, "_h", None):
            _lib.orc_params_free(self._h)
            self._h = None

    def galois(self, r: int) -> int:
        """g = 5^(r mod n) mod 2N (R2.7)."""
        return pow(5, r % self.n, 2 * self.N)

    def digit(self, j: int):
        """Limb indices of key-switch digit j over the full chain (R2.4)."""
        return range(j * self.dlen, min((j + 1) * self.dlen, self.nq))


# --------------------------------------------------------------------------- randomness (R2.3)
# Counter-based generator, spec in DESIGN.md section 4 (R2.3); the CUDA library's host code
# carries its own, independently written copy.
_M64 = (1 << 64) - 1
_GAMMA = 0x9E3779B97F4A7C15
ATTEMPTS = 64  # counter slots reserved per coefficient

PURPOSE_SECRET, PURPOSE_EVK_A, PURPOSE_EVK_E, PURPOSE_ENC_A, PURPOSE_ENC_E = 1, 2, 3, 4, 5
RELIN_KEY_ID = 1 << 40  # key id of the relinearisation key; rotation key ids are r in [1, n)


def mix64(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def stream_key(seed: int, purpose: int, a: int = 0, b: int = 0, c: int = 0) -> int:
    k = mix64(seed ^ _GAMMA)
    for v in (purpose, a, b, c):
        k = mix64(k + v)
    return k


def _mix64_np(z):
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def draws(key: int, counters):
    """draw(key, n) = mix64(key + (n+1)*GAMMA) for an array of counters n."""
    with np.errstate(over="ignore"):
        c = np.asarray(counters, dtype=np.uint64)
        return _mix64_np(np.uint64(key) + (c + np.uint64(1)) * np.uint64(_GAMMA))


def sample_uniform(key: int, N: int, q: int):
    """Coefficient i: draws at counters i*64+a, a=0,1,..: keep the low ceil(log2 q) bits, accept the first < q."""
    mask = np.uint64((1 << (q - 1).bit_length()) - 1)
    out = np.zeros(N, dtype=np.uint64)
    todo = np.arange(N, dtype=np.uint64)
    for a in range(ATTEMPTS):
        x = draws(key, todo * np.uint64(ATTEMPTS) + np.uint64(a)) & mask
        ok = x < np.uint64(q)
        out[todo[ok]] = x[ok]
        if a == ATTEMPTS - 1:
            out[todo[~ok]] = x[~ok] % np.uint64(q)
        todo = todo[~ok]
        if todo.size == 0:
            break
    return out


def sample_ternary(key: int, N: int):
    """Low 2 bits of a draw: 0 -> -1, 1 -> 0, 2 -> +1, 3 -> redraw (uniform ternary, dense)."""
    out = np.zeros(N, dtype=np.int64)
    todo = np.arange(N, dtype=np.uint64)
    for a in range(ATTEMPTS):
        x = draws(key, todo * np.uint64(ATTEMPTS) + np.uint64(a)) & np.uint64(3)
        ok = x < np.uint64(3)
        out[todo[ok]] = x[ok].astype(np.int64) - 1
        todo = todo[~ok]
        if todo.size == 0:
            break
    return out


# C[x] = floor(2^64 * Pr(|X| <= x)), X discrete Gaussian sigma = 3.2 cut at |x| <= 19; C[19] = 2^64.
# Pinned against 80-digit decimal arithmetic in tests/test_oracle_ckks.py.
GAUSS_CDT = [
    0x1FEA56814B22FE3A, 0x5CB44BA97E1C801C, 0x9135C4D2AB6097AC, 0xBA57841EC437E30A, 0xD790D29879901FE9,
    0xEA65B1358D74FB9D, 0xF5672D96E886CF31, 0xFB3C9D22CC87D60F, 0xFE0A92B033D640A2, 0xFF439D38007352AE,
    0xFFBF67E425D189D1, 0xFFEBCDF3A4629F98, 0xFFFA3F2F78880D45, 0xFFFE81F40111A23B, 0xFFFFA5D06BC38AFB,
    0xFFFFECA4870DFE3C, 0xFFFFFC3B68ED3B4A, 0xFFFFFF58143B9611, 0xFFFFFFE850CE70A6,
]  # 19 entries for x = 0..18; x = 19 is the "always accept" case


def sample_gauss(key: int, N: int):
    """u = draw(i*64): magnitude = least x with u < C[x]; if x > 0, low bit of draw(i*64+1) = 1 -> negative."""
    idx = np.arange(N, dtype=np.uint64) * np.uint64(ATTEMPTS)
    u = draws(key, idx)
    mag = np.searchsorted(np.array(GAUSS_CDT, dtype=np.uint64), u, side="right").astype(np.int64)
    sign = (draws(key, idx + np.uint64(1)) & np.uint64(1)).astype(np.int64)
    return np.where(sign == 1, -mag, mag)


# --------------------------------------------------------------------------- encode / decode (R2.2)
def slot_exponents(N: int):
    """e_j = 5^j mod 2N: slot j is the evaluation point zeta^{e_j}, zeta = exp(i*pi/N)."""
    e, out = 1, np.empty(N // 2, dtype=np.int64)
    for j in range(N // 2):
        out[j] = e
        e = e * 5 % (2 * N)
    return out


def encode_coeffs(z, N: int, scale) -> np.ndarray:
    """m_t = round((2s/N) Re(sum_j z_j conj(zeta_j)^t)), t in [0,N): centred integers (int64).

    sum_j z_j exp(-2 pi i e_j t / 2N) is a length-2N DFT of the vector holding z_j at index e_j."""
    z = np.asarray(z, dtype=np.complex128)
    assert z.shape == (N // 2,)
    A = np.zeros(2 * N, dtype=np.complex128)
    A[slot_exponents(N)] = z
    F = np.fft.fft(A)[:N]
    m = np.rint(F.real * (2.0 * float(scale) / N))
    assert np.all(np.abs(m) < 2.0 ** 62)
    return m.astype(np.int64)


def encode_coeffs_def(z, N: int, scale) -> np.ndarray:
    """The O(N^2) definition itself (small N only)."""
    z = np.asarray(z, dtype=np.complex128)
    e = slot_exponents(N)
    t = np.arange(N)
    ang = -np.pi * np.outer(t, e) / N
    acc = (np.exp(1j * ang) * z[None, :]).sum(axis=1)
    return np.rint(acc.real * (2.0 * float(scale) / N)).astype(np.int64)


def decode_coeffs(m, N: int, scale) -> np.ndarray:
    """z_j = (1/s) sum_t m_t zeta_j^t with m_t centred integers (Python ints or int64)."""
    mf = np.array([float(Fraction(int(v)) / Fraction(scale)) for v in m], dtype=np.float64)
    A = np.zeros(2 * N, dtype=np.complex128)
    A[:N] = mf
    F = np.fft.ifft(A) * (2 * N)
    return F[slot_exponents(N)]


class Plaintext:
    def __init__(self, params: Params, coeffs_i64, L: int, scale):
        self.L, self.scale = L, Fraction(scale)
        m = np.ascontiguousarray(coeffs_i64, dtype=np.int64)
        self.coeffs = m
        self.c = np.zeros((L, params.N), dtype=np.uint64)
        _lib.orc_reduce_signed(params._h, L, m.ctypes.data_as(_i64p), _p(self.c))


def encode(params: Params, z, L: int, scale=None) -> Plaintext:
    scale = params.scale if scale is None else Fraction(scale)
    return Plaintext(params, encode_coeffs(z, params.N, scale), L, scale)


class Ciphertext:
    """c: uint64 [2][L][N], coefficient domain, canonical residues; scale an exact rational (R2.8)."""

    def __init__(self, c, L, scale):
        self.c, self.L, self.scale = c, L, Fraction(scale)


# --------------------------------------------------------------------------- keys (R2.4)
class Keys:
    def __init__(self, params: Params, seed: int):
        self.params, self.seed = params, seed
        self.s = sample_ternary(stream_key(seed, PURPOSE_SECRET), params.N)  # int64 in {-1,0,1}
        self.s_rns = _signed_to_rns(params, self.s, range(len(params.mod)))  # [nq+np][N]
        self.evk = {}  # key id -> (b, a), each [beta_max][nq+np][N]


def _signed_to_rns(params, v, limbs):
    out = np.zeros((len(limbs), params.N), dtype=np.uint64)
    for k, t in enumerate(limbs):
        q = params.mod[t]
        out[k] = np.where(v >= 0, v, v + q).astype(np.uint64)
    return out


def _polymul(params, t, a, b):
    out = np.zeros(params.N, dtype=np.uint64)
    _lib.orc_polymul(params.N, params.mod[t], params.psi[t], _p(np.ascontiguousarray(a)), _p(np.ascontiguousarray(b)), _p(out))
    return out


def _switching_key(params: Params, keys: Keys, key_id: int, s_from_rns):
    """For every digit j, over all nq+np limbs t: a_j[t] uniform, b_j[t] = -a_j[t] s + e_j + f_{j,t} s' (mod t),
    f_{j,t} = (P mod t) if t in D_j else 0 (R2.4)."""
    A = len(params.mod)
    b = np.zeros((params.beta_max, A, params.N), dtype=np.uint64)
    a = np.zeros_like(b)
    for j in range(params.beta_max):
        e = sample_gauss(stream_key(keys.seed, PURPOSE_EVK_E, key_id, j), params.N)
        for t in range(A):
            q = params.mod[t]
            a[j, t] = sample_uniform(stream_key(keys.seed, PURPOSE_EVK_A, key_id, j, t), params.N, q)
            as_ = _polymul(params, t, a[j, t], keys.s_rns[t])
            e_t = np.where(e >= 0, e, e + q).astype(np.uint64)
            v = (np.uint64(q) - as_) % np.uint64(q)
            v = (v + e_t) % np.uint64(q)
            if t in params.digit(j):
                f = params.P % q
                fs = np.array([int(x) * f % q for x in s_from_rns[t]], dtype=np.uint64)
                v = (v + fs) % np.uint64(q)
            b[j, t] = v
    return b, a


def keygen(params: Params, seed: int, rot_steps=(), want_relin=False) -> Keys:
    keys = Keys(params, seed)
    A = len(params.mod)
    for r in rot_steps:
        r = r % params.n
        if r == 0 or r in keys.evk:
            continue
        g = params.galois(r)
        s_rot = np.zeros((A, params.N), dtype=np.uint64)
        for t in range(A):
            _lib.orc_automorph(params.N, params.mod[t], g, _p(keys.s_rns[t].copy()), _p(s_rot[t]))
        keys.evk[r] = _switching_key(params, keys, r, s_rot)
    if want_relin:
        s2 = np.stack([_polymul(params, t, keys.s_rns[t], keys.s_rns[t]) for t in range(A)])
        keys.evk[RELIN_KEY_ID] = _switching_key(params, keys, RELIN_KEY_ID, s2)
    return keys


# --------------------------------------------------------------------------- encrypt / decrypt (R2.5)
def encrypt(params: Params, keys: Keys, pt: Plaintext, enc_seed: int) -> Ciphertext:
    """Symmetric: c1[t] = a[t] uniform per limb; c0[t] = -a[t] s + e + m (mod t)."""
    L = pt.L
    c = np.zeros((2, L, params.N), dtype=np.uint64)
    e = sample_gauss(stream_key(enc_seed, PURPOSE_ENC_E), params.N)
    for t in range(L):
        q = params.mod[t]
        a = sample_uniform(stream_key(enc_seed, PURPOSE_ENC_A, t), params.N, q)
        as_ = _polymul(params, t, a, keys.s_rns[t])
        e_t = np.where(e >= 0, e, e + q).astype(np.uint64)
        v = (np.uint64(q) - as_) % np.uint64(q)
        v = (v + e_t) % np.uint64(q)
        c[0, t] = (v + pt.c[t]) % np.uint64(q)
        c[1, t] = a
    return Ciphertext(c, L, pt.scale)


def crt_centre(params: Params, residues, L: int):
    """CRT-combine [L][N] residues into Python integers centred in (-Q_L/2, Q_L/2]."""
    Q = math.prod(params.q[:L])
    acc = [0] * params.N
    for t in range(L):
        q = params.q[t]
        Qh = Q // q
        w = Qh * pow(Qh % q, -1, q)
        col = residues[t].tolist()
        for n in range(params.N):
            acc[n] += col[n] * w
    out = []
    for v in acc:
        v %= Q
        out.append(v - Q if v > Q // 2 else v)
    return out


def decrypt_coeffs(params: Params, keys: Keys, ct: Ciphertext):
    """mu[t] = c0[t] + c1[t] s, CRT-combined and centred: a list of Python ints."""
    mu = np.zeros((ct.L, params.N), dtype=np.uint64)
    for t in range(ct.L):
        q = np.uint64(params.mod[t])
        mu[t] = (ct.c[0, t] + _polymul(params, t, ct.c[1, t], keys.s_rns[t])) % q
    return crt_centre(params, mu, ct.L)


def decrypt_decode(params: Params, keys: Keys, ct: Ciphertext) -> np.ndarray:
    return decode_coeffs(decrypt_coeffs(params, keys, ct), params.N, ct.scale)


# --------------------------------------------------------------------------- primitives (R2.6-R2.8)
def rotate(params: Params, keys: Keys, ct: Ciphertext, r: int) -> Ciphertext:
    """Rot(ct, r): slots move left by r (Eq. 1; R2.7).  Level and scale unchanged."""
    r %= params.n
    if r == 0:
        return Ciphertext(ct.c.copy(), ct.L, ct.scale)
    b, a = keys.evk[r]
    out = np.zeros_like(ct.c)
    _lib.orc_rotate(params._h, ct.L, params.galois(r), _p(ct.c), _p(b), _p(a), _p(out))
    return Ciphertext(out, ct.L, ct.scale)


def rotate_hoisted(params: Params, keys: Keys, ct: Ciphertext, r: int) -> Ciphertext:
    """Rot(ct, r) with the decomposition hoisted out of the rotation (R2.7b): ModUp of the unrotated c1, automorphism on
    the extended digits.  Decrypts like rotate(); the limbs differ (a multiple of Q_j per digit before ModDown)."""
    r %= params.n
    if r == 0:
        return Ciphertext(ct.c.copy(), ct.L, ct.scale)
    b, a = keys.evk[r]
    out = np.zeros_like(ct.c)
    _lib.orc_rotate_hoisted(params._h, ct.L, params.galois(r), _p(ct.c), _p(b), _p(a), _p(out))
    return Ciphertext(out, ct.L, ct.scale)


def add(params: Params, x: Ciphertext, y: Ciphertext) -> Ciphertext:
    assert x.L == y.L and x.scale == y.scale
    out = np.zeros_like(x.c)
    _lib.orc_add(params._h, x.L, 2, _p(x.c), _p(y.c), _p(out))
    return Ciphertext(out, x.L, x.scale)


def pmult_acc(params: Params, acc, ct: Ciphertext, pt: Plaintext):
    """acc += ct (*) pt (both polynomials, per limb); acc is a raw [2][L][N] array."""
    assert pt.L == ct.L
    _lib.orc_pmult_acc(params._h, ct.L, _p(ct.c), _p(pt.c), _p(acc))


def pmult(params: Params, ct: Ciphertext, pt: Plaintext) -> Ciphertext:
    acc = np.zeros_like(ct.c)
    pmult_acc(params, acc, ct, pt)
    return Ciphertext(acc, ct.L, ct.scale * pt.scale)


def rescale(params: Params, ct: Ciphertext) -> Ciphertext:
    """Drop q_{L-1} with floor rounding on the canonical representative (R2.8, A10)."""
    assert ct.L >= 2
    out = np.zeros((2, ct.L - 1, params.N), dtype=np.uint64)
    for k in range(2):
        _lib.orc_rescale(params._h, ct.L, _p(ct.c[k]), _p(out[k]))
    return Ciphertext(out, ct.L - 1, ct.scale / params.q[ct.L - 1])


def keyswitch(params: Params, L: int, d, evk):
    """KS(d; key): d [L][N] -> (ks0, ks1) each [L][N] (R2.6)."""
    b, a = evk
    o0 = np.zeros((L, params.N), dtype=np.uint64)
    o1 = np.zeros_like(o0)
    _lib.orc_keyswitch(params._h, L, _p(np.ascontiguousarray(d)), _p(b), _p(a), _p(o0), _p(o1))
    return o0, o1


def square_relin(params: Params, keys: Keys, ct: Ciphertext) -> Ciphertext:
    """d0 = c0 c0, d1 = 2 c0 c1, d2 = c1 c1; (d0, d1) + KS(d2; relin); then rescale (R2.12)."""
    L, N = ct.L, params.N
    d0 = np.zeros((L, N), dtype=np.uint64)
    d1 = np.zeros_like(d0)
    d2 = np.zeros_like(d0)
    _lib.orc_polymul_rns(params._h, L, _p(ct.c[0]), _p(ct.c[0]), _p(d0))
    _lib.orc_polymul_rns(params._h, L, _p(ct.c[0]), _p(ct.c[1]), _p(d1))
    _lib.orc_polymul_rns(params._h, L, _p(ct.c[1]), _p(ct.c[1]), _p(d2))
    k0, k1 = keyswitch(params, L, d2, keys.evk[RELIN_KEY_ID])
    out = np.zeros_like(ct.c)
    for t in range(L):
        q = np.uint64(params.mod[t])
        out[0, t] = (d0[t] + k0[t]) % q
        out[1, t] = ((d1[t] + d1[t]) % q + k1[t]) % q
    return rescale(params, Ciphertext(out, L, ct.scale * ct.scale))


def square_sum_relin(params: Params, keys: Keys, cts) -> Ciphertext:
    """Sum of squares with ONE relinearisation (R2.12c; x^2 followed by sum-pooling): the tensor products
    are added component-wise first, (D0, D1, D2) = sum_i (c0_i c0_i, 2 c0_i c1_i, c1_i c1_i), then
    (D0, D1) + KS(D2; relin) and one rescale.  Decrypts to sum_i x_i^2; for a single ciphertext it is square_relin."""
    L, N = cts[0].L, params.N
    D = np.zeros((3, L, N), dtype=np.uint64)
    t0 = np.zeros((L, N), dtype=np.uint64)
    for ct in cts:
        assert ct.L == L and ct.scale == cts[0].scale
        for k, (a, b) in enumerate(((0, 0), (0, 1), (1, 1))):
            _lib.orc_polymul_rns(params._h, L, _p(ct.c[a]), _p(ct.c[b]), _p(t0))
            for t in range(L):
                q = np.uint64(params.mod[t])
                term = (t0[t] + t0[t]) % q if k == 1 else t0[t]
                D[k, t] = (D[k, t] + term) % q
    k0, k1 = keyswitch(params, L, D[2], keys.evk[RELIN_KEY_ID])
    out = np.zeros_like(cts[0].c)
    for t in range(L):
        q = np.uint64(params.mod[t])
        out[0, t] = (D[0, t] + k0[t]) % q
        out[1, t] = (D[1, t] + k1[t]) % q
    return rescale(params, Ciphertext(out, L, cts[0].scale * cts[0].scale))


# --------------------------------------------------------------------------- CMult, PMultConst, degree-3 activation (R2.8, R2.12)
def cmult_relin(params: Params, keys: Keys, x: Ciphertext, y: Ciphertext) -> Ciphertext:
    """(d0, d1, d2) = (x0 y0, x0 y1 + x1 y0, x1 y1); (d0, d1) + KS(d2; relin); then rescale (PAPER.md:63 CMult; R2.12)."""
    assert x.L == y.L
    L, N = x.L, params.N
    d0, d1, d1b, d2 = (np.zeros((L, N), dtype=np.uint64) for _ in range(4))
    _lib.orc_polymul_rns(params._h, L, _p(x.c[0]), _p(y.c[0]), _p(d0))
    _lib.orc_polymul_rns(params._h, L, _p(x.c[0]), _p(y.c[1]), _p(d1))
    _lib.orc_polymul_rns(params._h, L, _p(x.c[1]), _p(y.c[0]), _p(d1b))
    _lib.orc_polymul_rns(params._h, L, _p(x.c[1]), _p(y.c[1]), _p(d2))
    k0, k1 = keyswitch(params, L, d2, keys.evk[RELIN_KEY_ID])
    out = np.zeros_like(x.c)
    for t in range(L):
        q = np.uint64(params.mod[t])
        out[0, t] = (d0[t] + k0[t]) % q
        out[1, t] = ((d1[t] + d1b[t]) % q + k1[t]) % q
    return rescale(params, Ciphertext(out, L, x.scale * y.scale))


def round_half_up(x) -> int:
    return math.floor(Fraction(x) + Fraction(1, 2))


def mul_const(params: Params, ct: Ciphertext, c, E) -> Ciphertext:
    """PMultConst(ct, c, E): every limb times round_half_up(c E) with c, E exact rationals; scale multiplies by E (R2.8)."""
    k = round_half_up(Fraction(c) * Fraction(E))
    kt = np.array([k % q for q in params.q[:ct.L]], dtype=np.uint64)
    out = np.zeros_like(ct.c)
    for j in range(2):
        _lib.orc_mul_scalar(params._h, ct.L, _p(ct.c[j]), _p(kt), _p(out[j]))
    return Ciphertext(out, ct.L, ct.scale * Fraction(E))


def add_const(params: Params, ct: Ciphertext, k: int) -> Ciphertext:
    """the integer k added to coefficient 0 of c0 (the encoding of the real constant k / scale in every slot, R2.2)."""
    out = ct.c.copy()
    for t in range(ct.L):
        q = params.q[t]
        out[0, t, 0] = np.uint64((int(out[0, t, 0]) + k) % q)
    return Ciphertext(out, ct.L, ct.scale)


POLY3 = (Fraction(1, 2), Fraction(197, 1000), Fraction(-4, 1000))  # BASELINE config 3: x -> 0.5 + 0.197 x - 0.004 x^3


def poly3(params: Params, keys: Keys, x: Ciphertext, coef=POLY3) -> Ciphertext:
    """Degree-3 activation a0 + a1 x + a3 x^3 in two levels (R2.12): x2 = Rescale(Relin(x x));
    t = Rescale(PMultConst(x, a3, q_{L-1})); x3 = Rescale(Relin(x2 t)) at scale s3 = s^3/(q_{L-1} q_{L-2});
    u = Rescale(Rescale(PMultConst(x, a1, s^2))) (same scale); out = x3 + u + round_half_up(a0 s3) on coefficient 0."""
    a0, a1, a3 = coef
    L, s = x.L, x.scale
    x2 = cmult_relin(params, keys, x, x)
    t = rescale(params, mul_const(params, x, a3, params.q[L - 1]))
    x3 = cmult_relin(params, keys, x2, t)
    u = rescale(params, rescale(params, mul_const(params, x, a1, s * s)))
    assert x3.scale == u.scale == s ** 3 / (params.q[L - 1] * params.q[L - 2])
    return add_const(params, add(params, x3, u), round_half_up(Fraction(a0) * x3.scale))
