// fenc_host.cpp -- host-side mathematics of libfenc: prime chains, roots and twiddle tables, the counter-based
// generator (host copy, used for the secret), fp64 encode / decode, and the CRT lift used by decryption.
// Written independently of oracle/ (the two share no code); the rules are those of DESIGN.md section 4.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <complex>
#include <map>
#include <mutex>

#include "fenc_internal.h"

namespace fh {

u64 mulmod(u64 a, u64 b, u64 q) { return (u64)((u128)a * b % q); }
u64 powmod(u64 a, u64 e, u64 q) {
  u64 r = 1 % q;
  a %= q;
  for (; e; e >>= 1) {
    if (e & 1) r = mulmod(r, a, q);
    a = mulmod(a, a, q);
  }
  return r;
}
u64 invmod(u64 a, u64 q) { return powmod(a % q, q - 2, q); }

// deterministic Miller-Rabin, exact below 2^64 with the first twelve prime bases
bool is_prime(u64 n) {
  static const u64 bases[12] = {2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37};
  if (n < 2) return false;
  for (u64 p : bases) {
    if (n == p) return true;
    if (n % p == 0) return false;
  }
  u64 d = n - 1;
  int s = 0;
  while ((d & 1) == 0) d >>= 1, s++;
  for (u64 a : bases) {
    u64 x = powmod(a, d, n);
    if (x == 1 || x == n - 1) continue;
    bool comp = true;
    for (int i = 1; i < s && comp; i++) {
      x = mulmod(x, x, n);
      if (x == n - 1) comp = false;
    }
    if (comp) return false;
  }
  return true;
}

// the `count` largest primes p < 2^bits with p = 1 (mod 2N), descending (BASELINE.json configs; R1)
bool find_primes(int logN, int bits, int count, std::vector<u64> &out) {
  const u64 twoN = 2ull << logN;
  const u64 bound = 1ull << bits;
  u64 c = (bound - 1) / twoN * twoN + 1;
  if (c >= bound) c -= twoN;
  out.clear();
  while ((int)out.size() < count) {
    if (c <= twoN) return false;
    if (is_prime(c)) out.push_back(c);
    c -= twoN;
  }
  return true;
}

// any primitive 2N-th root of unity (which one is implementation private, R2.1)
u64 find_psi(u64 q, u64 N) {
  for (u64 x = 2;; x++) {
    u64 psi = powmod(x, (q - 1) / (2 * N), q);
    if (powmod(psi, N, q) == q - 1) return psi;
  }
}

u64 shoup(u64 c, u64 q) { return (u64)(((u128)c << 64) / q); }
u64 to_mont(u64 c, u64 q) { return (u64)(((u128)c << 64) % q); }
u64 neg_qinv(u64 q) {
  u64 x = q;  // Newton iteration for q^{-1} mod 2^64 (q odd): 3 bits correct, doubling
  for (int i = 0; i < 6; i++) x *= 2 - q * x;
  return (u64)0 - x;
}

static u32 bitrev(u32 x, int bits) {
  u32 r = 0;
  for (int i = 0; i < bits; i++) r = (r << 1) | ((x >> i) & 1);
  return r;
}

// fwd[k] = psi^bitrev(k), inv[k] = psi^-bitrev(k), each with its Shoup companion
// Butterflies of this modulus multiply on the FP64 pipe (fenc_device.cuh): "narrow" moduli below 2^45 everywhere, moduli
// below 2^50 only with the compile-time tile schedules (ring degree >= 2^12), whose rounds re-centre the values.
bool f64_narrow(u64 q) {
  static const bool off = getenv("FENC_NO_F64") != nullptr;  // diagnostics: integer butterflies everywhere
  return !off && q < (1ull << 45);
}
bool f64_modulus(u64 q, int logN) {
  static const bool off = getenv("FENC_NO_F64") != nullptr;
  static const bool no_wide = getenv("FENC_NO_F64_WIDE") != nullptr;
  if (off) return false;
  return q < (1ull << 45) || (!no_wide && logN >= 12 && q < (1ull << 50));
}
void build_twiddles(u64 q, u64 psi, int logN, ShoupC *fwd, ShoupC *inv) {
  const u32 N = 1u << logN;
  std::vector<u64> pw(N), ipw(N);
  const u64 ipsi = invmod(psi, q);
  pw[0] = ipw[0] = 1;
  for (u32 i = 1; i < N; i++) pw[i] = mulmod(pw[i - 1], psi, q), ipw[i] = mulmod(ipw[i - 1], ipsi, q);
  const bool f64 = f64_modulus(q, logN);
  auto bits = [](double d) { u64 b; memcpy(&b, &d, 8); return b; };
  for (u32 k = 0; k < N; k++) {
    u32 r = bitrev(k, logN);
    if (f64) {  // {(double) w, (double) (w / q)}: the quotient estimate needs c/q to within a few ulp (fenc_device.cuh)
      fwd[k].c = bits((double)pw[r]), fwd[k].cs = bits((double)((long double)pw[r] / (long double)q));
      inv[k].c = bits((double)ipw[r]), inv[k].cs = bits((double)((long double)ipw[r] / (long double)q));
    } else {
      fwd[k].c = pw[r], fwd[k].cs = shoup(pw[r], q);
      inv[k].c = ipw[r], inv[k].cs = shoup(ipw[r], q);
    }
  }
}


// ------------------------------------------------------------------ counter-based generator (R2.3)
static const u64 GAMMA = 0x9E3779B97F4A7C15ull;
u64 mix64(u64 z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
u64 stream_key(u64 seed, u64 purpose, u64 a, u64 b, u64 c) {
  u64 k = mix64(seed ^ GAMMA);
  k = mix64(k + purpose);
  k = mix64(k + a);
  k = mix64(k + b);
  k = mix64(k + c);
  return k;
}
static inline u64 draw(u64 key, u64 n) { return mix64(key + (n + 1) * GAMMA); }

// uniform ternary: low two bits of a draw, 0 -> -1, 1 -> 0, 2 -> +1, 3 -> next counter (64 per coefficient)
void sample_ternary(u64 key, int N, int64_t *out) {
  for (int i = 0; i < N; i++) {
    out[i] = 0;
    for (int a = 0; a < 64; a++) {
      u64 x = draw(key, (u64)i * 64 + a) & 3;
      if (x < 3) {
        out[i] = (int64_t)x - 1;
        break;
      }
    }
  }
}

// ------------------------------------------------------------------ encode / decode (R2.2)
typedef std::complex<double> cd;
struct FftPlan {
  int logn;
  std::vector<cd> w;      // w[k] = exp(-2 pi i k / n), k < n/2
  std::vector<u32> rev;
};
static const FftPlan &plan_for(int logn) {
  static std::map<int, FftPlan> plans;
  static std::mutex mu;
  std::lock_guard<std::mutex> lk(mu);
  auto it = plans.find(logn);
  if (it != plans.end()) return it->second;
  FftPlan p;
  p.logn = logn;
  const size_t n = (size_t)1 << logn;
  p.w.resize(n / 2);
  const long double two_pi = 6.283185307179586476925286766559005768L;
  for (size_t k = 0; k < n / 2; k++) {
    long double a = -two_pi * (long double)k / (long double)n;
    p.w[k] = cd((double)cosl(a), (double)sinl(a));
  }
  p.rev.resize(n);
  for (size_t i = 0; i < n; i++) p.rev[i] = bitrev((u32)i, logn);
  return plans.emplace(logn, std::move(p)).first->second;
}
// in-place DFT: a[t] <- sum_k a[k] exp(sign * 2 pi i k t / n), sign = -1 (forward) or +1
static void fft(std::vector<cd> &a, int logn, int sign) {
  const FftPlan &p = plan_for(logn);
  const size_t n = (size_t)1 << logn;
  for (size_t i = 0; i < n; i++)
    if (i < p.rev[i]) std::swap(a[i], a[p.rev[i]]);
  for (size_t len = 2; len <= n; len <<= 1) {
    const size_t step = n / len;
    for (size_t s = 0; s < n; s += len)
      for (size_t k = 0; k < len / 2; k++) {
        cd w = p.w[k * step];
        if (sign > 0) w = std::conj(w);
        cd x = a[s + k], y = a[s + k + len / 2] * w;
        a[s + k] = x + y;
        a[s + k + len / 2] = x - y;
      }
  }
}
static const std::vector<u32> &slot_exponents(int logN) {  // e_j = 5^j mod 2N
  static std::map<int, std::vector<u32>> tabs;
  static std::mutex mu;
  std::lock_guard<std::mutex> lk(mu);
  auto it = tabs.find(logN);
  if (it != tabs.end()) return it->second;
  const u32 N = 1u << logN;
  std::vector<u32> e(N / 2);
  u64 x = 1;
  for (u32 j = 0; j < N / 2; j++) e[j] = (u32)x, x = x * 5 % (2 * N);
  return tabs.emplace(logN, std::move(e)).first->second;
}
// m_t = round((2 s / N) Re(sum_j z_j conj(zeta_j)^t)): a 2N-point DFT of the vector holding z_j at index e_j
void encode_slots(int logN, const double *re, const double *im, double scale, int64_t *coeffs) {
  const u32 N = 1u << logN;
  const std::vector<u32> &e = slot_exponents(logN);
  std::vector<cd> a(2 * (size_t)N, cd(0, 0));
  for (u32 j = 0; j < N / 2; j++) a[e[j]] = cd(re[j], im ? im[j] : 0.0);
  fft(a, logN + 1, -1);
  const double f = 2.0 * scale / (double)N;
  for (u32 t = 0; t < N; t++) coeffs[t] = (int64_t)std::nearbyint(a[t].real() * f);
}
// z_j = sum_t (m_t / s) zeta_j^t
void decode_coeffs(int logN, const long double *m_over_scale, double *re, double *im) {
  const u32 N = 1u << logN;
  const std::vector<u32> &e = slot_exponents(logN);
  std::vector<cd> a(2 * (size_t)N, cd(0, 0));
  for (u32 t = 0; t < N; t++) a[t] = cd((double)m_over_scale[t], 0.0);
  fft(a, logN + 1, +1);
  for (u32 j = 0; j < N / 2; j++) {
    re[j] = a[e[j]].real();
    if (im) im[j] = a[e[j]].imag();
  }
}

// ------------------------------------------------------------------ CRT lift (decrypt, R2.5)
// Garner mixed-radix digits v_i of X in [0,Q): X = v_0 + q_0 (v_1 + q_1 (v_2 + ...)).  X > (Q-1)/2 means the centred
// value is X - Q = -((Q-1-X) + 1), and Q-1-X has digits q_i-1-v_i with no borrows; Horner in long double.
void crt_centre_scaled(const u64 *q, int L, int N, const u64 *res, long double scale, long double *out) {
  std::vector<u64> inv((size_t)L * L, 0);  // inv[i*L+k] = q_k^{-1} mod q_i, k < i
  for (int i = 0; i < L; i++)
    for (int k = 0; k < i; k++) inv[(size_t)i * L + k] = invmod(q[k] % q[i], q[i]);
  std::vector<u64> half(L);  // digits of (Q-1)/2: Garner of residues (q_i-1)/2
  std::vector<u64> v(L);
  auto garner = [&](const u64 *r, size_t stride, u64 *dig) {
    for (int i = 0; i < L; i++) {
      u64 x = r[(size_t)i * stride] % q[i];
      for (int k = 0; k < i; k++) {
        u64 d = dig[k] % q[i];
        x = x >= d ? x - d : x + q[i] - d;
        x = mulmod(x, inv[(size_t)i * L + k], q[i]);
      }
      dig[i] = x;
    }
  };
  std::vector<u64> hr(L);
  for (int i = 0; i < L; i++) hr[i] = (q[i] - 1) / 2;
  garner(hr.data(), 1, half.data());
  for (int n = 0; n < N; n++) {
    garner(res + n, (size_t)N, v.data());
    bool neg = false;
    for (int i = L - 1; i >= 0; i--) {
      if (v[i] != half[i]) {
        neg = v[i] > half[i];
        break;
      }
    }
    long double acc = 0.0L;
    for (int i = L - 1; i >= 0; i--) {
      u64 d = neg ? q[i] - 1 - v[i] : v[i];
      acc = acc * (long double)q[i] + (long double)d;
    }
    if (neg) acc = -(acc + 1.0L);
    out[n] = acc / scale;
  }
}

}  // namespace fh
