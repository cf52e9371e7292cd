// fenc_device.cuh -- device-side modular arithmetic and the shared-memory NTT tile engine (sm_100a).
//
// Arithmetic: 64-bit words on the 32-bit integer pipes (IMAD.WIDE on the fma pipe, IADD3/LOP3 on the alu pipe).
//  - constant operands (twiddles, scaling constants): Shoup multiplication with a precomputed floor(c 2^64 / q),
//    lazy butterflies: forward values grow by at most 2q per stage without any correction for q < 2^58 (one
//    full reduction at the end), Harvey's [0,4q) form for larger q; inverse values stay in [0,2q); needs q < 2^61.
//  - variable x variable sums (evk inner product, plaintext MAC, base conversion): 128-bit lazy accumulation of
//    x * y_mont products followed by ONE Montgomery reduction (y stored as y 2^64 mod q).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "fenc_internal.h"

#define DEVI __device__ __forceinline__

DEVI u64 csub(u64 x, u64 q) { return x >= q ? x - q : x; }

// x * c mod q in [0, 2q) for any x < 2^64 (cs = floor(c 2^64 / q), c < q)
DEVI u64 shoup_lazy(u64 x, u64 c, u64 cs, u64 q) {
  u64 hi = __umul64hi(x, cs);
  return x * c - hi * q;
}
DEVI u64 shoup_mul(u64 x, u64 c, u64 cs, u64 q) { return csub(shoup_lazy(x, c, cs, q), q); }

// (hi:lo) += a * b
DEVI void mac128(u64 &lo, u64 &hi, u64 a, u64 b) {
  asm("mad.lo.cc.u64 %0, %2, %3, %0;\n\tmadc.hi.u64 %1, %2, %3, %1;" : "+l"(lo), "+l"(hi) : "l"(a), "l"(b));
}
// Montgomery reduction: (hi:lo) 2^-64 mod q, canonical; requires (hi:lo) < q 2^64
DEVI u64 mont_redc(u64 lo, u64 hi, u64 q, u64 qinv_neg) {
  u64 m = lo * qinv_neg;
  u64 t = hi + __umul64hi(m, q) + (lo != 0 ? 1ull : 0ull);
  return csub(t, q);
}
// a * b_mont 2^-64 mod q  (= a*b mod q when b_mont = b 2^64 mod q)
DEVI u64 mont_mul(u64 a, u64 b, u64 q, u64 qinv_neg) {
  u64 lo = a * b, hi = __umul64hi(a, b);
  return mont_redc(lo, hi, q, qinv_neg);
}
DEVI u64 addmod(u64 a, u64 b, u64 q) { return csub(a + b, q); }
DEVI u64 submod(u64 a, u64 b, u64 q) { return a >= b ? a - b : a + q - b; }

// NTT-domain index map of the Galois automorphism sigma_g (R2.7): position p of the transform holds the
// evaluation at psi^(2 brev(p) + 1); sigma_g(a) evaluated there is a evaluated at psi^((2 brev(p) + 1) g).
DEVI u32 galois_src(u32 p, u32 g, int logN) {
  u32 e = __brev(p) >> (32 - logN);
  u32 r = ((g * (2u * e + 1u)) >> 1) & ((1u << logN) - 1u);
  return __brev(r) >> (32 - logN);
}

// shared-memory swizzle: XOR of low index bits with bits 4..6 so that the radix-8 register rounds at window
// positions 0, 2, 3 and >= 5 as well as linear accesses are bank-conflict free for 64-bit words.
DEVI int swz(int e) { return e ^ (((e >> 4) & 1) << 1) ^ (((e >> 5) & 1) << 2) ^ (((e >> 6) & 1) * 9); }

// Tile geometry: tile element e (0 <= e < 2^lt) is global coefficient
//   j = ((e >> lc) << sh) | (tile << lc) | (e & (2^lc - 1)).
// Row pass: lc = lt (contiguous tile).  Column pass: lc = log2(columns per tile), sh = brow.
struct TileGeo {
  int lt, lc, sh, logN;
  u32 tile;
  DEVI u32 gidx(int e) const { return ((u32)(e >> lc) << sh) | (tile << lc) | ((u32)e & ((1u << lc) - 1u)); }
  DEVI int gbit(int pb) const { return pb < lc ? pb : pb - lc + sh; }  // global bit of tile bit pb
};

// v mod q for any v < 2^64: v - floor(v qbar / 2^64) q lies in [0, 2q) (qbar = floor(2^64 / q)), then one correction
DEVI u64 fullred(u64 v, u64 q, u64 qbar) { return csub(v - __umul64hi(v, qbar) * q, q); }

// ---------------------------------------------------------------------------------------------- fp64 twiddle multiply
// For moduli below 2^45 (ModConst.f64 != 0) the butterflies multiply on the FP64 pipe: on B200 every integer multiply
// shares the fmaheavy pipe (70-75 % busy in the NTT kernels, their top stall) while DFMA issues at 64 lanes/clk/SM on a
// pipe of its own.  x c mod q for x < 2^51: with xd = x as a double, h + l = xd c exactly (h = rn(xd c),
// l = fma(xd, c, -h)), k = rint(xd (c/q)) is floor or ceil of the true quotient (the relative error of c/q is 2^-53 and
// the quotient is below 2^51), so t = (h - k q) + l is the exact integer x c - k q in (-q, q): fma(-k, q, h) is exact
// because its result, t - l, is an integer below 2^42.  The return value t + q lies in (0, 2q), the range
// shoup_lazy promises, so the lazy bounds of the integer butterflies carry over unchanged and the canonical results
// are identical.  Twiddle tables of such moduli hold the pair {(double) w, (double) (w / q)} instead of {w, w'}.
#define FENC_F64_MAX_BITS 45
DEVI double u2d52(u64 x) {  // exact for x < 2^52
  return __dadd_rn(__hiloint2double((int)((u32)(x >> 32) | 0x43300000u), (int)(u32)x), -4503599627370496.0);
}
struct F64Mod { double q, qinv; };  // q and 1/q
DEVI F64Mod f64mod(u64 q, u64 qinv_bits) { return F64Mod{(double)q, __longlong_as_double((long long)qinv_bits)}; }
#define F64_RINT_MAGIC 6755399441055744.0  // 1.5 2^52: fma(a, b, MAGIC) - MAGIC = rint(a b) for |a b| < 2^51
// x c - k q in (-q, q) for a double x holding an integer, |x| < 2^51
DEVI double mulmod_dd(double xd, double c, double cq, const F64Mod &m) {
  const double h = __dmul_rn(xd, c);
  const double l = __fma_rn(xd, c, -h);
  const double k = __dadd_rn(__fma_rn(xd, cq, F64_RINT_MAGIC), -F64_RINT_MAGIC);
  return __dadd_rn(__fma_rn(-k, m.q, h), l);
}
// v - rint(v / q) q: |result| <= q/2 (+1 when v/q is within 2^-53 relative of a half-integer)
DEVI double reduce_dd(double v, const F64Mod &m) {
  const double k = __dadd_rn(__fma_rn(v, m.qinv, F64_RINT_MAGIC), -F64_RINT_MAGIC);
  return __fma_rn(-k, m.q, v);
}
// a double holding an integer in [-off, 2^52 - off) -> that integer + off as u64 (off an integer below 2^52)
DEVI u64 d2u_off(double v, double off_magic /* off + 2^52 */) {
  return (u64)__double_as_longlong(__dadd_rn(v, off_magic)) & 0xFFFFFFFFFFFFFull;
}
DEVI u64 mulmod_f64(u64 x, u64 c_bits, u64 cq_bits, const F64Mod &m) {  // (0, 2q), the range of shoup_lazy
  const double t = mulmod_dd(u2d52(x), __longlong_as_double((long long)c_bits), __longlong_as_double((long long)cq_bits), m);
  return d2u_off(t, m.q + 4503599627370496.0);
}

// ---------------------------------------------------------------------------------------------- tile engine
// A pass transforms the active tile bits [lo, lo+nb) in radix-8 register rounds (3 stages per round) through
// swizzled shared memory.  FWD: Cooley-Tukey, high bit first.  INV: Gentleman-Sande, low bit first, values in [0,2q).
// Forward laziness: T = shoup_lazy(Y) is < 2q for ANY 64-bit Y, so X' = X + T and Y' = X - T + 2q grow by at most
// 2q per stage and need no correction while (1 + 2 log2 N) q < 2^64 (LAZY: q < 2^58); otherwise X is brought back
// below 2q in every butterfly (Harvey), keeping values below 4q.
// Indexing: a round's window [PW, PW+3) maps to contiguous global bits starting at gpw, so element k is global
// j0 + (k << gpw), its stage-s twiddle is tw[((N + j0) >> (gpw+s+1)) + (k >> (s+1))], and, swz being XOR-linear, its
// shared-memory slot is swz(ebase) ^ swz(k << PW): one base computation per thread and round.

// compile-time round: window position and active stages [SLO, SHI) are constants (production geometries)
// FIRST / LAST (fp64 rounds): whether this is the first / last round of the transform.  Between the rounds of one
// transform the tile holds the values as DOUBLES (signed, exact integers; reduced to at most q/2 in magnitude wherever a
// round ends with a reduction); only the first round converts from the unsigned words of the fill and only the last one
// back to the unsigned lazy words every consumer expects.  ncu on the fused column kernel (profiles/r02_cfg4_step_ncu.md):
// FP64 pipe 59 % busy, and a quarter of its FP64 instructions were these per-round conversions.
// TWS: `tw` points at a copy of the pass's twiddles in SHARED memory (a "slab", see tw_slab_fill) that the block filled
// once and reuses for every tile it transforms with these twiddles; the caller passes the geometry the copy is indexed
// by.  Without it every round fetches its seven twiddle pairs from L2 -- for a row pass 16 KB of twiddles per 8 KB tile,
// and the first multiply of every round waits for them (ncu, divide pass: 9 % of all stall samples on that one DFMA).
template <int TWS>
DEVI ulonglong2 tw_load(const ulonglong2 *p) {
  if constexpr (TWS != 0) return *p;
  else return __ldg(p);
}
// REGIN (first round only): the round's eight inputs come from registers, vin[k] = element ebase + (k << PW) of the tile
// (round_ebase<PW>(tid)), instead of shared memory: a kernel that loads the tile in that order skips the fill's stores,
// the round's loads and one barrier per tile.
template <int PW>
DEVI int round_ebase(int tid) { return ((tid >> PW) << (PW + 3)) | (tid & ((1 << PW) - 1)); }
// REGOUT (last round only): the round's eight results stay in registers, vout[k] = element ebase + (k << PW), in the
// form the round would have stored (unsigned lazy words); the caller drains them itself.
template <bool FWD, bool LAZY, int PW, int SLO, int SHI, int F64, bool FIRST = true, bool LAST = true, int TWS = 0, bool REGIN = false, bool REGOUT = false>  // F64: 0 integer, 1 fp64 narrow (q < 2^45), 2 fp64 wide
DEVI void tile_round_ct(u64 *sm, const TileGeo &G, const ShoupC *tw, u64 q, u64 q2, int tid, u64 f64, const u64 *vin = nullptr, u64 *vout = nullptr) {
  const int ebase = ((tid >> PW) << (PW + 3)) | (tid & ((1 << PW) - 1));
  const int gpw = G.gbit(PW);
  const u32 nj = (1u << G.logN) + G.gidx(ebase);
  const ulonglong2 *twv = reinterpret_cast<const ulonglong2 *>(tw);
  ulonglong2 t2 = make_ulonglong2(0, 0), t1[2], t0[4];
  // twiddles first: their L2 latency overlaps the shared-memory loads
  if (2 >= SLO && 2 < SHI) t2 = tw_load<TWS>(twv + (nj >> (gpw + 3)));
  if constexpr (TWS == 2 && PW == 0) {
    // row slab, round over the lowest bits: thread tid owns elements 8 tid .. 8 tid + 7, whose two (four) twiddles of
    // bit 1 (bit 0) are adjacent entries -- a stride of 32 (64) bytes between threads, a 2-way (4-way) bank conflict.
    // tw_slab_fill stores these two levels transposed, [i][tid], so each of the loads is unit-stride.
    const int nth = 1 << (G.logN - 3);
#pragma unroll
    for (int i = 0; i < 2; i++) t1[i] = (1 >= SLO && 1 < SHI) ? twv[(2 + i) * nth + tid] : t2;
#pragma unroll
    for (int i = 0; i < 4; i++) t0[i] = (0 >= SLO && 0 < SHI) ? twv[(4 + i) * nth + tid] : t2;
  } else {
#pragma unroll
    for (int i = 0; i < 2; i++) t1[i] = (1 >= SLO && 1 < SHI) ? tw_load<TWS>(twv + (nj >> (gpw + 2)) + i) : t2;
#pragma unroll
    for (int i = 0; i < 4; i++) t0[i] = (0 >= SLO && 0 < SHI) ? tw_load<TWS>(twv + (nj >> (gpw + 1)) + i) : t2;
  }
  const int sbase = swz(ebase);
  if constexpr (F64 != 0) {
    // The eight values stay doubles (signed, exact integers) through the round's stages; T is in (-q, q).
    // Narrow moduli (q < 2^45): a forward stage moves a value by less than q either way, so after the (at most 16) stages
    // of a pass a value that entered below 2^50 is below 2^50 + 16 q < 2^51 in magnitude, inside what the multiply
    // accepts, and no forward round reduces; an inverse round ends with v - rint(v/q) q (+ q in the last round: [0, 2q)).
    // Wide moduli (2^45 <= q < 2^50, compile-time schedules only): every round starts from values in [0, 2q], centred
    // to [-q, q] while converting, and ends with the same reduction in both directions; an operand that can exceed 2q
    // (third forward stage, second and third inverse stage) is reduced before it is multiplied, so the quotient
    // estimate stays below 2^51 and every sum below 2^53.
    const F64Mod fm = f64mod(q, f64);
    constexpr bool wide = F64 == 2;
    const double in_off = wide ? -(4503599627370496.0 + fm.q) : -4503599627370496.0;
    double x[8];
#pragma unroll
    for (int k = 0; k < 8; k++) {
      const u64 v = (REGIN && FIRST) ? vin[k] : sm[sbase ^ swz(k << PW)];
      x[k] = FIRST ? __dadd_rn(__hiloint2double((int)((u32)(v >> 32) | 0x43300000u), (int)(u32)v), in_off) : __longlong_as_double((long long)v);
    }
    int done = 0;
#pragma unroll
    for (int ss = 0; ss < 3; ss++) {
      const int s = FWD ? 2 - ss : ss;
      if (s < SLO || s >= SHI) continue;
      const bool pre = wide && (FWD ? done >= 2 : done >= 1);
      done++;
#pragma unroll
      for (int k = 0; k < 8; k++) {
        if (k & (1 << s)) continue;
        const int k2 = k | (1 << s);
        const ulonglong2 w = s == 2 ? t2 : (s == 1 ? t1[k >> 2] : t0[k >> 1]);
        const double c = __longlong_as_double((long long)w.x), cq = __longlong_as_double((long long)w.y);
        if (FWD) {
          const double X = x[k], Y = pre ? reduce_dd(x[k2], fm) : x[k2];
          const double T = mulmod_dd(Y, c, cq, fm);
          x[k] = __dadd_rn(X, T);
          x[k2] = __dadd_rn(X, -T);
        } else {
          const double U = x[k], V = x[k2];
          const double D = __dadd_rn(U, -V);
          x[k] = __dadd_rn(U, V);
          x[k2] = mulmod_dd(pre ? reduce_dd(D, fm) : D, c, cq, fm);
        }
      }
    }
    const bool red = !FWD || wide;
    if (LAST) {
      // narrow forward values are signed and have moved by less than q per stage since the fill (at most 16 stages): + 16 q
      // makes them non-negative and keeps them below 2^52; reduced values (+ q) land in (0, 2q)
      const double off = red ? __dadd_rn(fm.q, 4503599627370496.0) : __fma_rn(16.0, fm.q, 4503599627370496.0);
#pragma unroll
      for (int k = 0; k < 8; k++) {
        const u64 r = d2u_off(red ? reduce_dd(x[k], fm) : x[k], off);
        if (REGOUT) vout[k] = r;
        else sm[sbase ^ swz(k << PW)] = r;
      }
    } else {
#pragma unroll
      for (int k = 0; k < 8; k++) sm[sbase ^ swz(k << PW)] = (u64)__double_as_longlong(red ? reduce_dd(x[k], fm) : x[k]);
    }
  } else {
  u64 x[8];
#pragma unroll
  for (int k = 0; k < 8; k++) x[k] = (REGIN && FIRST) ? vin[k] : sm[sbase ^ swz(k << PW)];
#pragma unroll
  for (int ss = 0; ss < 3; ss++) {
    const int s = FWD ? 2 - ss : ss;
    if (s < SLO || s >= SHI) continue;
#pragma unroll
    for (int k = 0; k < 8; k++) {
      if (k & (1 << s)) continue;
      const int k2 = k | (1 << s);
      const ulonglong2 w = s == 2 ? t2 : (s == 1 ? t1[k >> 2] : t0[k >> 1]);
      if (FWD) {
        const u64 X = LAZY ? x[k] : csub(x[k], q2);
        const u64 T = shoup_lazy(x[k2], w.x, w.y, q);
        x[k] = X + T;
        x[k2] = X - T + q2;
      } else {
        const u64 U = x[k], V = x[k2];
        x[k] = csub(U + V, q2);
        x[k2] = shoup_lazy(U - V + q2, w.x, w.y, q);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < 8; k++) {
    if (REGOUT && LAST) vout[k] = x[k];
    else sm[sbase ^ swz(k << PW)] = x[k];
  }
  }
}

// GRP: the tile belongs to a 128-thread group of a larger block; its rounds meet on the named barrier `bar` (1..15)
template <bool GRP>
DEVI void tile_sync(int bar) {
  if constexpr (GRP) asm volatile("bar.sync %0, 128;" ::"r"(bar) : "memory");
  else __syncthreads();
}
struct NoAfter { DEVI void operator()() const {} };
// AF: called by every thread right after the first round (a REGIN caller requests the next tile into the registers the
// round has just consumed)
template <bool FWD, bool LAZY, int LT, int LO, int NB, int DONE, int F64 = 0, bool GRP = false, int TWS = 0, bool REGIN = false, class AF = NoAfter, bool REGOUT = false>
DEVI void tile_rounds_ct(u64 *sm, const TileGeo &G, const ShoupC *tw, u64 q, u64 q2, int tid, u64 f64 = 0, int bar = 0, const u64 *vin = nullptr, AF af = AF(), u64 *vout = nullptr) {
  if constexpr (DONE < NB) {
    constexpr int take = NB - DONE < 3 ? NB - DONE : 3;
    constexpr int cur = FWD ? LO + NB - DONE : LO + DONE;         // FWD: exclusive top; INV: inclusive bottom
    constexpr int p = FWD ? cur - take : cur;
    constexpr int pw = p < LT - 3 ? p : LT - 3;
    constexpr bool last = DONE + take >= NB;
    if (tid < (1 << (LT - 3))) tile_round_ct<FWD, LAZY, pw, p - pw, p - pw + take, F64, DONE == 0, last, TWS, REGIN, REGOUT>(sm, G, tw, q, q2, tid, f64, vin, vout);
    if constexpr (DONE == 0) af();
    if constexpr (!(REGOUT && last)) tile_sync<GRP>(bar);  // (a REGOUT caller synchronises before the tile is written again)
    tile_rounds_ct<FWD, LAZY, LT, LO, NB, DONE + take, F64, GRP, TWS, false, NoAfter, REGOUT>(sm, G, tw, q, q2, tid, f64, bar, nullptr, NoAfter(), vout);
  }
}
// window position of the LAST round of a compile-time schedule (the order a REGOUT caller drains in)
template <bool FWD, int LT, int LO, int NB>
struct LastRound {
  static constexpr int rem = NB % 3 == 0 ? 3 : NB % 3;                 // stages of the last round
  static constexpr int p = FWD ? LO : LO + NB - rem;
  static constexpr int pw = p < LT - 3 ? p : LT - 3;
};
// window position of the FIRST round of a compile-time schedule (the order a REGIN caller loads the tile in)
template <bool FWD, int LT, int LO, int NB>
struct FirstRound {
  static constexpr int take = NB < 3 ? NB : 3, p = FWD ? LO + NB - take : LO;
  static constexpr int pw = p < LT - 3 ? p : LT - 3;
};

// runtime round (toy ring degrees and any geometry without a compile-time instance)
template <bool FWD, bool F64>
DEVI void tile_round_rt(u64 *sm, const TileGeo &G, int pw, int s_lo, int s_hi, const ShoupC *tw, u64 q, u64 q2, int tid, u64 f64) {
  const F64Mod fm = f64mod(q, f64);
  const int ebase = ((tid >> pw) << (pw + 3)) | (tid & ((1 << pw) - 1));
  u64 x[8];
#pragma unroll
  for (int k = 0; k < 8; k++) x[k] = sm[swz(ebase | (k << pw))];
  const u32 nj = (1u << G.logN) + G.gidx(ebase);
  const int gpw = G.gbit(pw);
#pragma unroll
  for (int ss = 0; ss < 3; ss++) {
    const int s = FWD ? 2 - ss : ss;
    if (s < s_lo || s >= s_hi) continue;
#pragma unroll
    for (int k = 0; k < 8; k++) {
      if (k & (1 << s)) continue;
      const int k2 = k | (1 << s);
      const ShoupC w = tw[(nj >> (gpw + s + 1)) + (k >> (s + 1))];
      if (FWD) {
        u64 X = csub(x[k], q2);
        u64 T = F64 ? mulmod_f64(x[k2], w.c, w.cs, fm) : shoup_lazy(x[k2], w.c, w.cs, q);
        x[k] = X + T;
        x[k2] = X - T + q2;
      } else {
        u64 U = x[k], V = x[k2];
        x[k] = csub(U + V, q2);
        x[k2] = F64 ? mulmod_f64(U - V + q2, w.c, w.cs, fm) : shoup_lazy(U - V + q2, w.c, w.cs, q);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < 8; k++) sm[swz(ebase | (k << pw))] = x[k];
}

// compile-time schedule over active tile bits [LO, LO+NB) of a 2^LT-element tile; picks the lazy forward butterflies
// for q < 2^58.  Every thread of the block must call this (it synchronises).
template <bool FWD, int LT, int LO, int NB, bool GRP = false, int TWS = 0, bool REGIN = false, bool REGOUT = false>
DEVI void tile_transform_ct(u64 *sm, const TileGeo &G, const ShoupC *tw, u64 q, int tid, u64 f64, int bar = 0, const u64 *vin = nullptr, u64 *vout = nullptr) {
  const u64 q2 = q + q;
  if (f64 && q < (1ull << FENC_F64_MAX_BITS)) tile_rounds_ct<FWD, true, LT, LO, NB, 0, 1, GRP, TWS, REGIN, NoAfter, REGOUT>(sm, G, tw, q, q2, tid, f64, bar, vin, NoAfter(), vout);
  else if (f64) tile_rounds_ct<FWD, true, LT, LO, NB, 0, 2, GRP, TWS, REGIN, NoAfter, REGOUT>(sm, G, tw, q, q2, tid, f64, bar, vin, NoAfter(), vout);
  else if (FWD && q < (1ull << 58)) tile_rounds_ct<FWD, true, LT, LO, NB, 0, 0, GRP, TWS, REGIN, NoAfter, REGOUT>(sm, G, tw, q, q2, tid, 0, bar, vin, NoAfter(), vout);
  else tile_rounds_ct<FWD, false, LT, LO, NB, 0, 0, GRP, TWS, REGIN, NoAfter, REGOUT>(sm, G, tw, q, q2, tid, 0, bar, vin, NoAfter(), vout);
}

// The twiddles of a ROW pass over the 2^LT contiguous coefficients of tile `tile`, copied to shared memory in heap order:
// slab[(2^LT + e) >> (g + 1)] is the twiddle of global bit g (0 <= g < LT) for the tile-local element e, i.e. entry
// idx in [2^lvl, 2^(lvl+1)) is tw[((N + tile 2^LT) >> (LT - lvl)) + idx - 2^lvl].  A round indexes the slab exactly as it
// indexes the table when it is given the geometry row_slab_geo(): ring degree 2^LT, tile 0 -- except the two lowest
// levels (bits 1 and 0), which are stored transposed for the round over the lowest bits (TWS = 2 in tile_round_ct): entry
// 2^(LT-2) + 2 t + i sits at (2 + i) 2^(LT-3) + t and entry 2^(LT-1) + 4 t + i at (4 + i) 2^(LT-3) + t.
// 2^LT entries of 16 bytes (entry 0 unused), copied with cp.async: the caller commits, waits and synchronises before the
// first transform.
DEVI void cp_async8(u64 *dst_smem, const u64 *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((u32)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
DEVI void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
DEVI void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
DEVI void cp_async16(void *dst_smem, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
template <int LT>
DEVI void tw_slab_fill(ShoupC *slab, const ShoupC *tw, int logN, u32 tile, int tid, int nth) {
  constexpr int NT8 = 1 << (LT - 3);
  const u32 base = (1u << logN) + (tile << LT);
  for (int idx = tid; idx < (1 << LT); idx += nth) {
    if (idx == 0) continue;
    const int lvl = 31 - __clz(idx), loc = idx - (1 << lvl);
    const int pos = lvl == LT - 1 ? (4 + (loc & 3)) * NT8 + (loc >> 2) : (lvl == LT - 2 ? (2 + (loc & 1)) * NT8 + (loc >> 1) : idx);
    cp_async16(slab + pos, tw + (base >> (LT - lvl)) + loc);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
}
DEVI void tw_slab_wait() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
template <int LT>
DEVI TileGeo row_slab_geo() { return TileGeo{LT, LT, 0, LT, 0}; }

// GEO selects the schedule: 0 = runtime (any lo/nb), 1 = row pass of 2048-element tiles with 8 stages,
// 4..8 = column pass with GEO stages over tiles of 2^(GEO+4) elements (16 columns).
// Every thread of the block must call this (it synchronises).  Outputs: forward < 33q (use fullred), inverse < 2q.
template <bool FWD, int GEO, int TWS = 0, bool REGIN = false, class AF = NoAfter, bool REGOUT = false>
DEVI void tile_transform(u64 *sm, const TileGeo &G, int lo, int nb, const ShoupC *tw, u64 q, int tid, u64 f64, const u64 *vin = nullptr, AF af = AF(), u64 *vout = nullptr) {
  const u64 q2 = q + q;
  static_assert(!((TWS || REGIN) && GEO == 0), "twiddle slabs and register inputs exist for the compile-time schedules only");
  if constexpr (GEO == 0) {
    const bool active = tid < (1 << (G.lt - 3));
    if (FWD) {
      int cur = lo + nb;
      while (cur > lo) {
        int take = cur - lo < 3 ? cur - lo : 3;
        int p = cur - take;
        int pw = p < G.lt - 3 ? p : G.lt - 3;
        if (active) { if (f64) tile_round_rt<true, true>(sm, G, pw, p - pw, cur - pw, tw, q, q2, tid, f64); else tile_round_rt<true, false>(sm, G, pw, p - pw, cur - pw, tw, q, q2, tid, 0); }
        __syncthreads();
        cur = p;
      }
    } else {
      int cur = lo;
      while (cur < lo + nb) {
        int take = lo + nb - cur < 3 ? lo + nb - cur : 3;
        int pw = cur < G.lt - 3 ? cur : G.lt - 3;
        if (active) { if (f64) tile_round_rt<false, true>(sm, G, pw, cur - pw, cur + take - pw, tw, q, q2, tid, f64); else tile_round_rt<false, false>(sm, G, pw, cur - pw, cur + take - pw, tw, q, q2, tid, 0); }
        __syncthreads();
        cur += take;
      }
    }
  } else {
    constexpr int LT = GEO == 1 ? FENC_ROW_LT : GEO + 4, LO = GEO == 1 ? 0 : 4, NB = GEO == 1 ? 8 : GEO;
    if (f64 && q < (1ull << FENC_F64_MAX_BITS)) tile_rounds_ct<FWD, true, LT, LO, NB, 0, 1, false, TWS, REGIN, AF, REGOUT>(sm, G, tw, q, q2, tid, f64, 0, vin, af, vout);
    else if (f64) tile_rounds_ct<FWD, true, LT, LO, NB, 0, 2, false, TWS, REGIN, AF, REGOUT>(sm, G, tw, q, q2, tid, f64, 0, vin, af, vout);
    else if (FWD && q < (1ull << 58)) tile_rounds_ct<FWD, true, LT, LO, NB, 0, 0, false, TWS, REGIN, AF, REGOUT>(sm, G, tw, q, q2, tid, 0, 0, vin, af, vout);
    else tile_rounds_ct<FWD, false, LT, LO, NB, 0, 0, false, TWS, REGIN, AF, REGOUT>(sm, G, tw, q, q2, tid, 0, 0, vin, af, vout);
  }
}
