// fenc_elem.cu -- element-wise kernels of the hot path: plaintext MAC (a7), the scalar MAC of factored weights (R2.9c),
// ciphertext sums, encrypt / decrypt combines, the counter-based samplers (R2.3) and Montgomery-form
// conversions.  sm_100a.  Limb-major, one pass; the sums, the streaming scalar MAC and the hoisted inner product use
// 16-byte accesses, the grouped MACs 8-byte ones (one coefficient per thread, up to 8 outputs per loaded word).
#include "fenc_device.cuh"

#define PROF(k, id, bytes) if ((k).prof) prof_begin((k).prof, (k).stream, id, (double)(bytes))
#define PROF2(k, id, bytes, ops) if ((k).prof) prof_begin((k).prof, (k).stream, id, (double)(bytes), (double)(ops))
#define LAUNCH_CHECK(k)                            \
  do {                                             \
    (*(k).launches)++;                             \
    if ((k).prof) prof_end((k).prof, (k).stream);  \
    cudaError_t e__ = cudaGetLastError();          \
    if (e__ != cudaSuccess) return (int)e__;       \
  } while (0)

static inline cudaStream_t S(const KCtx &k) { return (cudaStream_t)k.stream; }

// ------------------------------------------------------------------------------------------------ MAC (a7)
// A group = up to G outputs that read the SAME ciphertext sequence with different plaintexts (the output channel
// groups of one fragment and diagonal): each ciphertext word is loaded once and multiplied into G accumulators
// (register tiling), each plaintext word is read once.  out[i][c][l][n] = sum_t ct_t[c][l][n] * pt_{i,t}[l][n];
// products accumulate in 128 bits and are reduced once per max_lazy terms (max_lazy = floor(2^64 / q_max) keeps the
// accumulator below q 2^64).  Blocks of one coefficient chunk are adjacent across groups (blockIdx.x = group), so
// plaintexts shared by neighbouring groups (deduplicated weights) are served from L2.
struct MacP {
  const MacGroup *groups; const u64 *const *term_ct; const u64 *const *term_pt; u64 *const *outs; const ModConst *mods;
  int L, logN, max_lazy;
};
#define MAC_TILE 64  // terms whose pointers are staged in shared memory at a time
// Accumulation modes (chosen from the largest modulus in use):
//  MODE 0  any modulus: x w accumulated in 128 bits (mad.lo.cc / madc.hi), reduced every max_lazy terms.
//  MODE 1  moduli < 2^52: operands split in 26-bit limbs, x = x1 2^26 + x0; the partial sums sum x0 w0,
//          sum (x0 w1 + x1 w0), sum x1 w1 are plain 64-bit integers (IMAD.WIDE, no carries), recombined once per flush.
//  MODE 2  moduli < 2^40: 20-bit limbs held as DOUBLES; every product (< 2^40) and every partial sum (< 2^53 for up to
//          2048 terms) is exact in fp64, so the partial sums are accumulated by DFMA.  Measured on B200: DFMA issues at
//          64 lanes/clk/SM, IMAD.WIDE with a 64-bit addend at about 25, and the two use different pipes from the
//          integer ALU that does the limb splitting.
struct Acc3 { u64 a0, a1, a2; };
// (mad.wide.u32 spelled out: left to itself the compiler sums the two middle products first and adds them with a
// carry chain, twice the instructions)
DEVI void madw(u64 &acc, u32 a, u32 b) { asm("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc) : "r"(a), "r"(b)); }
DEVI void acc3_mac(Acc3 &A, u32 x0, u32 x1, u32 w0, u32 w1) {
  madw(A.a0, x0, w0);
  madw(A.a1, x0, w1);
  madw(A.a1, x1, w0);
  madw(A.a2, x1, w1);
}
template <int SH>
DEVI u64 limbs_redc(u64 a0, u64 a1, u64 a2, u64 q, u64 qinv_neg) {  // (a0 + a1 2^SH + a2 2^2SH) 2^-64 mod q
  u64 lo = a0, hi = 0, t;
  t = a1 << SH; lo += t; hi += (a1 >> (64 - SH)) + (lo < t ? 1 : 0);
  t = a2 << (2 * SH); lo += t; hi += (a2 >> (64 - 2 * SH)) + (lo < t ? 1 : 0);
  return mont_redc(lo, hi, q, qinv_neg);
}
struct AccD { double a0, a1, a2; };
DEVI double u2d(u32 v) { return __hiloint2double(0x43300000, (int)v) - 4503599627370496.0; }  // exact, v < 2^32
DEVI void accd_mac(AccD &A, double x0, double x1, double w0, double w1) {
  A.a0 = fma(x0, w0, A.a0);
  A.a1 = fma(x0, w1, A.a1);
  A.a1 = fma(x1, w0, A.a1);
  A.a2 = fma(x1, w1, A.a2);
}
template <int G, int MODE>
struct MacState {
  u64 lo0[MODE == 0 ? G : 1], hi0[MODE == 0 ? G : 1], lo1[MODE == 0 ? G : 1], hi1[MODE == 0 ? G : 1];
  Acc3 A0[MODE == 1 ? G : 1], A1[MODE == 1 ? G : 1];
  AccD D0[MODE == 2 ? G : 1], D1[MODE == 2 ? G : 1];
  int lazy, max_lazy;
  DEVI void set(int i, u64 v0, u64 v1) {  // accumulators := the small integers v0, v1
    if (MODE == 0) lo0[i] = v0, lo1[i] = v1, hi0[i] = hi1[i] = 0;
    if (MODE == 1) A0[i] = Acc3{v0, 0, 0}, A1[i] = Acc3{v1, 0, 0};
    if (MODE == 2) D0[i] = AccD{(double)v0, 0, 0}, D1[i] = AccD{(double)v1, 0, 0};
  }
  DEVI void init(int ctx_max_lazy) {
#pragma unroll
    for (int i = 0; i < G; i++) set(i, 0, 0);
    // one slot of every bound is left for the folded-back residue (< q)
    max_lazy = MODE == 0 ? ctx_max_lazy - 1 : (MODE == 1 ? 1023 : 2047);
    if (max_lazy < 1) max_lazy = 1;
    lazy = 0;
  }
  // the pending sum S as S 2^-64 mod q (canonical)
  DEVI u64 out0(int i, const ModConst &mc) const {
    if (MODE == 0) return mont_redc(lo0[i], hi0[i], mc.q, mc.qinv_neg);
    if (MODE == 1) return limbs_redc<26>(A0[i].a0, A0[i].a1, A0[i].a2, mc.q, mc.qinv_neg);
    return limbs_redc<20>((u64)D0[i].a0, (u64)D0[i].a1, (u64)D0[i].a2, mc.q, mc.qinv_neg);
  }
  DEVI u64 out1(int i, const ModConst &mc) const {
    if (MODE == 0) return mont_redc(lo1[i], hi1[i], mc.q, mc.qinv_neg);
    if (MODE == 1) return limbs_redc<26>(A1[i].a0, A1[i].a1, A1[i].a2, mc.q, mc.qinv_neg);
    return limbs_redc<20>((u64)D1[i].a0, (u64)D1[i].a1, (u64)D1[i].a2, mc.q, mc.qinv_neg);
  }
  DEVI void mac(u64 x0, u64 x1, const u64 (&w)[G], const ModConst &mc) {
    if (MODE == 0) {
#pragma unroll
      for (int i = 0; i < G; i++) mac128(lo0[i], hi0[i], x0, w[i]), mac128(lo1[i], hi1[i], x1, w[i]);
    } else if (MODE == 1) {
      const u32 m = (1u << 26) - 1;
      const u32 x00 = (u32)x0 & m, x01 = (u32)(x0 >> 26), x10 = (u32)x1 & m, x11 = (u32)(x1 >> 26);
#pragma unroll
      for (int i = 0; i < G; i++) {
        const u32 w0 = (u32)w[i] & m, w1 = (u32)(w[i] >> 26);
        acc3_mac(A0[i], x00, x01, w0, w1);
        acc3_mac(A1[i], x10, x11, w0, w1);
      }
    } else {
      const u32 m = (1u << 20) - 1;
      const double x00 = u2d((u32)x0 & m), x01 = u2d((u32)(x0 >> 20)), x10 = u2d((u32)x1 & m), x11 = u2d((u32)(x1 >> 20));
#pragma unroll
      for (int i = 0; i < G; i++) {
        const double w0 = u2d((u32)w[i] & m), w1 = u2d((u32)(w[i] >> 20));
        accd_mac(D0[i], x00, x01, w0, w1);
        accd_mac(D1[i], x10, x11, w0, w1);
      }
    }
    if (++lazy == max_lazy) {
      // fold: S 2^-64 mod q times 2^128 2^-64 = S mod q, a residue below q, becomes the new pending sum
#pragma unroll
      for (int i = 0; i < G; i++)
        set(i, mont_mul(out0(i, mc), mc.r2, mc.q, mc.qinv_neg), mont_mul(out1(i, mc), mc.r2, mc.q, mc.qinv_neg));
      lazy = 0;
    }
  }
};

#ifndef MAC_THREADS
#define MAC_THREADS 256
#endif
#ifndef MAC_RING
#define MAC_RING 3  // terms whose operands are in flight per thread (36 KiB of shared memory at 4 outputs per group)
#endif
DEVI void mac_cp_async8(u64 *dst_smem, const u64 *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((u32)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
template <int G, int MODE>
__global__ void __launch_bounds__(MAC_THREADS, 512 / MAC_THREADS) mac_kernel(MacP p) {
  __shared__ const u64 *s_ct[MAC_TILE];
  __shared__ const u64 *s_pt[G][MAC_TILE];
  __shared__ u64 s_ring[MODE == 2 ? 1 : MAC_RING][MODE == 2 ? 1 : 2 + G][MODE == 2 ? 1 : MAC_THREADS];
  const size_t LN = (size_t)p.L << p.logN;
  const size_t idx = (size_t)blockIdx.y * blockDim.x + threadIdx.x;
  const bool live = idx < LN;
  const MacGroup g = p.groups[blockIdx.x];
  const ModConst mc = p.mods[(live ? idx : 0) >> p.logN];
  MacState<G, MODE> st;
  st.init(p.max_lazy);
  for (int t0 = 0; t0 < g.n_terms; t0 += MAC_TILE) {
    const int nt = g.n_terms - t0 < MAC_TILE ? g.n_terms - t0 : MAC_TILE;
    __syncthreads();
    for (int j = threadIdx.x; j < nt * (G + 1); j += blockDim.x) {
      const int i = j / nt, t = j - i * nt;
      if (i == 0) s_ct[t] = p.term_ct[g.ct_start + t0 + t];
      else if (i - 1 < g.n_out) s_pt[i - 1][t] = p.term_pt[g.pt_start + (i - 1) * g.n_terms + t0 + t];
      else s_pt[i - 1][t] = p.term_pt[g.pt_start + t0 + t];  // unused lanes of a short group: any valid pointer
    }
    __syncthreads();
    if (!live) continue;
    // Integer modes (0, 1): the operands of the next MAC_RING - 1 terms are in flight while this term's products run, in a
    // per-thread cp.async ring in shared memory (every thread owns its slots: no barrier, no registers spent on the depth):
    // config 3's 26-bit-limb MAC -11 %.  The fp64 mode (2) keeps plain loads in batches of three terms.  ncu (config 2's
    // conv2, profiles/r02_late_captures.md): half of all stall samples sit on the first use of a loaded word, the FP64 pipe
    // is 41 % busy.  Measured against batches of two (2.40 ms of MAC per LeNet-5 step): batches of three 2.08 ms, of four
    // 2.41 ms; the ring +8 % (its shared-memory wavefronts compete with the loads); three register sets with the loads of
    // terms t+1, t+2 requested before term t's products 3.44 ms; groups of two outputs at three blocks per SM 2.59 ms; one
    // ciphertext component per thread (half the accumulators, up to twice the warps) 2.97-5.03 ms; 4-64 consecutive
    // coefficient chunks per group in the block order 2.11-2.47 ms.  More warps or more requests in flight make it slower.
    if (MODE == 2) {
#pragma unroll 3
      for (int t = 0; t < nt; t++) {
        const u64 *c = s_ct[t];
        const u64 x0 = __ldg(c + idx), x1 = __ldg(c + LN + idx);
        u64 w[G];
#pragma unroll
        for (int i = 0; i < G; i++) w[i] = __ldg(s_pt[i][t] + idx);
        st.mac(x0, x1, w, mc);
      }
      continue;
    }
    auto ring_issue = [&](int t) {
      if (t < nt) {
        const u64 *c = s_ct[t];
        mac_cp_async8(&s_ring[t % MAC_RING][0][threadIdx.x], c + idx);
        mac_cp_async8(&s_ring[t % MAC_RING][1][threadIdx.x], c + LN + idx);
#pragma unroll
        for (int i = 0; i < G; i++) mac_cp_async8(&s_ring[t % MAC_RING][2 + i][threadIdx.x], s_pt[i][t] + idx);
      }
      asm volatile("cp.async.commit_group;" ::: "memory");  // one group per term, empty past the end
    };
#pragma unroll
    for (int t = 0; t < MAC_RING - 1; t++) ring_issue(t);
#pragma unroll 2
    for (int t = 0; t < nt; t++) {
      ring_issue(t + MAC_RING - 1);  // overwrites the slot of term t - 1, already consumed by this thread
      asm volatile("cp.async.wait_group %0;" ::"n"(MAC_RING - 1) : "memory");
      const u64 x0 = s_ring[t % MAC_RING][0][threadIdx.x], x1 = s_ring[t % MAC_RING][1][threadIdx.x];
      u64 w[G];
#pragma unroll
      for (int i = 0; i < G; i++) w[i] = s_ring[t % MAC_RING][2 + i][threadIdx.x];
      st.mac(x0, x1, w, mc);
    }
  }
  if (!live) return;
#pragma unroll
  for (int i = 0; i < G; i++) {
    if (i < g.n_out) {
      u64 *out = p.outs[g.out_start + i];
      out[idx] = st.out0(i, mc);
      out[LN + idx] = st.out1(i, mc);
    }
  }
}
template <int MODE>
static void launch_mac(const MacP &p, dim3 grid, cudaStream_t st, int max_group) {
  if (max_group <= 1) mac_kernel<1, MODE><<<grid, MAC_THREADS, 0, st>>>(p);
  else if (max_group <= 2) mac_kernel<2, MODE><<<grid, MAC_THREADS, 0, st>>>(p);
  else mac_kernel<4, MODE><<<grid, MAC_THREADS, 0, st>>>(p);
}

// q_max = largest modulus among the L limbs in use (selects the accumulation mode)
int k_mac(const KCtx &k, const MacGroup *groups, int n_groups, int max_group, const u64 *const *term_ct, const u64 *const *term_pt,
          u64 *const *outs, int L, int max_lazy, u64 q_max, double alg_bytes) {
  if (n_groups == 0) return 0;
  MacP p{groups, term_ct, term_pt, outs, k.d_mods, L, k.geom.logN, max_lazy};
  dim3 grid(n_groups, (unsigned)(((size_t)L * k.N + MAC_THREADS - 1) / MAC_THREADS));
  PROF(k, K_MAC, alg_bytes);
  static const int force_mode = getenv("FENC_MAC_MODE") ? atoi(getenv("FENC_MAC_MODE")) : -1;  // diagnostics: a more general mode
  int mode = q_max < (1ull << 40) ? 2 : (q_max < (1ull << 52) ? 1 : 0);
  if (force_mode >= 0 && force_mode < mode) mode = force_mode;
  if (mode == 2) launch_mac<2>(p, grid, S(k), max_group);
  else if (mode == 1) launch_mac<1>(p, grid, S(k), max_group);
  else launch_mac<0>(p, grid, S(k), max_group);
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ scalar MAC (factored weights, R2.9c)
// out_i = sum over mask segments s of  M_s (*) ( sum_{t in s} k_{i,t} . ct_t ),  k an integer scalar per (weight, limb).
// A group = up to G outputs reading one ciphertext sequence with one segmentation (the output channels of one fragment):
// each ciphertext word is loaded once and multiplied into G x 2 accumulators -- a register-tiled modular GEMM whose
// "weights" are L words per scalar instead of L N words per plaintext.  The scalars of the block's limb are staged in
// shared memory (a block never straddles limbs), the products run on the FP64 pipe when every modulus in use is below
// 2^50: t = x k - rint(x k / q) q is an exact integer in (-q, q) (fenc_device.cuh mulmod_dd, |x| < 2^51), a sum of
// floor(2^53 / q) - 1 of them plus a reduced remainder (at most q/2 + 1 in magnitude) is exact in a double, then
// v - rint(v / q) q brings it back.  Integer mode (larger moduli): 128-bit lazy sums of x k_mont as in the plaintext MAC.
// Split modes (MODE 2, 3; moduli below 2^50 and small multipliers): the multiplier of a factored weight is the integer
// k = round_half_up(v E1), a SMALL signed number (|k| < 2^26 for |v| < 2 at E1 = 2^25), not a 50-bit quantity -- only its
// residue is.  With the ciphertext word split in P pieces of B bits, x = sum_p x_p 2^(pB), every product x_p k is below
// 2^B kmax and `max_lazy` of them sum EXACTLY in a double by plain DFMA: P DFMA per multiply-accumulate (2 for B = 25,
// 3 for B = 17) instead of the 7 operations of an exact 50 x 50-bit product, the pieces' conversions shared by the G
// outputs.  A mask segment ends with S = S_0 + S_1 2^B (+ S_2 2^2B) mod q (one or two exact products per accumulator).
// The residues are those of MODE 1 (k and k mod q differ by a multiple of q), so the outputs are bit-identical.
struct SmacP {
  const SmacGroup *groups; const u64 *const *term_ct; const int *kidx; const ShoupC *kpair; const int *seg_end;
  const u64 *const *seg_mask; u64 *const *outs; const ModConst *mods; int L, logN, max_lazy;
  int signed_k;  // kpair entries hold {(double) k, 0} with k the SIGNED multiplier (split modes) instead of {k mod q, (k mod q) / q}
  int cpb;       // consecutive coefficient chunks (of blockDim.x words, all in one limb) a block of smac_kernel walks over
};
#define SMAC_TILE 64
#ifndef SMAC_RING
#define SMAC_RING 4  // terms whose ciphertext words are in flight per thread (grouped kernel)
#endif
DEVI void smac_cp_async8(u64 *dst_smem, const u64 *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((u32)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
template <int G, int MODE>  // MODE 0: 128-bit integer sums; 1: exact fp64 products of residues; 2 / 3: split modes with 2 x 25 / 3 x 17 bits
__global__ void __launch_bounds__(256, (G >= 8 || MODE == 3) ? 2 : 3) smac_kernel(SmacP p) {
  constexpr bool F64 = MODE == 1;
  constexpr bool SPLIT = MODE >= 2;
  constexpr int NP = MODE == 3 ? 3 : 2, PB = MODE == 3 ? 17 : 25;  // pieces and bits per piece (split modes)
  // TS (groups of 4 and more outputs): the running totals over the mask segments live in shared memory (dynamic, one slot
  // per thread, output and component), touched at segment ends only.  In registers they took 4 G of the 128 a thread may
  // have beside the 4 G (6 G) accumulators, and the compiler rebuilt every loop invariant (thread index, limb offset,
  // ring addresses) in every term: 106 instructions per term around 32 DFMA (ncu, profiles/r02_late_captures.md).
  constexpr bool TS = G >= 4;
  extern __shared__ u64 s_tot[];  // TS: [G][2][blockDim.x]
  __shared__ const u64 *s_ct[SMAC_TILE];
  __shared__ ulonglong2 s_k[SPLIT ? 1 : G][SPLIT ? 1 : SMAC_TILE];
  __shared__ __align__(16) double s_kd[SPLIT ? SMAC_TILE : 1][SPLIT ? G : 1];  // split modes: the G multipliers of a term side by side
  __shared__ u64 s_ring[G >= 4 ? SMAC_RING : 1][2][G >= 4 ? 256 : 1];
  const u32 LN = (u32)p.L << p.logN;                           // L N < 2^32 (at most 2^7 limbs of 2^17 coefficients)
  // a block walks over p.cpb consecutive chunks of one limb: the pointers and multipliers of a group of at most SMAC_TILE
  // terms are staged once for all of them (a block of the pointwise layers lives for 32-64 terms only; ncu: 7 % of its
  // stall samples on the staging's dependent loads and barrier)
  u32 idx = blockIdx.y * p.cpb * blockDim.x + threadIdx.x;     // blockDim divides N: idx < L N, one limb per block
  const int limb = (int)((blockIdx.y * p.cpb * blockDim.x) >> p.logN);
  const SmacGroup g = p.groups[blockIdx.x];
  const ModConst mc = p.mods[limb];
  F64Mod fm = f64mod(mc.q, mc.f64);
  if (G >= 4) {  // (double) q is an integer-to-double conversion the compiler otherwise repeats per term
    asm volatile("mov.f64 %0, %0;" : "+d"(fm.q));
    asm volatile("mov.f64 %0, %0;" : "+d"(fm.qinv));
  }
  double acc[F64 ? G : 1][2];
  double sp[SPLIT ? G : 1][2][NP];
  u64 lo[MODE == 0 ? G : 1][2], hi[MODE == 0 ? G : 1][2], tot[TS ? 1 : G][2];
  for (int cc = 0; cc < p.cpb; cc++, idx += blockDim.x) {
#pragma unroll
  for (int i = 0; i < G; i++) {
    if (!TS) tot[i][0] = tot[i][1] = 0;
    if (F64) acc[i][0] = acc[i][1] = 0.0;
    if (MODE == 0) lo[i][0] = lo[i][1] = hi[i][0] = hi[i][1] = 0;
    if (SPLIT) {
#pragma unroll
      for (int c = 0; c < 2; c++)
#pragma unroll
        for (int q2 = 0; q2 < NP; q2++) sp[i][c][q2] = 0.0;
    }
  }
  u32 a_ring = (u32)__cvta_generic_to_shared(&s_ring[0][0][G >= 4 ? threadIdx.x : 0]);
  u32 a_ct = (u32)__cvta_generic_to_shared(&s_ct[0]);
  u32 idx_r = idx, ln_r = LN + idx, a_kd = (u32)__cvta_generic_to_shared(&s_kd[0][0]);
  if (G >= 4) {
    asm volatile("mov.u32 %0, %0;" : "+r"(a_kd));  // opaque copies: values the compiler must keep in registers instead of rebuilding them from special registers per term
    asm volatile("mov.u32 %0, %0;" : "+r"(a_ring));
    asm volatile("mov.u32 %0, %0;" : "+r"(a_ct));
    asm volatile("mov.u32 %0, %0;" : "+r"(idx_r));
    asm volatile("mov.u32 %0, %0;" : "+r"(ln_r));
  }
  int seg = 0, cur_end = p.seg_end[g.seg_start], lazy = 0;
  for (int t0 = 0; t0 < g.n_terms; t0 += SMAC_TILE) {
    const int nt = g.n_terms - t0 < SMAC_TILE ? g.n_terms - t0 : SMAC_TILE;
    if (cc == 0 || g.n_terms > SMAC_TILE) {  // a single tile of terms stays staged for the block's later chunks
    __syncthreads();
    for (int j = threadIdx.x; j < nt * (G + 1); j += blockDim.x) {
      const int i = j / nt, t = j - i * nt;
      if (i == 0) s_ct[t] = p.term_ct[g.ct_start + t0 + t];
      else {
        const int o = i - 1 < g.n_out ? i - 1 : 0;  // unused lanes of a short group repeat output 0 (never stored)
        const int w = p.kidx[g.k_start + o * g.n_terms + t0 + t];
        const ulonglong2 kk = __ldg(reinterpret_cast<const ulonglong2 *>(p.kpair) + (size_t)w * p.L + limb);
        if (SPLIT) s_kd[t][i - 1] = __longlong_as_double((long long)kk.x);
        else s_k[i - 1][t] = kk;
      }
    }
    __syncthreads();
    }
    // the next term's ciphertext words are requested before this term's products (register double buffer): with two blocks
    // of 8 warps per SM the loads would otherwise sit in front of 112 dependent FP64 operations
    // Groups of 4 and more outputs: the ciphertext words of the next SMAC_RING - 1 terms are in flight while this term's
    // products run.  A term's arithmetic (about 300 clocks per scheduler with four warps) is shorter than an L2 / HBM
    // round trip, so with one term ahead the loop ran at the memory latency (measured: 2 TB/s of operand traffic, a
    // quarter of what the FP64 pipe would allow).  The ring lives in shared memory (cp.async, 8 bytes per copy): each
    // thread owns its slots, so no barrier is needed and no register is spent on the depth.
    // (shared-memory addresses as 32-bit window offsets computed once: left to the compiler, the generic-to-shared
    // conversions of the ring slots were redone in every term)
    auto ring_issue = [&](int t) {
      if (t < nt) {
        u64 c;
        asm volatile("ld.shared.u64 %0, [%1];" : "=l"(c) : "r"(a_ct + (u32)t * 8u));
        const u32 slot = a_ring + ((u32)t % SMAC_RING) * (u32)(2 * 256 * sizeof(u64));
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(slot), "l"(c + (u64)idx_r * 8u) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(slot + (u32)(256 * sizeof(u64))), "l"(c + (u64)ln_r * 8u) : "memory");
      }
      asm volatile("cp.async.commit_group;" ::: "memory");  // a group per term, empty past the end: the wait below counts groups
    };
    if (G >= 4) {
#pragma unroll
      for (int t = 0; t < SMAC_RING - 1; t++) ring_issue(t);
    }
#pragma unroll 2
    for (int t = 0; t < nt; t++) {
      u64 x0, x1;
      if (G >= 4) {
        ring_issue(t + SMAC_RING - 1);  // overwrites the slot of term t - 1, already consumed by this thread
        asm volatile("cp.async.wait_group %0;" ::"n"(SMAC_RING - 1) : "memory");
        const u32 slot = a_ring + ((u32)t % SMAC_RING) * (u32)(2 * 256 * sizeof(u64));
        asm volatile("ld.shared.u64 %0, [%1];" : "=l"(x0) : "r"(slot) : "memory");
        asm volatile("ld.shared.u64 %0, [%1];" : "=l"(x1) : "r"(slot + (u32)(256 * sizeof(u64))) : "memory");
      } else {
        const u64 *c = s_ct[t];
        x0 = __ldg(c + idx), x1 = __ldg(c + LN + idx);
      }
      if (SPLIT) {
        constexpr u32 pm = (1u << PB) - 1u;
        double xp[2][NP];
#pragma unroll
        for (int c = 0; c < 2; c++) {
          const u64 x = c ? x1 : x0;  // below 2^50: the top piece fits 32 bits in both splits
          xp[c][0] = u2d((u32)x & pm);
          if (NP == 2) xp[c][1] = u2d((u32)(x >> PB));
          else xp[c][1] = u2d((u32)(x >> PB) & pm), xp[c][NP - 1] = u2d((u32)(x >> (2 * PB)));
        }
        double kds[G];
        if (G >= 4) {
#pragma unroll
          for (int i = 0; i < G; i += 2)
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(kds[i]), "=d"(kds[i + 1]) : "r"(a_kd + (u32)(t * G + i) * 8u) : "memory");
        } else {
#pragma unroll
          for (int i = 0; i < G; i++) kds[i] = s_kd[t][i];
        }
#pragma unroll
        for (int i = 0; i < G; i++) {
          const double kd = kds[i];
#pragma unroll
          for (int c = 0; c < 2; c++)
#pragma unroll
            for (int q2 = 0; q2 < NP; q2++) sp[i][c][q2] = __fma_rn(xp[c][q2], kd, sp[i][c][q2]);
        }
        if (++lazy == p.max_lazy) {  // every partial sum back to at most q/2 in magnitude (congruent mod q): exactness budget restored
#pragma unroll
          for (int i = 0; i < G; i++)
#pragma unroll
            for (int c = 0; c < 2; c++)
#pragma unroll
              for (int q2 = 0; q2 < NP; q2++) sp[i][c][q2] = reduce_dd(sp[i][c][q2], fm);
          lazy = 0;
        }
      } else if (F64) {
        const double xd0 = u2d52(x0), xd1 = u2d52(x1);
#pragma unroll
        for (int i = 0; i < G; i++) {
          const ulonglong2 kk = s_k[i][t];
          const double kd = __longlong_as_double((long long)kk.x), kq = __longlong_as_double((long long)kk.y);
          acc[i][0] = __dadd_rn(acc[i][0], mulmod_dd(xd0, kd, kq, fm));
          acc[i][1] = __dadd_rn(acc[i][1], mulmod_dd(xd1, kd, kq, fm));
        }
        if (++lazy == p.max_lazy) {
#pragma unroll
          for (int i = 0; i < G; i++) acc[i][0] = reduce_dd(acc[i][0], fm), acc[i][1] = reduce_dd(acc[i][1], fm);
          lazy = 1;  // the reduced remainder counts as one term
        }
      } else {
#pragma unroll
        for (int i = 0; i < G; i++) {
          const u64 km = s_k[i][t].x;
          mac128(lo[i][0], hi[i][0], x0, km), mac128(lo[i][1], hi[i][1], x1, km);
        }
        if (++lazy == p.max_lazy) {
          // fold: (S 2^-64 mod q) 2^128 2^-64 = S mod q, a residue below q, becomes the pending sum
#pragma unroll
          for (int i = 0; i < G; i++)
#pragma unroll
            for (int cpn = 0; cpn < 2; cpn++)
              lo[i][cpn] = mont_mul(mont_redc(lo[i][cpn], hi[i][cpn], mc.q, mc.qinv_neg), mc.r2, mc.q, mc.qinv_neg), hi[i][cpn] = 0;
          lazy = 1;
        }
      }
      if (t0 + t + 1 == cur_end) {  // end of a mask segment (uniform over the block): tot += M (*) S
        const u64 m = __ldg(p.seg_mask[g.seg_start + seg] + idx);
#pragma unroll
        for (int i = 0; i < G; i++)
#pragma unroll
          for (int cpn = 0; cpn < 2; cpn++) {
            u64 S;
            if (SPLIT) {
              // S_0 + S_1 2^B (+ S_2 2^2B) mod q: the powers of two as representatives in [-q/2, q/2], exact products
              const double c1 = reduce_dd((double)(1ull << PB), fm);
              double r = __dadd_rn(reduce_dd(sp[i][cpn][0], fm), mulmod_dd(reduce_dd(sp[i][cpn][1], fm), c1, __dmul_rn(c1, fm.qinv), fm));
              if (NP == 3) {
                const double c2 = reduce_dd((double)(1ull << (2 * PB)), fm);
                r = __dadd_rn(r, mulmod_dd(reduce_dd(sp[i][cpn][NP - 1], fm), c2, __dmul_rn(c2, fm.qinv), fm));
              }
              S = csub(d2u_off(reduce_dd(r, fm), fm.q + 4503599627370496.0), mc.q);
#pragma unroll
              for (int q2 = 0; q2 < NP; q2++) sp[i][cpn][q2] = 0.0;
            } else if (F64) {
              S = csub(d2u_off(reduce_dd(acc[i][cpn], fm), fm.q + 4503599627370496.0), mc.q);
              acc[i][cpn] = 0.0;
            } else {
              S = mont_redc(lo[i][cpn], hi[i][cpn], mc.q, mc.qinv_neg);
              lo[i][cpn] = hi[i][cpn] = 0;
            }
            const u64 prod = mont_mul(S, m, mc.q, mc.qinv_neg);
            if (TS) {
              // first segment: nothing to add; last segment: straight to the output (a one-segment group never touches s_tot)
              u64 *slot = s_tot + (size_t)(i * 2 + cpn) * blockDim.x + threadIdx.x;
              const u64 v = seg == 0 ? prod : addmod(*slot, prod, mc.q);
              if (seg + 1 < g.n_seg) *slot = v;
              else if (i < g.n_out) p.outs[g.out_start + i][(cpn ? LN : 0u) + idx] = v;
            } else {
              tot[i][cpn] = addmod(tot[i][cpn], prod, mc.q);
            }
          }
        lazy = 0;
        seg++;
        cur_end = seg < g.n_seg ? p.seg_end[g.seg_start + seg] : -1;
      }
    }
  }
  if (!TS || seg == 0) {  // TS: a group without any segment (no terms) is all zero
#pragma unroll
    for (int i = 0; i < G; i++)
      if (i < g.n_out) {
        u64 *out = p.outs[g.out_start + i];
        out[idx] = TS ? 0 : tot[i][0];
        out[LN + idx] = TS ? 0 : tot[i][1];
      }
  }
  }  // chunks of the block
}
// Single-output groups in fp64 mode (depthwise layers: every output has its own ciphertext sequence, nothing to share):
// a streaming kernel, two adjacent coefficients per thread with 16-byte loads, the loads of up to four terms of a mask
// segment in flight before their products.  HBM-bound: 16 (L N) bytes read per term and output.
__global__ void __launch_bounds__(256, 4) smac1_kernel(SmacP p) {
  __shared__ const u64 *s_ct[SMAC_TILE];
  __shared__ ulonglong2 s_k[SMAC_TILE];
  const size_t LN = (size_t)p.L << p.logN;
  const size_t idx = ((size_t)blockIdx.y * blockDim.x + threadIdx.x) * 2;
  const int limb = (int)(((size_t)blockIdx.y * blockDim.x * 2) >> p.logN);
  const SmacGroup g = p.groups[blockIdx.x];
  const ModConst mc = p.mods[limb];
  const F64Mod fm = f64mod(mc.q, mc.f64);
  double acc[4] = {0.0, 0.0, 0.0, 0.0};  // (c0, c1) x (even, odd coefficient)
  u64 tot[4] = {0, 0, 0, 0};
  int seg = 0, cur_end = p.seg_end[g.seg_start], lazy = 0;
  auto term = [&](const ulonglong2 &a, const ulonglong2 &b, int t) {
    const ulonglong2 kk = s_k[t];
    // (split-mode tables hold the SIGNED k, |k| < 2^35: x k is still exact as h + l and the quotient estimate from k / q holds)
    const double kd = __longlong_as_double((long long)kk.x), kq = __longlong_as_double((long long)kk.y);
    acc[0] = __dadd_rn(acc[0], mulmod_dd(u2d52(a.x), kd, kq, fm));
    acc[1] = __dadd_rn(acc[1], mulmod_dd(u2d52(a.y), kd, kq, fm));
    acc[2] = __dadd_rn(acc[2], mulmod_dd(u2d52(b.x), kd, kq, fm));
    acc[3] = __dadd_rn(acc[3], mulmod_dd(u2d52(b.y), kd, kq, fm));
    if (++lazy == p.max_lazy) {
#pragma unroll
      for (int i = 0; i < 4; i++) acc[i] = reduce_dd(acc[i], fm);
      lazy = 1;
    }
  };
  for (int t0 = 0; t0 < g.n_terms; t0 += SMAC_TILE) {
    const int nt = g.n_terms - t0 < SMAC_TILE ? g.n_terms - t0 : SMAC_TILE;
    __syncthreads();
    for (int t = threadIdx.x; t < nt; t += blockDim.x) {
      s_ct[t] = p.term_ct[g.ct_start + t0 + t];
      ulonglong2 kk = __ldg(reinterpret_cast<const ulonglong2 *>(p.kpair) + (size_t)p.kidx[g.k_start + t0 + t] * p.L + limb);
      if (p.signed_k) kk.y = (u64)__double_as_longlong(__dmul_rn(__longlong_as_double((long long)kk.x), fm.qinv));  // k / q for the signed k
      s_k[t] = kk;
    }
    __syncthreads();
    int t = 0;
    while (t < nt) {
      const int e = cur_end - t0 < nt ? cur_end - t0 : nt;  // end of this segment inside the tile
      for (; t + 4 <= e; t += 4) {
        ulonglong2 a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; u++) {
          const u64 *c = s_ct[t + u];
          a[u] = __ldg(reinterpret_cast<const ulonglong2 *>(c + idx));
          b[u] = __ldg(reinterpret_cast<const ulonglong2 *>(c + LN + idx));
        }
#pragma unroll
        for (int u = 0; u < 4; u++) term(a[u], b[u], t + u);
      }
      for (; t < e; t++) {
        const u64 *c = s_ct[t];
        term(__ldg(reinterpret_cast<const ulonglong2 *>(c + idx)), __ldg(reinterpret_cast<const ulonglong2 *>(c + LN + idx)), t);
      }
      if (t0 + t == cur_end) {  // tot += M (*) S
        const ulonglong2 m = __ldg(reinterpret_cast<const ulonglong2 *>(p.seg_mask[g.seg_start + seg] + idx));
        const double off = fm.q + 4503599627370496.0;
#pragma unroll
        for (int i = 0; i < 4; i++) {
          const u64 S = csub(d2u_off(reduce_dd(acc[i], fm), off), mc.q);
          tot[i] = addmod(tot[i], mont_mul(S, (i & 1) ? m.y : m.x, mc.q, mc.qinv_neg), mc.q);
          acc[i] = 0.0;
        }
        lazy = 0;
        seg++;
        cur_end = seg < g.n_seg ? p.seg_end[g.seg_start + seg] : 1 << 30;
      }
    }
  }
  u64 *out = p.outs[g.out_start];
  *reinterpret_cast<ulonglong2 *>(out + idx) = make_ulonglong2(tot[0], tot[1]);
  *reinterpret_cast<ulonglong2 *>(out + LN + idx) = make_ulonglong2(tot[2], tot[3]);
}
template <int G, int MODE>
static void launch_smac_g(const SmacP &p, dim3 grid, int nth, cudaStream_t st) {
  const size_t dyn = G >= 4 ? (size_t)G * 2 * nth * sizeof(u64) : 0;  // the totals over the mask segments (TS)
  static bool attr_set = false;  // static + dynamic shared memory pass 48 KB for G = 8
  if (dyn && !attr_set) {
    cudaFuncSetAttribute(smac_kernel<G, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)G * 2 * 256 * sizeof(u64)));
    attr_set = true;
  }
  smac_kernel<G, MODE><<<grid, nth, dyn, st>>>(p);
}
template <int MODE>
static void launch_smac(const SmacP &p, dim3 grid, int nth, cudaStream_t st, int max_group) {
  if (max_group <= 1) launch_smac_g<1, MODE>(p, grid, nth, st);
  else if (max_group <= 2) launch_smac_g<2, MODE>(p, grid, nth, st);
  else if (max_group <= 4 || MODE == 3) launch_smac_g<4, MODE>(p, grid, nth, st);  // MODE 3: the caller groups by 4 (3 sums per accumulator)
  else launch_smac_g<FENC_SMAC_GROUP, MODE>(p, grid, nth, st);
}
// k_mode: 0 integer, 1 fp64 residues, 2 / 3 signed multipliers with the ciphertext word split in 2 x 25 / 3 x 17 bits
int k_smac(const KCtx &k, const SmacGroup *groups, int n_groups, int max_group, const u64 *const *term_ct, const int *kidx,
           const ShoupC *kpair, const int *seg_end, const u64 *const *seg_mask, u64 *const *outs, int L, int k_mode,
           int max_lazy, double alg_bytes, double alg_mulaccs) {
  if (n_groups == 0) return 0;
  if (k_mode == 3 && max_group > 4) return -3;
  SmacP p{groups, term_ct, kidx, kpair, seg_end, seg_mask, outs, k.d_mods, L, k.geom.logN, max_lazy < 2 ? 2 : max_lazy, k_mode >= 2 ? 1 : 0, 1};
  const int nth = k.N < 256 ? k.N : 256;
  // chunks per block of the grouped kernel: SMAC_CPB when a limb has that many and the grid keeps eight waves of blocks
  const size_t chunks = ((size_t)L * k.N) / nth;
#ifndef SMAC_CPB
#define SMAC_CPB 8
#endif
  if ((k.N / nth) % SMAC_CPB == 0 && (size_t)n_groups * (chunks / SMAC_CPB) >= (size_t)8 * 148 * 2) p.cpb = SMAC_CPB;
  dim3 grid(n_groups, (unsigned)(chunks / p.cpb));
  PROF2(k, K_SMAC, alg_bytes, alg_mulaccs);  // second counter of this class: modular multiply-accumulates
  if (k_mode >= 1 && max_group <= 1 && k.N >= 512) smac1_kernel<<<dim3(n_groups, (unsigned)(((size_t)L * k.N) / 512)), 256, 0, S(k)>>>(p);
  else if (k_mode == 3) launch_smac<3>(p, grid, nth, S(k), max_group);
  else if (k_mode == 2) launch_smac<2>(p, grid, nth, S(k), max_group);
  else if (k_mode == 1) launch_smac<1>(p, grid, nth, S(k), max_group);
  else launch_smac<0>(p, grid, nth, S(k), max_group);
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ sum of ciphertexts
struct AddManyP { const u64 *const *term; const int *start; u64 *const *outs; const ModConst *mods; int L, logN; };
__global__ void __launch_bounds__(256) add_many_kernel(AddManyP p) {
  const size_t LN = (size_t)p.L << p.logN;
  const size_t idx = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 2;  // over [2][L][N]
  if (idx >= 2 * LN) return;
  const int o = blockIdx.y;
  const u64 q = p.mods[(idx % LN) >> p.logN].q;
  u64 a = 0, b = 0;
  for (int t = p.start[o]; t < p.start[o + 1]; t++) {
    const ulonglong2 x = __ldg(reinterpret_cast<const ulonglong2 *>(p.term[t] + idx));
    a = addmod(a, x.x, q); b = addmod(b, x.y, q);
  }
  *reinterpret_cast<ulonglong2 *>(p.outs[o] + idx) = make_ulonglong2(a, b);
}
int k_add_many(const KCtx &k, const u64 *const *term, const int *start, u64 *const *outs, int n_out, int L, int n_terms) {
  if (n_out == 0) return 0;
  AddManyP p{term, start, outs, k.d_mods, L, k.geom.logN};
  size_t pairs = (size_t)L * k.N;
  dim3 grid((unsigned)((pairs + 255) / 256), n_out);
  PROF(k, K_ADD_MANY, 16.0 * L * k.N * ((double)n_terms + n_out));
  add_many_kernel<<<grid, 256, 0, S(k)>>>(p);
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ generic row kernels
// grid (N/256, n_rows); row r uses modulus row_mod[r]
enum RowOp { OP_X_MINUS_AS, OP_TO_MONT, OP_FROM_MONT, OP_ADD_F_SP, OP_MUL, OP_ADD, OP_ADD_TWICE, OP_REDUCE_SIGNED };
struct RowP {
  const u64 *a; const u64 *b; const u64 *s; u64 *out; const int *row_mod; const ModConst *mods; const u64 *f;
  const i64 *coeffs; int logN; u32 g;
};
template <int OP>
__global__ void __launch_bounds__(256) row_kernel(RowP p) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y, N = 1 << p.logN;
  if (n >= N) return;
  const int mod = p.row_mod[r];
  const ModConst mc = p.mods[mod];
  const size_t i = (size_t)r * N + n;
  u64 v;
  if (OP == OP_X_MINUS_AS) v = submod(p.b[i], mont_mul(p.a[i], p.s[(size_t)mod * N + n], mc.q, mc.qinv_neg), mc.q);
  else if (OP == OP_TO_MONT) v = mont_mul(p.a[i], mc.r2, mc.q, mc.qinv_neg);
  else if (OP == OP_FROM_MONT) v = mont_redc(p.a[i], 0, mc.q, mc.qinv_neg);
  else if (OP == OP_ADD_F_SP) {
    const u64 sp = p.s[(size_t)mod * N + galois_src(n, p.g, p.logN)];  // sigma_g(s) in the NTT domain, Montgomery form
    v = addmod(p.a[i], mont_mul(p.f[mod], sp, mc.q, mc.qinv_neg), mc.q);
  } else if (OP == OP_MUL) v = mont_mul(p.a[i], mont_mul(p.b[i], mc.r2, mc.q, mc.qinv_neg), mc.q, mc.qinv_neg);
  else if (OP == OP_ADD) v = addmod(p.a[i], p.b[i], mc.q);
  else if (OP == OP_ADD_TWICE) v = addmod(addmod(p.a[i], p.b[i], mc.q), p.b[i], mc.q);
  else {  // OP_REDUCE_SIGNED: centred integer -> residue (negative -> q - |m| mod q)
    const i64 m = p.coeffs[n];
    const u64 mag = (u64)(m < 0 ? -m : m) % mc.q;
    v = (m < 0 && mag) ? mc.q - mag : mag;
  }
  p.out[i] = v;
}
template <int OP>
static int launch_row(const KCtx &k, RowP p, int n_rows) {
  if (n_rows == 0) return 0;
  p.mods = k.d_mods; p.logN = k.geom.logN;
  dim3 grid((k.N + 255) / 256, n_rows);
  PROF(k, K_ROWOP, 24.0 * k.N * n_rows);
  row_kernel<OP><<<grid, 256, 0, S(k)>>>(p);
  LAUNCH_CHECK(k);
  return 0;
}
int k_x_minus_as(const KCtx &k, const u64 *a, const u64 *x, const u64 *s_mont, u64 *out, const int *row_mod, int n_rows) {
  RowP p{}; p.a = a; p.b = x; p.s = s_mont; p.out = out; p.row_mod = row_mod;
  return launch_row<OP_X_MINUS_AS>(k, p, n_rows);
}
int k_mont_convert(const KCtx &k, const u64 *src, u64 *dst, const int *row_mod, int n_rows, bool to_mont) {
  RowP p{}; p.a = src; p.out = dst; p.row_mod = row_mod;
  return to_mont ? launch_row<OP_TO_MONT>(k, p, n_rows) : launch_row<OP_FROM_MONT>(k, p, n_rows);
}
int k_add_f_sprime(const KCtx &k, const u64 *x, const u64 *sp_mont, u32 g, const u64 *f, u64 *out, const int *row_mod,
                   int n_rows) {
  RowP p{}; p.a = x; p.s = sp_mont; p.g = g; p.f = f; p.out = out; p.row_mod = row_mod;
  return launch_row<OP_ADD_F_SP>(k, p, n_rows);
}
int k_mul_rows(const KCtx &k, const u64 *a, const u64 *b, u64 *out, const int *row_mod, int n_rows) {
  RowP p{}; p.a = a; p.b = b; p.out = out; p.row_mod = row_mod;
  return launch_row<OP_MUL>(k, p, n_rows);
}
int k_add_rows(const KCtx &k, const u64 *a, const u64 *b, u64 *out, const int *row_mod, int n_rows, bool twice) {
  RowP p{}; p.a = a; p.b = b; p.out = out; p.row_mod = row_mod;
  return twice ? launch_row<OP_ADD_TWICE>(k, p, n_rows) : launch_row<OP_ADD>(k, p, n_rows);
}
int k_reduce_signed(const KCtx &k, const i64 *coeffs, const int *row_mod, u64 *dst, int n_rows) {
  RowP p{}; p.coeffs = coeffs; p.out = dst; p.row_mod = row_mod;
  return launch_row<OP_REDUCE_SIGNED>(k, p, n_rows);
}

// tensor product per limb (a13, R2.12): (d0, d1, d2) = (a0 b0, a0 b1 + a1 b0, a1 b1); d: [n][3][L][N]
__global__ void __launch_bounds__(256) tensor_product_kernel(const u64 *const *ina, const u64 *const *inb, u64 *d, const ModConst *mods,
                                                             int L, int logN) {
  const size_t LN = (size_t)L << logN;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= LN) return;
  const ModConst mc = mods[i >> logN];
  const u64 *a = ina[blockIdx.y], *b = inb[blockIdx.y];
  const u64 a0 = a[i], a1 = a[LN + i], b0 = b[i], b1 = b[LN + i];
  const u64 b0m = mont_mul(b0, mc.r2, mc.q, mc.qinv_neg), b1m = mont_mul(b1, mc.r2, mc.q, mc.qinv_neg);
  u64 *o = d + (size_t)blockIdx.y * 3 * LN;
  o[i] = mont_mul(a0, b0m, mc.q, mc.qinv_neg);
  o[LN + i] = addmod(mont_mul(a0, b1m, mc.q, mc.qinv_neg), mont_mul(a1, b0m, mc.q, mc.qinv_neg), mc.q);
  o[2 * LN + i] = mont_mul(a1, b1m, mc.q, mc.qinv_neg);
}
// sums of squares (R2.12c): d[o] = sum over the group's ciphertexts in[o*group + i] of (c0 c0, 2 c0 c1, c1 c1); d: [n][3][L][N]
__global__ void __launch_bounds__(256) square_sum_kernel(const u64 *const *in, int group, u64 *d, const ModConst *mods, int L, int logN) {
  const size_t LN = (size_t)L << logN;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= LN) return;
  const ModConst mc = mods[i >> logN];
  u64 s0 = 0, s1 = 0, s2 = 0;
  for (int gidx = 0; gidx < group; gidx++) {
    const u64 *a = in[(size_t)blockIdx.y * group + gidx];
    const u64 a0 = a[i], a1 = a[LN + i];
    const u64 a0m = mont_mul(a0, mc.r2, mc.q, mc.qinv_neg), a1m = mont_mul(a1, mc.r2, mc.q, mc.qinv_neg);
    const u64 x = mont_mul(a0, a1m, mc.q, mc.qinv_neg);
    s0 = addmod(s0, mont_mul(a0, a0m, mc.q, mc.qinv_neg), mc.q);
    s1 = addmod(s1, addmod(x, x, mc.q), mc.q);
    s2 = addmod(s2, mont_mul(a1, a1m, mc.q, mc.qinv_neg), mc.q);
  }
  u64 *o = d + (size_t)blockIdx.y * 3 * LN;
  o[i] = s0, o[LN + i] = s1, o[2 * LN + i] = s2;
}
int k_square_sum(const KCtx &k, const u64 *const *in, int group, u64 *d, int n, int L) {
  if (n == 0) return 0;
  dim3 grid((unsigned)(((size_t)L * k.N + 255) / 256), n);
  PROF(k, K_ROWOP, (16.0 * group + 24.0) * L * k.N * n);
  square_sum_kernel<<<grid, 256, 0, S(k)>>>(in, group, d, k.d_mods, L, k.geom.logN);
  LAUNCH_CHECK(k);
  return 0;
}
int k_tensor_product(const KCtx &k, const u64 *const *ina, const u64 *const *inb, u64 *d, int n, int L) {
  if (n == 0) return 0;
  dim3 grid((unsigned)(((size_t)L * k.N + 255) / 256), n);
  PROF(k, K_ROWOP, 56.0 * L * k.N * n);
  tensor_product_kernel<<<grid, 256, 0, S(k)>>>(ina, inb, d, k.d_mods, L, k.geom.logN);
  LAUNCH_CHECK(k);
  return 0;
}
// out[b] = in[b] * k (both polynomials), k given per limb in Montgomery form; add_const: c0 += k (the constant polynomial
// k is k at every evaluation point), k given per limb as a canonical residue
__global__ void __launch_bounds__(256) scalar_kernel(const u64 *const *in, u64 *const *out, const u64 *kl, const ModConst *mods, int L,
                                                     int logN, int add_const) {
  const size_t LN = (size_t)L << logN;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= LN) return;
  const int t = (int)(i >> logN);
  const ModConst mc = mods[t];
  const u64 *a = in[blockIdx.y];
  u64 *o = out[blockIdx.y];
  if (add_const) {
    o[i] = addmod(a[i], kl[t], mc.q);
    o[LN + i] = a[LN + i];
  } else {
    o[i] = mont_mul(a[i], kl[t], mc.q, mc.qinv_neg);
    o[LN + i] = mont_mul(a[LN + i], kl[t], mc.q, mc.qinv_neg);
  }
}
int k_scalar(const KCtx &k, const u64 *const *in, u64 *const *out, const u64 *kl, int n, int L, bool add_const) {
  if (n == 0) return 0;
  dim3 grid((unsigned)(((size_t)L * k.N + 255) / 256), n);
  PROF(k, K_ROWOP, 32.0 * L * k.N * n);
  scalar_kernel<<<grid, 256, 0, S(k)>>>(in, out, kl, k.d_mods, L, k.geom.logN, add_const ? 1 : 0);
  LAUNCH_CHECK(k);
  return 0;
}

// out[t] = c0[t] + c1[t] * s[t]  (decrypt, R2.5)
__global__ void __launch_bounds__(256) dec_combine_kernel(const u64 *ct, const u64 *s_mont, u64 *out, const ModConst *mods, int L, int logN) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x, t = blockIdx.y, N = 1 << logN;
  if (n >= N) return;
  const ModConst mc = mods[t];
  const size_t i = (size_t)t * N + n;
  out[i] = addmod(ct[i], mont_mul(ct[(size_t)L * N + i], s_mont[i], mc.q, mc.qinv_neg), mc.q);
}
int k_dec_combine(const KCtx &k, const u64 *ct, const u64 *s_mont, u64 *out, int L) {
  dim3 grid((k.N + 255) / 256, L);
  PROF(k, K_ROWOP, 32.0 * k.N * L);
  dec_combine_kernel<<<grid, 256, 0, S(k)>>>(ct, s_mont, out, k.d_mods, L, k.geom.logN);
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ samplers (R2.3)
// draw(key, n) = mix64(key + (n+1) GAMMA); coefficient i owns counters i*64 .. i*64+63.
#define FENC_GAMMA 0x9E3779B97F4A7C15ull
DEVI u64 d_mix64(u64 z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
DEVI u64 d_draw(u64 key, u64 n) { return d_mix64(key + (n + 1) * FENC_GAMMA); }

// C[x] = floor(2^64 Pr(|X| <= x)), X discrete Gaussian sigma = 3.2 cut at |x| <= 19 (R2.3 table)
__constant__ u64 c_gauss_cdt[19] = {
    0x1fea56814b22fe3aull, 0x5cb44ba97e1c801cull, 0x9135c4d2ab6097acull, 0xba57841ec437e30aull, 0xd790d29879901fe9ull,
    0xea65b1358d74fb9dull, 0xf5672d96e886cf31ull, 0xfb3c9d22cc87d60full, 0xfe0a92b033d640a2ull, 0xff439d38007352aeull,
    0xffbf67e425d189d1ull, 0xffebcdf3a4629f98ull, 0xfffa3f2f78880d45ull, 0xfffe81f40111a23bull, 0xffffa5d06bc38afbull,
    0xffffeca4870dfe3cull, 0xfffffc3b68ed3b4aull, 0xffffff58143b9611ull, 0xffffffe850ce70a6ull};

__global__ void __launch_bounds__(256) sample_uniform_kernel(const u64 *keys, const int *row_mod, u64 *dst, const ModConst *mods, int logN) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y, N = 1 << logN;
  if (n >= N) return;
  const ModConst mc = mods[row_mod[r]];
  const u64 key = keys[r];
  u64 x = 0;
  bool ok = false;
  for (int a = 0; a < 64 && !ok; a++) {
    x = d_draw(key, (u64)n * 64 + a) & mc.mask;
    ok = x < mc.q;
  }
  if (!ok) x %= mc.q;
  dst[(size_t)r * N + n] = x;
}
int k_sample_uniform(const KCtx &k, const u64 *keys, const int *row_mod, u64 *dst, int n_rows) {
  if (n_rows == 0) return 0;
  dim3 grid((k.N + 255) / 256, n_rows);
  PROF(k, K_SAMPLE, 8.0 * k.N * n_rows);
  sample_uniform_kernel<<<grid, 256, 0, S(k)>>>(keys, row_mod, dst, k.d_mods, k.geom.logN);
  LAUNCH_CHECK(k);
  return 0;
}

__global__ void __launch_bounds__(256) sample_gauss_kernel(u64 key, const i64 *addend, const int *row_mod, u64 *dst, const ModConst *mods,
                                                           int logN, int n_rows) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x, N = 1 << logN;
  if (n >= N) return;
  const u64 u = d_draw(key, (u64)n * 64);
  int mag = 0;
  for (int x = 0; x < 19; x++) mag += (c_gauss_cdt[x] <= u) ? 1 : 0;  // least x with u < C[x]
  i64 v = (d_draw(key, (u64)n * 64 + 1) & 1) ? -(i64)mag : (i64)mag;
  if (addend) v += addend[n];
  for (int r = 0; r < n_rows; r++) {
    const u64 q = mods[row_mod[r]].q;
    const u64 m = (u64)(v < 0 ? -v : v) % q;
    dst[(size_t)r * N + n] = (v < 0 && m) ? q - m : m;
  }
}
int k_sample_gauss(const KCtx &k, u64 key, const i64 *addend, const int *row_mod, u64 *dst, int n_rows) {
  if (n_rows == 0) return 0;
  PROF(k, K_SAMPLE, 8.0 * k.N * n_rows);
  sample_gauss_kernel<<<(k.N + 255) / 256, 256, 0, S(k)>>>(key, addend, row_mod, dst, k.d_mods, k.geom.logN, n_rows);
  LAUNCH_CHECK(k);
  return 0;
}
