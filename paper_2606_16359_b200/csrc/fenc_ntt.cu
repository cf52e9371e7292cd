// fenc_ntt.cu -- batched negacyclic NTT / iNTT kernels (a1) and the key-switch kernels fused around them
// (a2 automorphism gather, a3 ModUp, a4 evk inner product, a5 ModDown, a8 rescale).  sm_100a.
//
// Transform (R2.1 and section 6): merged-twiddle Cooley-Tukey forward (natural in, bit-reversed out) and
// Gentleman-Sande inverse, split in two passes so that each pass works on a shared-memory tile:
//   forward = column pass (the bcol high stages, stride 2^brow) then row pass (the brow low stages, contiguous);
//   inverse = row pass then column pass.
// Each pass: coalesced tile load -> radix-8 register rounds through swizzled shared memory -> coalesced store.
// The first touch of a forward transform and the last touch of either direction carry the fused work; for ring degrees
// >= 2^12 the inverse column pass, the base conversion and the forward column pass of a key switch are ONE kernel
// (convert_cols_kernel) that keeps the converted limbs in shared memory.
// What the kernels stage in shared memory beside the tile (round 2, profiles/r02_late_captures.md): the row passes keep one
// tile position per block over several batch items with that position's twiddles ("slab") and the items' descriptors; the
// fused column kernel its targets' descriptors, each target's forward twiddles and base-conversion constants (cp.async);
// the key inner product its digit's key words.  Where the load / store order allows, the first and the last round of a
// transform work on registers (REGIN / REGOUT in fenc_device.cuh) instead of a fill / drain through shared memory.
#include "fenc_device.cuh"

// geometry dispatch: row kernels GEO in {0,1}; column kernels GEO in {0,4..8} (fenc_device.cuh tile_transform)
#define ROW_GEO(g, CALL)            \
  do {                              \
    if ((g).logN >= 12) { constexpr int GEO = 1; CALL; } \
    else { constexpr int GEO = 0; CALL; }                \
  } while (0)
#define COL_GEO(g, CALL)                                   \
  do {                                                     \
    switch ((g).logN >= 12 ? (g).bcol : 0) {               \
      case 4: { constexpr int GEO = 4; CALL; } break;      \
      case 5: { constexpr int GEO = 5; CALL; } break;      \
      case 6: { constexpr int GEO = 6; CALL; } break;      \
      case 7: { constexpr int GEO = 7; CALL; } break;      \
      case 8: { constexpr int GEO = 8; CALL; } break;      \
      default: { constexpr int GEO = 0; CALL; } break;     \
    }                                                      \
  } while (0)
// Tile fill / drain with all of a thread's (<= 8) global accesses independent and in flight together: the loads are issued
// first, the shared-memory stores after (a rolled loop would serialise one L2/HBM latency per element).
template <class F>
DEVI void tile_fill(u64 *sm, int T, int tid, int nth, F f) {
  u64 v[8];
#pragma unroll
  for (int i = 0; i < 8; i++) {
    const int e = tid + i * nth;
    if (e < T) v[i] = f(e);
  }
#pragma unroll
  for (int i = 0; i < 8; i++) {
    const int e = tid + i * nth;
    if (e < T) sm[swz(e)] = v[i];
  }
}
template <class F>
DEVI void tile_drain(const u64 *sm, int T, int tid, int nth, F f) {
#pragma unroll
  for (int i = 0; i < 8; i++) {
    const int e = tid + i * nth;
    if (e < T) f(e, sm[swz(e)]);
  }
}
static inline int nthreads_for(int lt) { int t = 1 << (lt - 3); return t < 32 ? 32 : t; }
#define PROF(k, id, bytes, bfly) if ((k).prof) prof_begin((k).prof, (k).stream, id, (double)(bytes), (double)(bfly))
#define HALF_N(k) (0.5 * (k).N)
#define LAUNCH_CHECK(k)                            \
  do {                                             \
    (*(k).launches)++;                             \
    if ((k).prof) prof_end((k).prof, (k).stream);  \
    cudaError_t e__ = cudaGetLastError();          \
    if (e__ != cudaSuccess) return (int)e__;       \
  } while (0)

// ------------------------------------------------------------------------------------------------ inverse, pass A
struct InttRowP {
  const BatchItem *items; const u64 *src; size_t src_bstride; u64 *dst; size_t dst_bstride;
  const RowDesc *rows; const ModConst *mods; const ShoupC *tw; NttGeom g;
  const ShoupC *comb_mul;  // COMB: rows with aux = 1 read src * comb_mul[mod] + items[b].add{aux2}[mod] (merged rescale)
};
template <bool GATHER, int GEO, bool COMB = false>
__global__ void __launch_bounds__(256, 5) intt_rowpass_kernel(InttRowP p) {
  extern __shared__ u64 sm[];
  const int tid = threadIdx.x, b = blockIdx.z;
  const RowDesc rd = p.rows[blockIdx.y];
  const int N = 1 << p.g.logN, T = 1 << p.g.lt_row;
  TileGeo G{p.g.lt_row, p.g.lt_row, 0, p.g.logN, blockIdx.x};
  const u64 *src = ((p.items && !COMB) ? p.items[b].ks_in : p.src + (size_t)b * p.src_bstride) + (size_t)rd.src_row * N;
  const u32 gal = GATHER ? p.items[b].g : 1u;
  const int logN = p.g.logN, nth = blockDim.x;
  const u64 q = p.mods[rd.mod].q;
  if (COMB && rd.aux) {
    const u64 *add = (rd.aux2 == 0 ? p.items[b].add0 : p.items[b].add1) + (size_t)rd.mod * N;
    const ShoupC mc = p.comb_mul[rd.mod];
    tile_fill(sm, T, tid, nth, [&](int e) {
      const u32 j = G.gidx(e);
      return addmod(shoup_mul(__ldg(src + j), mc.c, mc.cs, q), __ldg(add + j), q);
    });
  } else {
    tile_fill(sm, T, tid, nth, [&](int e) {
      const u32 j = G.gidx(e);
      return __ldg(src + (GATHER ? galois_src(j, gal, logN) : j));
    });
  }
  __syncthreads();
  tile_transform<false, GEO>(sm, G, 0, p.g.brow, p.tw + (size_t)rd.mod * N, q, tid, p.mods[rd.mod].f64);
  u64 *dst = p.dst + (size_t)b * p.dst_bstride + (size_t)rd.dst_row * N;
  tile_drain(sm, T, tid, nth, [&](int e, u64 v) { dst[G.gidx(e)] = v; });
}

// ------------------------------------------------------------------------------------------------ inverse, pass B
struct InttColP {
  u64 *dst; size_t dst_bstride; const RowDesc *rows; const ShoupC *scale; const ModConst *mods; const ShoupC *tw; NttGeom g;
};
template <int GEO>
__global__ void __launch_bounds__(512, 3) intt_colpass_kernel(InttColP p) {
  extern __shared__ u64 sm[];
  const int tid = threadIdx.x, b = blockIdx.z;
  const RowDesc rd = p.rows[blockIdx.y];
  const int N = 1 << p.g.logN, T = 1 << p.g.lt_col;
  TileGeo G{p.g.lt_col, p.g.lc_col, p.g.brow, p.g.logN, blockIdx.x};
  u64 *dst = p.dst + (size_t)b * p.dst_bstride + (size_t)rd.dst_row * N;
  const int nth = blockDim.x;
  tile_fill(sm, T, tid, nth, [&](int e) { return dst[G.gidx(e)]; });
  __syncthreads();
  const u64 q = p.mods[rd.mod].q;
  tile_transform<false, GEO>(sm, G, p.g.lc_col, p.g.bcol, p.tw + (size_t)rd.mod * N, q, tid, p.mods[rd.mod].f64);
  const ShoupC sc = p.scale[blockIdx.y];
  tile_drain(sm, T, tid, nth, [&](int e, u64 v) { dst[G.gidx(e)] = shoup_mul(v, sc.c, sc.cs, q); });
}

int k_intt(const KCtx &k, const BatchItem *items, const u64 *src, size_t src_bstride, bool gather, u64 *dst,
           size_t dst_bstride, const RowDesc *rows, int n_rows, const ShoupC *scale, int n_batch) {
  if (n_rows == 0 || n_batch == 0) return 0;
  cudaStream_t st = (cudaStream_t)k.stream;
  const NttGeom &g = k.geom;
  InttRowP a{items, src, src_bstride, dst, dst_bstride, rows, k.d_mods, k.d_tw_inv, g, nullptr};
  dim3 gridA(k.N >> g.lt_row, n_rows, n_batch);
  PROF(k, K_INTT_ROW, 16.0 * k.N * n_rows * n_batch, HALF_N(k) * g.brow * n_rows * n_batch);
  if (gather) ROW_GEO(g, (intt_rowpass_kernel<true, GEO><<<gridA, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, st>>>(a)));
  else ROW_GEO(g, (intt_rowpass_kernel<false, GEO><<<gridA, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, st>>>(a)));
  LAUNCH_CHECK(k);
  InttColP c{dst, dst_bstride, rows, scale, k.d_mods, k.d_tw_inv, g};
  dim3 gridB(k.N >> g.lt_col, n_rows, n_batch);
  PROF(k, K_INTT_COL, 16.0 * k.N * n_rows * n_batch, HALF_N(k) * g.bcol * n_rows * n_batch);
  COL_GEO(g, (intt_colpass_kernel<GEO><<<gridB, nthreads_for(g.lt_col), sizeof(u64) << g.lt_col, st>>>(c)));
  LAUNCH_CHECK(k);
  return 0;
}

int k_intt_rows_only(const KCtx &k, const BatchItem *items, const u64 *src, size_t src_bstride, bool gather, u64 *dst,
                     size_t dst_bstride, const RowDesc *rows, int n_rows, int n_batch, const ShoupC *comb_mul) {
  if (n_rows == 0 || n_batch == 0) return 0;
  cudaStream_t st = (cudaStream_t)k.stream;
  const NttGeom &g = k.geom;
  InttRowP a{items, src, src_bstride, dst, dst_bstride, rows, k.d_mods, k.d_tw_inv, g, comb_mul};
  dim3 gridA(k.N >> g.lt_row, n_rows, n_batch);
  PROF(k, K_INTT_ROW, 16.0 * k.N * n_rows * n_batch, HALF_N(k) * g.brow * n_rows * n_batch);
  if (comb_mul) ROW_GEO(g, (intt_rowpass_kernel<false, GEO, true><<<gridA, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, st>>>(a)));
  else if (gather) ROW_GEO(g, (intt_rowpass_kernel<true, GEO><<<gridA, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, st>>>(a)));
  else ROW_GEO(g, (intt_rowpass_kernel<false, GEO><<<gridA, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, st>>>(a)));
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ fused column kernel (a3 / a5 / a8)
// One block = one column tile (2^BCOL rows x 2^LC columns = 1024 coefficients) of one conversion group of one batch item.
// The group's source rows arrive from the inverse row pass; their inverse column stages and the scaling
// N^-1 (Qhat^-1) run here and the resulting coefficient-domain tiles STAY in shared memory while every target row of
// the group is produced from them: base conversion (R2.6) + forward column stages -> tmp.  Compared with
// separate kernels this removes the inverse column pass's round trip and the (targets x sources) re-reads of y.
struct ConvColP {
  u64 *y; size_t y_bstride; const ConvGroup *groups; const ShoupC *scale; const u64 *bc; const RowDesc *rows;
  u64 *tmp; size_t tmp_bstride; const ModConst *mods; const ShoupC *tw_fwd; const ShoupC *tw_inv; int logN, brow, max_terms;
  const ShoupC *mulc;  // MERGED: P^-1 mod q_t
  const ShoupC *bc_f64;  // {(double) c, (double)(c / t)} per entry of bc, used when source and target moduli are fp64 ones
  int smem_tiles;        // tiles ahead of the twiddle buffers and the target descriptors in shared memory
};
// What a target row's iteration needs, staged in shared memory when the block starts: from global memory the chain
// rows[] -> mods[] -> (constants, twiddles) put two dependent L2 latencies in front of every target (ncu on the config-4
// step: 9 % of the kernel's stall samples on the two instructions that first use them).
struct TgtDesc { int mod, dst_row, aux2, pad; u64 q, qinv_neg, qbar, f64; };
#define CONV_DESC_CAP 56            // targets per group staged; later ones are read from global memory
#define CONV_BC_CAP 32              // base-conversion constants of one target staged (groups of more sources read them from global memory)
#define CONV_TW_WORDS (512 + 4 * CONV_BC_CAP)  // u64 words of one group's buffer: tw[0 .. 256) of the target's modulus, then two buffers of constants
DEVI TgtDesc tgt_desc_load(const ConvColP &p, int row) {
  const RowDesc rd = p.rows[row];
  const ModConst mc = p.mods[rd.mod];
  return TgtDesc{rd.mod, rd.dst_row, rd.aux2, 0, mc.q, mc.qinv_neg, mc.qbar, mc.f64};
}
// sum over the first n source tiles of Y_s[e] * bc[s] for this thread's eight elements, Montgomery-reduced: canonical.
// YDBL: the tiles hold the values as doubles (see conv_dot_f64); they are exact integers below 2^50.
// CS: the constants were staged in shared memory (stride 2 words: they share the slots of the fp64 pairs)
template <int T, int NTH, bool CS = false>
DEVI void conv_dot(const u64 *smem, int n, const u64 *bc, const ModConst &mc, int max_terms, int tid, u64 (&out)[8], bool ydbl) {
  u64 lo[8], hi[8], r[8];
#pragma unroll
  for (int i = 0; i < 8; i++) lo[i] = hi[i] = r[i] = 0;
  int lazy = 0;
  for (int s = 0; s < n; s++) {
    const u64 c = CS ? bc[2 * s] : __ldg(bc + s);
    const u64 *Y = smem + (size_t)s * T;
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const u64 w = Y[swz(tid + i * NTH)];
      mac128(lo[i], hi[i], ydbl ? d2u_off(__longlong_as_double((long long)w), 4503599627370496.0) : w, c);
    }
    if (++lazy == max_terms) {
#pragma unroll
      for (int i = 0; i < 8; i++) r[i] = addmod(r[i], mont_redc(lo[i], hi[i], mc.q, mc.qinv_neg), mc.q), lo[i] = hi[i] = 0;
      lazy = 0;
    }
  }
#pragma unroll
  for (int i = 0; i < 8; i++) out[i] = addmod(r[i], mont_redc(lo[i], hi[i], mc.q, mc.qinv_neg), mc.q);
}
// The same sum on the FP64 pipe (groups flagged pad[0] & 2: every source modulus an fp64 one, i.e. below 2^50; and an fp64
// target): the source tiles hold the canonical values as DOUBLES, each term y c - rint(y c / t) t is an exact integer in
// (-t, t) (mulmod_dd: |y| < 2^51, c < t < 2^50), a sum of `lazy_max` = floor(2^53 / t) - 1 terms plus a reduced remainder
// (at most t/2 + 1) is exact, and v - rint(v / t) t + t in (0, 2t) is what the forward fp64 butterflies ask of their input.
// Measured (profiles/r02_convert_cols.md): the 128-bit integer form of this sum was 38 % IMAD + 18 % IADD3 of the kernel's
// instructions with the fp64 pipe 16 % busy.
template <int T, int NTH, bool CS = false>
DEVI void conv_dot_f64(const u64 *smem, int n, const ShoupC *bc, const F64Mod &fm, int lazy_max, int tid, u64 (&out)[8]) {
  double acc[8];
#pragma unroll
  for (int i = 0; i < 8; i++) acc[i] = 0.0;
  int lazy = 0;
  for (int s = 0; s < n; s++) {
    const ulonglong2 cc = CS ? *reinterpret_cast<const ulonglong2 *>(bc + s) : __ldg(reinterpret_cast<const ulonglong2 *>(bc + s));
    const double c = __longlong_as_double((long long)cc.x), cq = __longlong_as_double((long long)cc.y);
    const u64 *Y = smem + (size_t)s * T;
#pragma unroll
    for (int i = 0; i < 8; i++) acc[i] = __dadd_rn(acc[i], mulmod_dd(__longlong_as_double((long long)Y[swz(tid + i * NTH)]), c, cq, fm));
    if (++lazy == lazy_max) {
#pragma unroll
      for (int i = 0; i < 8; i++) acc[i] = reduce_dd(acc[i], fm);
      lazy = 1;
    }
  }
  const double off = __dadd_rn(fm.q, 4503599627370496.0);
#pragma unroll
  for (int i = 0; i < 8; i++) out[i] = d2u_off(reduce_dd(acc[i], fm), off);
}
// MERGED (ModDown followed by the rescale): the group's last source tile is Z = iNTT(acc[l] P^-1 + add[l]) of
// the limb l = q_{L-1} that the rescale drops (modulus index cg.pad[1]).  With V_t = sum_i y_i (Phat_i mod t):
//   out_l = Z - V_l P^-1 mod q_l        (the key-switched limb l in the coefficient domain, canonical)
//   u_t   = V_t P^-1 + (out_l mod t)    (what the divide epilogue subtracts:  c'_t = (acc_t P^-1 + add_t - NTT(u_t)) q_l^-1)
// NG > 1 (digit groups of 6 and more limbs, whose source tiles leave room for one or two blocks per SM only): the block
// holds NG groups of 128 threads that share the source tiles; group g inverse-transforms the sources s = g mod NG and
// produces the targets t = g mod NG in a work tile of its own, its rounds meeting on named barrier g + 1.
template <int BCOL, bool MERGED, int NG>
__global__ void __launch_bounds__(128 * NG, NG == 1 ? 5 : (NG == 2 ? 2 : 1)) convert_cols_kernel(ConvColP p) {
  static_assert(!(MERGED && NG > 1), "the merged ModDown+rescale runs one group per block");
  constexpr int LT = 10, LC = LT - BCOL, T = 1 << LT, NTH = T / 8;
  constexpr bool GRP = NG > 1;
  extern __shared__ u64 smem[];
  const int tid = threadIdx.x & (NTH - 1), grp = threadIdx.x / NTH, bar = grp + 1, b = blockIdx.z;
  const ConvGroup cg = p.groups[blockIdx.y];
  const int N = 1 << p.logN;
  TileGeo G{LT, LC, p.brow, p.logN, blockIdx.x};
  u64 *W = smem + (size_t)(cg.n_src + grp) * T;  // work tiles after the source tiles
  ShoupC *twb = reinterpret_cast<ShoupC *>(smem + (size_t)p.smem_tiles * T + (size_t)grp * CONV_TW_WORDS);  // this group's forward twiddles
  TgtDesc *sdesc = reinterpret_cast<TgtDesc *>(smem + (size_t)p.smem_tiles * T + (size_t)NG * CONV_TW_WORDS);
  for (int t = threadIdx.x; t < cg.n_tgt && t < CONV_DESC_CAP; t += NTH * NG) sdesc[t] = tgt_desc_load(p, cg.tgt_start + t);
  u64 *ybase = p.y + (size_t)b * p.y_bstride;
  const int n_conv = MERGED ? cg.n_src - 1 : cg.n_src;  // tiles entering the base conversion
  const bool ydbl = !MERGED && p.bc_f64 && (cg.pad[0] & 2);  // the converted tiles are kept as doubles (conv_dot_f64)
  const bool cstage = n_conv <= CONV_BC_CAP;
  // target t's constants -> a buffer of this group (cp.async; the caller commits): fp64 pairs, or the integers at stride 2
  auto stage_consts = [&](ShoupC *dst, int t, bool staged_desc) {
    if (!cstage || tid >= n_conv) return;
    const TgtDesc d = staged_desc && t < CONV_DESC_CAP ? sdesc[t] : tgt_desc_load(p, cg.tgt_start + t);
    if (ydbl && d.f64) cp_async16(dst + tid, p.bc_f64 + d.aux2 + tid);
    else cp_async8(reinterpret_cast<u64 *>(dst + tid), p.bc + d.aux2 + tid);
  };
  if (grp < cg.n_tgt) stage_consts(twb + 256, grp, false);  // the descriptors in shared memory are not published yet
  cp_async_commit();
  // ---- sources: fill, inverse column stages, scale -> canonical coefficient tiles in shared memory
  for (int s = grp; s < cg.n_src; s += NG) {
    const u64 *src = ybase + (size_t)(cg.src_row + s) * N;
    tile_fill(smem + (size_t)s * T, T, tid, NTH, [&](int e) { return src[G.gidx(e)]; });
  }
  tile_sync<GRP>(bar);
  for (int s = grp; s < cg.n_src; s += NG) {
    u64 *Y = smem + (size_t)s * T;
    const int mod = (MERGED && s == n_conv) ? cg.pad[1] : cg.src_mod + s;
    const u64 q = p.mods[mod].q;
    tile_transform_ct<false, LT, LC, BCOL, GRP>(Y, G, p.tw_inv + (size_t)mod * N, q, tid, p.mods[mod].f64, bar);
    const ShoupC sc = p.scale[cg.scale_off + s];
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const int e = swz(tid + i * NTH);
      const u64 y = shoup_mul(Y[e], sc.c, sc.cs, q);
      Y[e] = ydbl ? (u64)__double_as_longlong(u2d52(y)) : y;
    }
  }
  cp_async_wait_all();
  __syncthreads();
  u64 outl[8];
  if (MERGED) {
    const int l = cg.pad[1];
    const ModConst ml = p.mods[l];
    const ShoupC pl = p.mulc[l];
    u64 v[8];
    conv_dot<T, NTH>(smem, n_conv, p.bc + (size_t)l * n_conv, ml, p.max_terms, tid, v, false);
    const u64 *Z = smem + (size_t)n_conv * T;
#pragma unroll
    for (int i = 0; i < 8; i++) outl[i] = submod(Z[swz(tid + i * NTH)], shoup_mul(v[i], pl.c, pl.cs, ml.q), ml.q);
  }
  // ---- targets
  int it = 0;
  for (int t = grp; t < cg.n_tgt; t += NG, it++) {
    const TgtDesc rd = t < CONV_DESC_CAP ? sdesc[t] : tgt_desc_load(p, cg.tgt_start + t);
    const ModConst mc{rd.q, rd.qinv_neg, 0, 0, rd.qbar, rd.f64, {0, 0}};
    // the 255 twiddles of this target's forward column stages and the NEXT target's base-conversion constants arrive in
    // shared memory while the base conversion runs (read per source term from global memory, the first use of a constant
    // was 9 % of the ModUp launches' stall samples: an L2 latency per term with nothing to overlap it)
    const bool f64dot = ydbl && mc.f64;
    ShoupC *cb = twb + 256 + (it & 1) * CONV_BC_CAP;
    {
      const ShoupC *twg = p.tw_fwd + (size_t)rd.mod * N;
      for (int i = tid; i < 256; i += NTH) cp_async16(twb + i, twg + i);
      if (t + NG < cg.n_tgt) stage_consts(twb + 256 + ((it + 1) & 1) * CONV_BC_CAP, t + NG, true);
      cp_async_commit();
    }
    u64 v[8];
    if (f64dot) {
      const int lazy_max = mc.q < (1ull << FENC_F64_MAX_BITS) ? 255 : 7;
      if (cstage) conv_dot_f64<T, NTH, true>(smem, n_conv, cb, f64mod(mc.q, mc.f64), lazy_max, tid, v);
      else conv_dot_f64<T, NTH>(smem, n_conv, p.bc_f64 + rd.aux2, f64mod(mc.q, mc.f64), lazy_max, tid, v);
    } else if (cstage) conv_dot<T, NTH, true>(smem, n_conv, reinterpret_cast<const u64 *>(cb), mc, p.max_terms, tid, v, ydbl);
    else conv_dot<T, NTH>(smem, n_conv, p.bc + rd.aux2, mc, p.max_terms, tid, v, ydbl);
    if (MERGED) {
      const ShoupC pt = p.mulc[rd.mod];
#pragma unroll
      for (int i = 0; i < 8; i++) v[i] = addmod(shoup_mul(v[i], pt.c, pt.cs, mc.q), fullred(outl[i], mc.q, mc.qbar), mc.q);
    }
    // the converted values go straight into the first forward round: its window sits on the top three tile bits, so the
    // elements it gives thread tid are tid + i NTH, the ones this thread has just produced
    static_assert(FirstRound<true, LT, LC, BCOL>::pw == LT - 3, "first forward round over the top tile bits");
    cp_async_wait_all();
    tile_sync<GRP>(bar);  // the twiddles are in place
    // ... and the last round's results leave from registers (same 32-byte runs per row as a drain through shared memory)
    constexpr int PWL = LastRound<true, LT, LC, BCOL>::pw;
    u64 r[8];
    tile_transform_ct<true, LT, LC, BCOL, GRP, 1, true, true>(W, G, twb, mc.q, tid, mc.f64, bar, v, r);
    u64 *dst = p.tmp + (size_t)b * p.tmp_bstride + (size_t)rd.dst_row * N;
    const int ebl = round_ebase<PWL>(tid);
#pragma unroll
    for (int k = 0; k < 8; k++) dst[G.gidx(ebl + (k << PWL))] = r[k];  // lazy, below 33q
    tile_sync<GRP>(bar);  // every thread is done with W before the next target's first round writes it
  }
}

// thread groups per block of the fused column kernel for digit groups of n_src limbs
// digits of 6-9 limbs: two groups per block, two blocks per SM; from 10 limbs four groups, one block per SM (config 5,
// measured: digits of 8 with two groups 4464 rotations/s, with four 4397; digits of 12 with two groups 3789, with four 4275)
#define CONV_NG4_FROM 10
static inline int convert_groups(int n_src, bool merged) { return (merged || n_src < 6) ? 1 : (n_src < CONV_NG4_FROM ? 2 : 4); }
static inline size_t convert_smem(int n_src, int ng) {  // source + work tiles, twiddle buffers, target descriptors
  return (size_t)(n_src + ng) * 8192 + (size_t)ng * CONV_TW_WORDS * 8 + (size_t)CONV_DESC_CAP * sizeof(TgtDesc);
}
bool convert_cols_fits(int logN, int n_src, bool merged) {
  return logN >= 12 && convert_smem(n_src, convert_groups(n_src, merged)) <= 227 * 1024;
}

int k_convert_cols(const KCtx &k, u64 *y, size_t y_bstride, const ConvGroup *groups, int n_groups, int n_src_max,
                   const ShoupC *scale, const u64 *bc, const RowDesc *rows, int n_tgt_total, u64 *tmp, size_t tmp_bstride,
                   int n_batch, int max_terms, const ShoupC *merged_pinv, const ShoupC *bc_f64) {
  if (n_groups == 0 || n_batch == 0) return 0;
  const NttGeom &g = k.geom;
  if (!convert_cols_fits(g.logN, n_src_max, merged_pinv != nullptr)) return -2;
  const int ng = convert_groups(n_src_max, merged_pinv != nullptr);
  const size_t smem = convert_smem(n_src_max, ng);
  ConvColP p{y, y_bstride, groups, scale, bc, rows, tmp, tmp_bstride, k.d_mods, k.d_tw_fwd, k.d_tw_inv, g.logN, g.brow, max_terms,
             merged_pinv, bc_f64, n_src_max + ng};
  dim3 grid(k.N >> 10, n_groups, n_batch);
  // algorithmic bytes: every target row written once (+ the sources, counted by the caller's row pass); butterflies: the
  // forward column stages of every target AND the inverse column stages of every source row (y holds y_bstride / N of them
  // per item at every call site); the base-conversion products (targets x sources per coefficient) are not counted
  PROF(k, K_NTT_COL_BCONV, 8.0 * k.N * n_batch * (double)n_tgt_total,
       HALF_N(k) * g.bcol * ((double)n_tgt_total + (double)(y_bstride / (size_t)k.N)) * n_batch);
#define LAUNCH_CONV1(B, M, G)                                                                                                         \
  do {                                                                                                                                \
    if (smem > 48 * 1024) cudaFuncSetAttribute(convert_cols_kernel<B, M, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
    convert_cols_kernel<B, M, G><<<grid, 128 * G, smem, (cudaStream_t)k.stream>>>(p);                                                 \
  } while (0)
#define LAUNCH_CONV(B)                         \
  do {                                         \
    if (merged_pinv) LAUNCH_CONV1(B, true, 1); \
    else if (ng == 4) LAUNCH_CONV1(B, false, 4); \
    else if (ng == 2) LAUNCH_CONV1(B, false, 2); \
    else LAUNCH_CONV1(B, false, 1);            \
  } while (0)
  switch (g.bcol) {
    case 4: LAUNCH_CONV(4); break;
    case 5: LAUNCH_CONV(5); break;
    case 6: LAUNCH_CONV(6); break;
    case 7: LAUNCH_CONV(7); break;
    default: LAUNCH_CONV(8); break;
  }
#undef LAUNCH_CONV
#undef LAUNCH_CONV1
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ forward, pass 1
struct NttColP {
  const u64 *src; size_t src_bstride; const u64 *bc; u64 *dst; size_t dst_bstride;
  const RowDesc *rows; const ModConst *mods; const ShoupC *tw; NttGeom g; int max_terms;
};
template <bool BCONV, int GEO>
__global__ void __launch_bounds__(512, 2) ntt_colpass_kernel(NttColP p) {
  extern __shared__ u64 sm[];
  const int tid = threadIdx.x, b = blockIdx.z;
  const RowDesc rd = p.rows[blockIdx.y];
  const int N = 1 << p.g.logN, T = 1 << p.g.lt_col;
  TileGeo G{p.g.lt_col, p.g.lc_col, p.g.brow, p.g.logN, blockIdx.x};
  const ModConst mc = p.mods[rd.mod];
  const u64 *src = p.src + (size_t)b * p.src_bstride + (size_t)rd.src_row * N;
  const int nth = blockDim.x;
  if (BCONV) {
    // fused base conversion (R2.6): sum_s y_s * (Qhat_s mod t), one Montgomery reduction
    const u64 *bc = p.bc + rd.aux2;
    const int ns = rd.aux;
    // source-major in two halves: the 4 elements' loads of one source row are in flight together
#pragma unroll
    for (int h = 0; h < 8; h += 4) {
      u64 lo[4], hi[4], r[4];
      u32 j[4];
#pragma unroll
      for (int i = 0; i < 4; i++) lo[i] = hi[i] = r[i] = 0, j[i] = G.gidx((tid + (h + i) * nth) & (T - 1));
      int lazy = 0;
      for (int s = 0; s < ns; s++) {
        const u64 c = __ldg(bc + s);
        u64 y[4];
#pragma unroll
        for (int i = 0; i < 4; i++) y[i] = __ldg(src + (size_t)s * N + j[i]);
#pragma unroll
        for (int i = 0; i < 4; i++) mac128(lo[i], hi[i], y[i], c);
        if (++lazy == p.max_terms) {  // keep the 128-bit sum below t 2^64 (only many 60-bit sources get here)
#pragma unroll
          for (int i = 0; i < 4; i++) r[i] = addmod(r[i], mont_redc(lo[i], hi[i], mc.q, mc.qinv_neg), mc.q), lo[i] = hi[i] = 0;
          lazy = 0;
        }
      }
#pragma unroll
      for (int i = 0; i < 4; i++) {
        const int e = tid + (h + i) * nth;
        if (e < T) sm[swz(e)] = addmod(r[i], mont_redc(lo[i], hi[i], mc.q, mc.qinv_neg), mc.q);
      }
    }
  } else {
    tile_fill(sm, T, tid, nth, [&](int e) { return __ldg(src + G.gidx(e)); });
  }
  __syncthreads();
  tile_transform<true, GEO>(sm, G, p.g.lc_col, p.g.bcol, p.tw + (size_t)rd.mod * N, mc.q, tid, mc.f64);
  u64 *dst = p.dst + (size_t)b * p.dst_bstride + (size_t)rd.dst_row * N;
  tile_drain(sm, T, tid, nth, [&](int e, u64 v) { dst[G.gidx(e)] = v; });  // lazy, below 33q
}

// ------------------------------------------------------------------------------------------------ forward, pass 2 (plain)
struct NttRowP {
  const u64 *src; size_t src_bstride; u64 *dst; size_t dst_bstride; const RowDesc *rows; const ModConst *mods;
  const ShoupC *tw; NttGeom g; int src_is_dst_row;
  int n_batch, bpb;  // SLAB: batch items per block
};
// ROW_TPB consecutive tiles of one row per block (compile-time geometries): the next tile's words are requested into
// registers before the current tile is transformed, so a block keeps loads in flight during its arithmetic (one tile
// per block left about 13 KB per SM in flight on average, a third of what HBM's latency needs).
// SLAB (batches of FENC_SLAB_MIN_BATCH items and more): the block stays on ONE tile position of its row and walks over
// p.bpb batch items, so the row pass's twiddles for that position (16 KB, twice the tile) are copied to shared memory
// once per block instead of being fetched from L2 by every round of every tile; the next item's tile is prefetched into
// registers all the same.
#ifndef FENC_ROW_TPB
#define FENC_ROW_TPB 4
#endif
#ifndef FENC_SLAB_MIN_BATCH
#define FENC_SLAB_MIN_BATCH 4
#endif
// batch items per block: the longer the walk, the fewer copies of the twiddles (config-4 step, 32 images: 2 items 618.5 ms,
// 4 items 605.9, 8 items 600.6, 16 items 599.1), as long as the grid still has blocks for every SM
// (8 waves of 148 x 6 blocks; config 2's grids at N = 2^14 are small and keep 4: with 16 its step went 6.49 -> 6.60 ms)
static inline int slab_bpb(long blocks_per_item, int n_batch) {
  for (int b = 16; b > 4; b >>= 1)
    if (blocks_per_item * ((n_batch + b - 1) / b) >= 8L * 148 * 6) return b;
  return 4;
}
static inline bool use_slab(const NttGeom &g, int n_batch) { return g.logN >= 12 && n_batch >= FENC_SLAB_MIN_BATCH; }
static inline size_t slab_bytes(const NttGeom &g) {  // tile, twiddle slab, the item descriptors of the divide pass
  return (sizeof(u64) << g.lt_row) + (sizeof(ShoupC) << g.lt_row) + 16 * sizeof(BatchItem);
}
template <int GEO, bool SLAB = false>
__global__ void __launch_bounds__(GEO == 1 ? 128 : 256, GEO == 1 ? 6 : 4) ntt_rowpass_kernel(NttRowP p) {
  static_assert(!SLAB || GEO == 1, "slabs: compile-time row geometry");
  extern __shared__ u64 sm[];
  const int tid = threadIdx.x;
  const RowDesc rd = p.rows[blockIdx.y];
  const int N = 1 << p.g.logN, T = 1 << p.g.lt_row;
  constexpr int TPB = GEO == 1 ? FENC_ROW_TPB : 1;
  const int b0 = SLAB ? blockIdx.z * p.bpb : blockIdx.z;
  const int n_it = SLAB ? min(p.bpb, p.n_batch - b0) : TPB;
  const size_t src_off = (size_t)(p.src_is_dst_row ? rd.dst_row : rd.src_row) * N, dst_off = (size_t)rd.dst_row * N;
  const int nth = blockDim.x;
  const ModConst mc = p.mods[rd.mod];
  ShoupC *slab = reinterpret_cast<ShoupC *>(sm + T);
  u64 v[8];
  // REG (compile-time row geometry, slab form or not): the tile is loaded in the order of the transform's first round
  // (element round_ebase(tid) + (i << PW0): runs of 32 consecutive words per warp and i), which takes it from the registers:
  // no fill, one barrier less per tile, and the next tile is requested into the same registers right behind that round
  constexpr bool REG = GEO == 1;
  constexpr int PW0 = FirstRound<true, FENC_ROW_LT, 0, 8>::pw;
  const int eb0 = round_ebase<PW0>(tid);
  auto request = [&](int k) {
    TileGeo G{p.g.lt_row, p.g.lt_row, 0, p.g.logN, SLAB ? blockIdx.x : blockIdx.x * TPB + k};
    const u64 *src = p.src + (size_t)(SLAB ? b0 + k : b0) * p.src_bstride + src_off;
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const int e = REG ? eb0 + (i << PW0) : tid + i * nth;
      if (e < T) v[i] = src[G.gidx(e)];
    }
  };
  request(0);
  if constexpr (SLAB) tw_slab_fill<FENC_ROW_LT>(slab, p.tw + (size_t)rd.mod * N, p.g.logN, blockIdx.x, tid, nth);
#pragma unroll 1
  for (int k = 0; k < n_it; k++) {
    TileGeo G{p.g.lt_row, p.g.lt_row, 0, p.g.logN, SLAB ? blockIdx.x : blockIdx.x * TPB + k};
    u64 *dst = p.dst + (size_t)(SLAB ? b0 + k : b0) * p.dst_bstride + dst_off;
    if constexpr (REG) {
      if (SLAB && k == 0) {
        tw_slab_wait();
        __syncthreads();
      }
      auto next = [&]() { if (k + 1 < n_it) request(k + 1); };
      // the last round (window on the lowest bits) leaves its eight consecutive results in registers: 64 bytes per thread,
      // stored as four 16-byte words
      static_assert(LastRound<true, FENC_ROW_LT, 0, 8>::pw == 0, "last forward row round over the lowest tile bits");
      u64 r[8];
      if constexpr (SLAB) tile_transform<true, GEO, 2, true, decltype(next), true>(sm, row_slab_geo<FENC_ROW_LT>(), 0, p.g.brow, slab, mc.q, tid, mc.f64, v, next, r);
      else tile_transform<true, GEO, 0, true, decltype(next), true>(sm, G, 0, p.g.brow, p.tw + (size_t)rd.mod * N, mc.q, tid, mc.f64, v, next, r);
      ulonglong2 *d2 = reinterpret_cast<ulonglong2 *>(dst + G.gidx(8 * tid));
#pragma unroll
      for (int i = 0; i < 4; i++) d2[i] = make_ulonglong2(fullred(r[2 * i], mc.q, mc.qbar), fullred(r[2 * i + 1], mc.q, mc.qbar));
    } else {
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const int e = tid + i * nth;
      if (e < T) sm[swz(e)] = v[i];
    }
    __syncthreads();
    if (k + 1 < n_it) request(k + 1);
    tile_transform<true, GEO>(sm, G, 0, p.g.brow, p.tw + (size_t)rd.mod * N, mc.q, tid, mc.f64);
    tile_drain(sm, T, tid, nth, [&](int e, u64 x) { dst[G.gidx(e)] = fullred(x, mc.q, mc.qbar); });
    }
    if (k + 1 < n_it) __syncthreads();  // every thread is done with the tile before the next one overwrites it
  }
}
// launch of the forward row pass over (rows x batch), slab form for batches
static void launch_ntt_rowpass(const KCtx &k, NttRowP r, int n_rows, int n_batch) {
  const NttGeom &g = k.geom;
  cudaStream_t st = (cudaStream_t)k.stream;
  r.n_batch = n_batch, r.bpb = slab_bpb((long)(k.N >> g.lt_row) * n_rows, n_batch);
  if (use_slab(g, n_batch)) {
    dim3 sgrid(k.N >> g.lt_row, n_rows, (n_batch + r.bpb - 1) / r.bpb);
    ntt_rowpass_kernel<1, true><<<sgrid, nthreads_for(g.lt_row), slab_bytes(g), st>>>(r);
  } else {
    dim3 grid2((unsigned)((k.N >> g.lt_row) / (g.logN >= 12 ? FENC_ROW_TPB : 1)), n_rows, n_batch);
    ROW_GEO(g, (ntt_rowpass_kernel<GEO><<<grid2, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, st>>>(r)));
  }
}
static inline unsigned row_grid_x(const NttGeom &g, int N) { return (unsigned)((N >> g.lt_row) / (g.logN >= 12 ? FENC_ROW_TPB : 1)); }

int k_ntt(const KCtx &k, const u64 *src, size_t src_bstride, u64 *dst, size_t dst_bstride, const RowDesc *rows, int n_rows,
          int n_batch) {
  if (n_rows == 0 || n_batch == 0) return 0;
  cudaStream_t st = (cudaStream_t)k.stream;
  const NttGeom &g = k.geom;
  NttColP a{src, src_bstride, nullptr, dst, dst_bstride, rows, k.d_mods, k.d_tw_fwd, g, 1 << 30};
  dim3 grid1(k.N >> g.lt_col, n_rows, n_batch);
  PROF(k, K_NTT_COL, 16.0 * k.N * n_rows * n_batch, HALF_N(k) * g.bcol * n_rows * n_batch);
  COL_GEO(g, (ntt_colpass_kernel<false, GEO><<<grid1, nthreads_for(g.lt_col), sizeof(u64) << g.lt_col, st>>>(a)));
  LAUNCH_CHECK(k);
  NttRowP r{dst, dst_bstride, dst, dst_bstride, rows, k.d_mods, k.d_tw_fwd, g, 1};
  PROF(k, K_NTT_ROW, 16.0 * k.N * n_rows * n_batch, HALF_N(k) * g.brow * n_rows * n_batch);
  launch_ntt_rowpass(k, r, n_rows, n_batch);
  LAUNCH_CHECK(k);
  return 0;
}

// forward pass 2 alone, in place on rows[r].dst_row of buf (rows that a column kernel left in their lazy form): canonical
int k_ntt_rows_only(const KCtx &k, u64 *buf, size_t bstride, const RowDesc *rows, int n_rows, int n_batch) {
  if (n_rows == 0 || n_batch == 0) return 0;
  const NttGeom &g = k.geom;
  NttRowP r{buf, bstride, buf, bstride, rows, k.d_mods, k.d_tw_fwd, g, 1};
  PROF(k, K_NTT_ROW, 16.0 * k.N * n_rows * n_batch, HALF_N(k) * g.brow * n_rows * n_batch);
  launch_ntt_rowpass(k, r, n_rows, n_batch);
  LAUNCH_CHECK(k);
  return 0;
}

int k_ntt_cols_bconv(const KCtx &k, const u64 *y, size_t y_bstride, const u64 *bc, u64 *tmp, size_t tmp_bstride,
                     const RowDesc *rows, int n_rows, int n_batch, int n_src_rows, int max_terms) {
  if (n_rows == 0 || n_batch == 0) return 0;
  const NttGeom &g = k.geom;
  NttColP a{y, y_bstride, bc, tmp, tmp_bstride, rows, k.d_mods, k.d_tw_fwd, g, max_terms};
  dim3 grid1(k.N >> g.lt_col, n_rows, n_batch);
  // algorithmic bytes: every source row read once, every target row written once
  PROF(k, K_NTT_COL_BCONV, 8.0 * k.N * ((double)n_src_rows + n_rows) * n_batch, HALF_N(k) * g.bcol * n_rows * n_batch);
  COL_GEO(g, (ntt_colpass_kernel<true, GEO><<<grid1, nthreads_for(g.lt_col), sizeof(u64) << g.lt_col, (cudaStream_t)k.stream>>>(a)));
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ forward pass 2 + evk inner product (a4)
// One block = one tile of one target row t for one batch item; it loops over the beta digits, finishing the NTT of
// ModUp_j(d)[t] in shared memory and accumulating x * evk_j.{b,a}[t] in 128-bit registers: the extended digits never
// exist in NTT form in HBM, and each evk element is read exactly once per batch item (blocks of one tile that differ
// only in the batch index are adjacent in launch order, so the key tile is served from L2 after its first read).
struct KeyMacP {
  const BatchItem *items; const int *tmp_index; const u64 *tmp; size_t tmp_bstride; u64 *acc; size_t acc_bstride;
  const ModConst *mods; const ShoupC *tw; NttGeom g; int L, E, beta, A, nq, n_batch;
};
// 3 blocks of 128 threads per SM: 168 registers hold the 32 128-bit accumulators and the fp64 butterflies without
// spilling (4 blocks at 128 registers spill 160 bytes and run 10 % slower)
#define KEYMAC_BLOCKS 3
template <int EPT, int GEO>  // elements per thread
__global__ void __launch_bounds__(GEO == 1 ? 128 : 256, GEO == 1 ? KEYMAC_BLOCKS : 2) ntt_rows_keymac_kernel(KeyMacP p) {
  extern __shared__ u64 sm_all[];  // two tiles: the next digit's words arrive (cp.async) while this one is transformed
  const int tid = threadIdx.x;
  // batch index fastest: blockIdx.x = tile * n_batch + b
  const int nb = p.n_batch, b = blockIdx.x % nb, tile = blockIdx.x / nb, t = blockIdx.y;
  const int N = 1 << p.g.logN, T = 1 << p.g.lt_row;
  TileGeo G{p.g.lt_row, p.g.lt_row, 0, p.g.logN, (u32)tile};
  const int mod = t < p.L ? t : p.nq + (t - p.L);
  const ModConst mc = p.mods[mod];
  const BatchItem it = p.items[b];
  u64 a0l[EPT], a0h[EPT], a1l[EPT], a1h[EPT];
#pragma unroll
  for (int i = 0; i < EPT; i++) a0l[i] = a0h[i] = a1l[i] = a1h[i] = 0;
  const int nth = blockDim.x;
  constexpr int HB = EPT < 4 ? EPT : 4;
  auto request = [&](int j) {  // digit j's tile of the ModUp temp -> buffer j & 1 (nothing to fetch inside the digit)
    const int ti = p.tmp_index[j * p.E + t];
    if (ti >= 0) {
      const u64 *src = p.tmp + (size_t)b * p.tmp_bstride + (size_t)ti * N;
      u64 *dst = sm_all + (size_t)(j & 1) * T;
#pragma unroll
      for (int i = 0; i < EPT; i++) {
        const int e = tid + i * nth;
        if (e < T) cp_async8(dst + swz(e), src + G.gidx(e));
      }
    }
    cp_async_commit();
  };
  request(0);
  // compile-time row geometry: the beta transforms of the block share tile position and modulus, so their twiddles are
  // copied to shared memory once (the slab of the row passes, behind the tiles and the key words)
  ShoupC *slab = reinterpret_cast<ShoupC *>(sm_all + 4 * (size_t)T);
  if constexpr (GEO == 1) tw_slab_fill<FENC_ROW_LT>(slab, p.tw + (size_t)mod * N, p.g.logN, (u32)tile, tid, nth);
  for (int j = 0; j < p.beta; j++) {
    const int ti = p.tmp_index[j * p.E + t];
    const u64 *kb = it.evk + ((size_t)(j * 2 + 0) * p.A + mod) * N;
    const u64 *ka = it.evk + ((size_t)(j * 2 + 1) * p.A + mod) * N;
    u64 *sm = sm_all + (size_t)(j & 1) * T;
    cp_async_wait_all();
    __syncthreads();  // digit j's tile is complete, and every thread is done with the other buffer (digit j-1)
    if (j + 1 < p.beta) request(j + 1);
    // KEYS (compile-time row geometry): this digit's key words for the thread's own elements are requested into shared
    // memory before the transform and read after it (every thread owns its slots: no barrier).  Loaded after the transform
    // in two batches of four elements, their latency was exposed twice per digit: the kernel has 12 warps per SM at 168
    // registers to hide it with.
    constexpr bool KEYS = GEO == 1;
    u64 *skb = sm_all + 2 * (size_t)T, *ska = skb + T;
    if constexpr (KEYS) {
#pragma unroll
      for (int i = 0; i < EPT; i++) {
        const int e = (tid + i * nth) & (T - 1);
        const u32 jj = G.gidx(e);
        cp_async8(skb + e, kb + jj);
        cp_async8(ska + e, ka + jj);
      }
      cp_async_commit();
    }
    if (ti >= 0) {
      if constexpr (GEO == 1) tile_transform<true, GEO, 2>(sm, row_slab_geo<FENC_ROW_LT>(), 0, p.g.brow, slab, mc.q, tid, mc.f64);
      else tile_transform<true, GEO>(sm, G, 0, p.g.brow, p.tw + (size_t)mod * N, mc.q, tid, mc.f64);
    }
    if constexpr (KEYS) cp_async_wait_all();  // (the next digit's tile has had the transform's time as well)
    // the key words (and, inside the digit, the permuted input words) of 4 elements are loaded together, then used
#pragma unroll
    for (int h = 0; h < EPT; h += HB) {
      u64 x[HB], vb[HB], va[HB];
      u32 jj[HB];
#pragma unroll
      for (int i = 0; i < HB; i++) {
        const int e = (tid + (h + i) * nth) & (T - 1);
        jj[i] = G.gidx(e);
        vb[i] = KEYS ? skb[e] : __ldg(kb + jj[i]);
        va[i] = KEYS ? ska[e] : __ldg(ka + jj[i]);
        if (ti >= 0) x[i] = sm[swz(e)];
        else x[i] = __ldg(it.ks_in + (size_t)t * N + galois_src(jj[i], it.g, p.g.logN));
      }
#pragma unroll
      for (int i = 0; i < HB; i++) {
        if (tid + (h + i) * nth < T) {
          // fp64 rows: the transform's output is below 2^52 with q < 2^45, beta x k stays far below q 2^64: no reduction
          const u64 xx = (ti >= 0 && !mc.f64) ? fullred(x[i], mc.q, mc.qbar) : x[i];
          mac128(a0l[h + i], a0h[h + i], xx, vb[i]);
          mac128(a1l[h + i], a1h[h + i], xx, va[i]);
        }
      }
    }
  }
  u64 *o0 = p.acc + (size_t)b * p.acc_bstride + (size_t)t * N;
  u64 *o1 = o0 + (size_t)p.E * N;
#pragma unroll
  for (int i = 0; i < EPT; i++) {
    const int e = tid + i * nth;
    if (e < T) {
      const u32 jj = G.gidx(e);
      o0[jj] = mont_redc(a0l[i], a0h[i], mc.q, mc.qinv_neg);
      o1[jj] = mont_redc(a1l[i], a1h[i], mc.q, mc.qinv_neg);
    }
  }
}

int k_ntt_rows_keymac(const KCtx &k, const BatchItem *items, int L, int E, int beta, const int *tmp_index, const u64 *tmp,
                      size_t tmp_bstride, u64 *acc, size_t acc_bstride, int n_batch, int n_up, int n_distinct_keys) {
  if (n_batch == 0) return 0;
  const NttGeom &g = k.geom;
  KeyMacP p{items, tmp_index, tmp, tmp_bstride, acc, acc_bstride, k.d_mods, k.d_tw_fwd, g, L, E, beta, k.nq + k.np, k.nq,
            n_batch};
  const int nth = nthreads_for(g.lt_row);
  dim3 grid((k.N >> g.lt_row) * n_batch, E, 1);
  const int ept = ((1 << g.lt_row) + nth - 1) / nth;
  // algorithmic bytes: ModUp temp + the switched polynomial read once, accumulators written once, each key once
  PROF(k, K_KEYMAC, 8.0 * k.N * (((double)n_up + L + 2.0 * E) * n_batch + 2.0 * beta * E * n_distinct_keys),
       HALF_N(k) * g.brow * n_up * n_batch);
  if (g.logN >= 12) {  // two tiles + the key words + the twiddle slab: 48 KiB
    static bool attr_set = false;
    if (!attr_set) {
      cudaFuncSetAttribute(ntt_rows_keymac_kernel<8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(6 * (sizeof(u64) << FENC_ROW_LT)));
      attr_set = true;
    }
    ntt_rows_keymac_kernel<8, 1><<<grid, nth, 6 * (sizeof(u64) << g.lt_row), (cudaStream_t)k.stream>>>(p);
  }
  else if (ept <= 1) ntt_rows_keymac_kernel<1, 0><<<grid, nth, 2 * (sizeof(u64) << g.lt_row), (cudaStream_t)k.stream>>>(p);
  else if (ept <= 4) ntt_rows_keymac_kernel<4, 0><<<grid, nth, 2 * (sizeof(u64) << g.lt_row), (cudaStream_t)k.stream>>>(p);
  else ntt_rows_keymac_kernel<8, 0><<<grid, nth, 2 * (sizeof(u64) << g.lt_row), (cudaStream_t)k.stream>>>(p);
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ evk inner product of a hoisted rotation (R2.7b)
// The extended digits of the source ciphertext's c1 are already in NTT form (up: [source][n_up][N], canonical; the
// digit's own limbs are the ciphertext's): a rotation is the Galois gather of those rows times its key, accumulated over
// the digits -- no transform.  Rotations of one source re-read its rows from L2; items sharing a key are neighbours.
struct HoistMacP {
  const BatchItem *items; const int *tmp_index; const u64 *up; size_t up_sstride; u64 *acc; size_t acc_bstride;
  const ModConst *mods; int logN, L, E, beta, A, nq, n_batch;
};
// Each thread owns the adjacent positions 2i, 2i+1: their Galois sources are adjacent too (the lowest position bit is
// the highest bit of the exponent index, which an odd multiplier maps to itself), so x, b and a all arrive as 16-byte
// loads; the loads of digit j+1 are issued before the products of digit j.
struct HoistOperands { ulonglong2 x, b, a; };
__global__ void __launch_bounds__(256, 4) hoisted_keymac_kernel(HoistMacP p) {
  const int tid = threadIdx.x, nb = p.n_batch, b = blockIdx.x % nb, chunk = blockIdx.x / nb, t = blockIdx.y;
  const int N = 1 << p.logN;
  const int mod = t < p.L ? t : p.nq + (t - p.L);
  const ModConst mc = p.mods[mod];
  const BatchItem it = p.items[b];
  const u32 pos = 2u * ((u32)chunk * 256u + tid);
  if (pos >= (u32)N) return;
  const u32 src = galois_src(pos, it.g, p.logN);  // source of pos; pos + 1 reads src ^ 1
  const bool swap = src & 1u;
  auto fetch = [&](int j) {
    const int ti = p.tmp_index[j * p.E + t];
    const u64 *x = ti >= 0 ? p.up + (size_t)it.pad * p.up_sstride + (size_t)ti * N : it.ks_in + (size_t)t * N;
    const u64 *kb = it.evk + ((size_t)(j * 2 + 0) * p.A + mod) * N;
    const u64 *ka = it.evk + ((size_t)(j * 2 + 1) * p.A + mod) * N;
    HoistOperands o;
    o.x = __ldg(reinterpret_cast<const ulonglong2 *>(x + (src & ~1u)));
    o.b = __ldg(reinterpret_cast<const ulonglong2 *>(kb + pos));
    o.a = __ldg(reinterpret_cast<const ulonglong2 *>(ka + pos));
    return o;
  };
  u64 a0l[2] = {0, 0}, a0h[2] = {0, 0}, a1l[2] = {0, 0}, a1h[2] = {0, 0};
  HoistOperands cur = fetch(0);
  for (int j = 0; j < p.beta; j++) {
    HoistOperands nxt = cur;
    if (j + 1 < p.beta) nxt = fetch(j + 1);
    const u64 x0 = swap ? cur.x.y : cur.x.x, x1 = swap ? cur.x.x : cur.x.y;
    mac128(a0l[0], a0h[0], x0, cur.b.x), mac128(a1l[0], a1h[0], x0, cur.a.x);
    mac128(a0l[1], a0h[1], x1, cur.b.y), mac128(a1l[1], a1h[1], x1, cur.a.y);
    cur = nxt;
  }
  u64 *o0 = p.acc + (size_t)b * p.acc_bstride + (size_t)t * N;
  u64 *o1 = o0 + (size_t)p.E * N;
  *reinterpret_cast<ulonglong2 *>(o0 + pos) =
      make_ulonglong2(mont_redc(a0l[0], a0h[0], mc.q, mc.qinv_neg), mont_redc(a0l[1], a0h[1], mc.q, mc.qinv_neg));
  *reinterpret_cast<ulonglong2 *>(o1 + pos) =
      make_ulonglong2(mont_redc(a1l[0], a1h[0], mc.q, mc.qinv_neg), mont_redc(a1l[1], a1h[1], mc.q, mc.qinv_neg));
}
int k_hoisted_keymac(const KCtx &k, const BatchItem *items, int L, int E, int beta, const int *tmp_index, const u64 *up,
                     size_t up_sstride, u64 *acc, size_t acc_bstride, int n_batch, int n_distinct_keys, int n_sources, int n_up) {
  if (n_batch == 0) return 0;
  HoistMacP p{items, tmp_index, up, up_sstride, acc, acc_bstride, k.d_mods, k.geom.logN, L, E, beta, k.nq + k.np, k.nq, n_batch};
  if (k.N < 2) return -2;
  const int chunks = (k.N / 2 + 255) / 256;
  dim3 grid(chunks * n_batch, E, 1);
  // algorithmic bytes: accumulators written once, each key and each source's extended digits read once
  PROF(k, K_KEYMAC, 8.0 * k.N * (2.0 * E * n_batch + 2.0 * beta * E * n_distinct_keys + ((double)n_up + L) * n_sources), 0);
  hoisted_keymac_kernel<<<grid, 256, 0, (cudaStream_t)k.stream>>>(p);
  LAUNCH_CHECK(k);
  return 0;
}

// ------------------------------------------------------------------------------------------------ forward pass 2 + divide epilogue (a5, a8)
// X = NTT(Conv_{dropped -> t}(.)) finished here; out = (minuend - X) * mul[t] (+ addend through the Galois gather).
struct DivideP {
  const BatchItem *items; const u64 *tmp; size_t tmp_bstride; const u64 *acc; size_t acc_bstride; const ShoupC *mul;
  const RowDesc *rows; const ModConst *mods; const ShoupC *tw; NttGeom g; int from_items;
  const ShoupC *mul2;  // MERGED: out = ((minuend mul2 + addend) - X) mul   (mul2 = P^-1, mul = q_{L-1}^-1)
  int n_batch, bpb;    // SLAB: batch items per block
};
// SLAB (batches of FENC_SLAB_MIN_BATCH items and more): the block stays on ONE tile position of its row and walks over
// p.bpb batch items, so the row pass's twiddles for that position (16 KB, twice the tile) are copied to shared memory
// once per block instead of being fetched from L2 by every round of every tile; the next item's tile is prefetched into
// registers as before.  Otherwise: FENC_ROW_TPB consecutive tiles of one item's row per block.
template <int GEO, bool MERGED = false, bool SLAB = false>
__global__ void __launch_bounds__(GEO == 1 ? 128 : 256, 4) ntt_rows_divide_kernel(DivideP p) {
  static_assert(!SLAB || GEO == 1, "slabs: compile-time row geometry");
  extern __shared__ u64 sm[];
  const int tid = threadIdx.x;
  const RowDesc rd = p.rows[blockIdx.y];
  const int N = 1 << p.g.logN, T = 1 << p.g.lt_row;
  constexpr int TPB = GEO == 1 ? FENC_ROW_TPB : 1;  // tiles per block, the next one prefetched (see ntt_rowpass_kernel)
  const int nth = blockDim.x, logN = p.g.logN;
  const ModConst mq = p.mods[rd.mod];
  const u64 q = mq.q;
  const ShoupC mc = p.mul[rd.mod];
  const F64Mod fm = f64mod(q, mq.f64);
  const int b0 = SLAB ? blockIdx.z * p.bpb : blockIdx.z;
  const int n_it = SLAB ? min(p.bpb, p.n_batch - b0) : TPB;
  ShoupC *slab = reinterpret_cast<ShoupC *>(sm + T);
  u64 v[8];
  constexpr int PW0 = FirstRound<true, FENC_ROW_LT, 0, 8>::pw;  // SLAB: tile loaded in the first round's order (ntt_rowpass_kernel)
  const int eb0 = round_ebase<PW0>(tid);
  auto request = [&](int k) {  // iteration k's tile of the temp
    TileGeo G{p.g.lt_row, p.g.lt_row, 0, p.g.logN, SLAB ? blockIdx.x : blockIdx.x * TPB + k};
    const u64 *src = p.tmp + (size_t)(SLAB ? b0 + k : b0) * p.tmp_bstride + (size_t)rd.src_row * N;
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const int e = SLAB ? eb0 + (i << PW0) : tid + i * nth;
      if (e < T) v[i] = src[G.gidx(e)];
    }
  };
  request(0);
  // SLAB: the descriptors of the block's items are copied to shared memory behind the slab (read from global memory one
  // iteration ahead, their first use -- a pointer moved to a uniform register -- still held 5 % of the stall samples)
  BatchItem *s_items = reinterpret_cast<BatchItem *>(sm + 3 * (size_t)T);
  if constexpr (SLAB) {
    tw_slab_fill<FENC_ROW_LT>(slab, p.tw + (size_t)rd.mod * N, logN, blockIdx.x, tid, nth);
    static_assert(sizeof(BatchItem) % 8 == 0, "copied as 64-bit words");
    for (int i = tid; i < n_it * (int)(sizeof(BatchItem) / 8); i += nth)
      reinterpret_cast<u64 *>(s_items)[i] = reinterpret_cast<const u64 *>(p.items + b0)[i];
  }
#pragma unroll 1
  for (int k = 0; k < n_it; k++) {
    const int b = SLAB ? b0 + k : b0;
    TileGeo G{p.g.lt_row, p.g.lt_row, 0, p.g.logN, SLAB ? blockIdx.x : blockIdx.x * TPB + k};
    if constexpr (SLAB) {
      if (k == 0) {
        tw_slab_wait();
        __syncthreads();  // slab and item descriptors are in place
      }
    } else {
#pragma unroll
      for (int i = 0; i < 8; i++) {
        const int e = tid + i * nth;
        if (e < T) sm[swz(e)] = v[i];
      }
      __syncthreads();
    }
    const BatchItem it = SLAB ? s_items[k] : p.items[b0];
    const u64 *minuend = (p.from_items ? it.sub_in : p.acc + (size_t)b * p.acc_bstride) + (size_t)rd.aux2 * N;
    const u64 *addend = rd.aux == 0 ? it.add0 : it.add1;
    if (addend) addend += (size_t)rd.mod * N;
    u64 *dst = it.out + (size_t)rd.dst_row * N;
    const u32 gal = it.g;
    // epilogue operands of this tile and the words of the next tile are fetched BEFORE the transform: their latency hides behind it
    // SLAB: the last round keeps its results in registers (eight consecutive coefficients per thread), so the epilogue's
    // operands are fetched in that order (16-byte loads) and the output leaves as four 16-byte stores
    u64 mi[8], ad[8], xr[8];
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const u32 j = G.gidx(SLAB ? 8 * tid + i : (tid + i * nth) & (T - 1));
      if (!SLAB) mi[i] = __ldg(minuend + j);
      ad[i] = addend ? __ldg(addend + galois_src(j, gal, logN)) : 0;
    }
    if constexpr (SLAB) {
      const ulonglong2 *m2p = reinterpret_cast<const ulonglong2 *>(minuend + G.gidx(8 * tid));
#pragma unroll
      for (int i = 0; i < 4; i++) {
        const ulonglong2 m = __ldg(m2p + i);
        mi[2 * i] = m.x, mi[2 * i + 1] = m.y;
      }
      auto next = [&]() { if (k + 1 < n_it) request(k + 1); };
      tile_transform<true, GEO, 2, true, decltype(next), true>(sm, row_slab_geo<FENC_ROW_LT>(), 0, p.g.brow, slab, q, tid, mq.f64, v, next, xr);
    } else {
      if (k + 1 < n_it) request(k + 1);
      tile_transform<true, GEO>(sm, G, 0, p.g.brow, p.tw + (size_t)rd.mod * N, q, tid, mq.f64);
    }
    u64 res[8];
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const int e = SLAB ? 8 * tid + i : tid + i * nth;
      if (e < T) {
        // fp64 rows: X mod q as v - rint(v/q) q + q in (0, 2q) on the FP64 pipe; the Shoup multiply takes any 64-bit input
        const bool fp = mq.f64 != 0;
        const u64 xv = SLAB ? xr[i] : sm[swz(e)];
        const u64 x = fp ? d2u_off(reduce_dd(u2d52(xv), fm), fm.q + 4503599627370496.0) : fullred(xv, q, mq.qbar);
        u64 r;
        if (MERGED) {
          const ShoupC m2 = p.mul2[rd.mod];
          r = addmod(shoup_mul(mi[i], m2.c, m2.cs, q), ad[i], q);
          r = shoup_mul(fp ? r + 2 * q - x : submod(r, x, q), mc.c, mc.cs, q);
        } else {
          r = shoup_mul(fp ? mi[i] + 2 * q - x : submod(mi[i], x, q), mc.c, mc.cs, q);
          r = addmod(r, ad[i], q);
        }
        if (SLAB) res[i] = r;
        else dst[G.gidx(e)] = r;
      }
    }
    if constexpr (SLAB) {
      ulonglong2 *d2 = reinterpret_cast<ulonglong2 *>(dst + G.gidx(8 * tid));
#pragma unroll
      for (int i = 0; i < 4; i++) d2[i] = make_ulonglong2(res[2 * i], res[2 * i + 1]);
    }
    if (k + 1 < n_it) __syncthreads();
  }
}

int k_ntt_rows_divide(const KCtx &k, const BatchItem *items, const u64 *tmp, size_t tmp_bstride, const u64 *acc,
                      size_t acc_bstride, bool minuend_from_items, const ShoupC *mul, const RowDesc *rows, int n_rows,
                      int n_batch, const ShoupC *merged_mul2) {
  if (n_rows == 0 || n_batch == 0) return 0;
  const NttGeom &g = k.geom;
  DivideP p{items, tmp, tmp_bstride, acc, acc_bstride, mul, rows, k.d_mods, k.d_tw_fwd, g, minuend_from_items ? 1 : 0, merged_mul2,
            n_batch, slab_bpb((long)(k.N >> g.lt_row) * n_rows, n_batch)};
  dim3 grid(row_grid_x(g, k.N), n_rows, n_batch);
  PROF(k, K_DIVIDE, 8.0 * k.N * (3.5 * n_rows) * n_batch, HALF_N(k) * g.brow * n_rows * n_batch);  // temp + minuend + output, addend on half the rows
  if (use_slab(g, n_batch)) {
    dim3 sgrid(k.N >> g.lt_row, n_rows, (n_batch + p.bpb - 1) / p.bpb);
    if (merged_mul2) ntt_rows_divide_kernel<1, true, true><<<sgrid, nthreads_for(g.lt_row), slab_bytes(g), (cudaStream_t)k.stream>>>(p);
    else ntt_rows_divide_kernel<1, false, true><<<sgrid, nthreads_for(g.lt_row), slab_bytes(g), (cudaStream_t)k.stream>>>(p);
  } else if (merged_mul2)
    ROW_GEO(g, (ntt_rows_divide_kernel<GEO, true><<<grid, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, (cudaStream_t)k.stream>>>(p)));
  else
    ROW_GEO(g, (ntt_rows_divide_kernel<GEO><<<grid, nthreads_for(g.lt_row), sizeof(u64) << g.lt_row, (cudaStream_t)k.stream>>>(p)));
  LAUNCH_CHECK(k);
  return 0;
}
