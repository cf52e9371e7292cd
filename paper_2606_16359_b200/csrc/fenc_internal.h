// fenc_internal.h -- shared declarations of libfenc's translation units (not part of the public ABI).
// Nothing here is shared with oracle/ (the CPU oracle is an independent program).
#pragma once
#include <stddef.h>
#include <string.h>
#include <stdint.h>

#include <vector>

#include "../../include/fenc.h"

typedef uint64_t u64;
typedef uint32_t u32;
typedef unsigned __int128 u128;
typedef long long i64;

#define FENC_MAX_MOD 96
#ifndef FENC_ROW_LT
#define FENC_ROW_LT 10  // log2 elements of a row-pass tile for N >= 2^12 (8 stages on 2^FENC_ROW_LT contiguous coefficients)
#endif  // moduli per context (n_q + n_p)

// ---------------------------------------------------------------- device-visible tables
struct ModConst {  // one per modulus, device global memory
  u64 q;           // prime, < 2^61
  u64 qinv_neg;    // -q^{-1} mod 2^64 (Montgomery)
  u64 r2;          // 2^128 mod q: mont_mul(x, r2) = x 2^64 mod q
  u64 mask;        // 2^ceil(log2 q) - 1 (uniform rejection sampler)
  u64 qbar;        // floor(2^64 / q): full reduction of a lazy 64-bit value
  u64 f64;         // != 0: fp64 butterflies (q < 2^45, or q < 2^50 with N >= 2^12): the bits of (double)(1/q); the twiddle
                   // tables of this modulus hold fp64 pairs (fenc_device.cuh mulmod_dd)
  u64 pad[2];
};

struct ShoupC {  // constant c with its Shoup companion floor(c 2^64 / q)
  u64 c, cs;
};

// one job row of a batched NTT launch
struct RowDesc {
  int mod;      // modulus index
  int src_row;  // row in the source tensor (first source row for a base conversion)
  int dst_row;  // row in the destination tensor
  int aux;      // base conversion: number of source rows; divide epilogue: component (0/1)
  int aux2;     // base conversion: offset of this row's constants; divide epilogue: row in the minuend tensor
  int pad[3];
};

#define FENC_MAC_GROUP 4
struct MacGroup {
  int n_out, n_terms, ct_start, pt_start, out_start, pad[3];
};

// one element of a batch of key switches (rotations, relinearisations, rescales)
struct BatchItem {
  const u64 *ks_in;  // polynomial to switch [L][N] (NTT domain); rotation: c1 of the input
  const u64 *sub_in; // rescale: the input ciphertext [2][L][N] (minuend of the divide epilogue)
  u64 *out;          // output ciphertext [2][L_out][N]
  const u64 *evk;    // switching key [beta_max][2][A][N] (NTT domain, Montgomery form)
  const u64 *add0;   // epilogue addend for component 0 ([L][N], read through the Galois gather) or NULL
  const u64 *add1;   // epilogue addend for component 1 or NULL
  u32 g;             // Galois element (1 = identity)
  u32 pad;           // hoisted rotations: index of the source ciphertext whose extended digits this item reads
};

// geometry of the 2-pass NTT for one ring degree
struct NttGeom {
  int logN;
  int brow;    // stages done by the row pass (contiguous sub-transforms of 2^brow points)
  int bcol;    // stages done by the column pass (stride 2^brow)
  int lt_row;  // log2 tile elements of the row pass
  int lt_col;  // log2 tile elements of the column pass
  int lc_col;  // log2 columns per tile of the column pass
};

// per-kernel-class timing with CUDA events on the launching stream (measurement only; off by default)
enum KernelId {
  K_INTT_ROW, K_INTT_COL, K_NTT_COL, K_NTT_COL_BCONV, K_NTT_ROW, K_KEYMAC, K_DIVIDE, K_MAC, K_ADD_MANY, K_ROWOP, K_SAMPLE,
  K_SMAC, K_COUNT
};
struct Prof;
void prof_begin(Prof *p, void *stream, int id, double alg_bytes, double alg_butterflies = 0);
void prof_end(Prof *p, void *stream);

// one base-conversion group of the fused column kernel: n_src consecutive source rows (row src_row.. of the inverse
// row-pass output, moduli src_mod.., scaling constants scale[scale_off..]) converted to n_tgt targets rows[tgt_start..]
struct ConvGroup {
  int src_row, src_mod, n_src, scale_off, tgt_start, n_tgt, pad[2];
};

struct KCtx {  // what kernels need from a context
  void *stream;  // cudaStream_t
  NttGeom geom;
  const ModConst *d_mods;
  const ShoupC *d_tw_fwd;  // [nmod][N] forward twiddles psi^bitrev(k)
  const ShoupC *d_tw_inv;  // [nmod][N] inverse twiddles
  u64 *launches;           // host counter of kernel launches
  int N, nq, np;
  Prof *prof;              // NULL unless profiling is enabled
};

// ---------------------------------------------------------------- launchers (fenc_ntt.cu, fenc_elem.cu); return cudaError_t (0 = ok)
// inverse NTT (both passes).  Source row r of batch b: (items ? items[b].ks_in : src + b*src_bstride) +
// rows[r].src_row*N, read through the Galois gather of items[b].g when gather.  Result: coefficient domain,
// canonical, times scale[r], at dst + b*dst_bstride + rows[r].dst_row*N.
int k_intt(const KCtx &k, const BatchItem *items, const u64 *src, size_t src_bstride, bool gather, u64 *dst,
           size_t dst_bstride, const RowDesc *rows, int n_rows, const ShoupC *scale, int n_batch);
// forward NTT of plain rows: src + b*src_bstride + rows[r].src_row*N -> dst + b*dst_bstride + rows[r].dst_row*N
int k_ntt(const KCtx &k, const u64 *src, size_t src_bstride, u64 *dst, size_t dst_bstride, const RowDesc *rows, int n_rows,
          int n_batch);
// forward pass 1 (column stages) with fused base conversion (ModUp a3 / ModDown's Conv / rescale's mod):
// value = sum_{s < rows[r].aux} y[b][rows[r].src_row + s][.] * bc[rows[r].aux2 + s] (Montgomery constants)
int k_ntt_cols_bconv(const KCtx &k, const u64 *y, size_t y_bstride, const u64 *bc, u64 *tmp, size_t tmp_bstride,
                     const RowDesc *rows, int n_rows, int n_batch, int n_src_rows, int max_terms);
// inverse row pass only (pass A): rows land lazily (< 2q) in dst; the column stages follow in k_convert_cols
int k_intt_rows_only(const KCtx &k, const BatchItem *items, const u64 *src, size_t src_bstride, bool gather, u64 *dst,
                     size_t dst_bstride, const RowDesc *rows, int n_rows, int n_batch, const ShoupC *comb_mul = nullptr);
// (comb_mul != nullptr: merged ModDown + rescale -- rows with aux = 1 read src * comb_mul[mod] + items[b].add{aux2}[mod],
//  all rows come from src, never through the gather)
// fused column kernel (needs N >= 2^12): for every group, the inverse column stages + scaling of its source rows (kept
// in shared memory), then for each target the base conversion and the forward column stages -> tmp rows (lazy).
// Returns -2 when the group does not fit shared memory (the caller falls back to k_intt + k_ntt_cols_bconv).
// forward pass 2 alone, in place on rows[r].dst_row of buf (+ b*bstride): canonical results
int k_ntt_rows_only(const KCtx &k, u64 *buf, size_t bstride, const RowDesc *rows, int n_rows, int n_batch);
// hoisted rotations (R2.7b): acc[b] = sum_j gather_{g_b}(x_j) (*) evk_b,j over the E target rows, x_j[t] = row
// tmp_index[j*E+t] of up + items[b].pad*up_sstride, or items[b].ks_in[t] for the digit's own limbs; Montgomery-reduced
int k_hoisted_keymac(const KCtx &k, const BatchItem *items, int L, int E, int beta, const int *tmp_index, const u64 *up,
                     size_t up_sstride, u64 *acc, size_t acc_bstride, int n_batch, int n_distinct_keys, int n_sources, int n_up);
// whether the fused column kernel can hold a conversion group of n_src limbs (its tiles + the work tiles) in shared memory
bool convert_cols_fits(int logN, int n_src, bool merged);
int k_convert_cols(const KCtx &k, u64 *y, size_t y_bstride, const ConvGroup *groups, int n_groups, int n_src_max,
                   const ShoupC *scale, const u64 *bc, const RowDesc *rows, int n_tgt_total, u64 *tmp, size_t tmp_bstride,
                   int n_batch, int max_terms, const ShoupC *merged_pinv = nullptr, const ShoupC *bc_f64 = nullptr);
// (bc_f64: fp64 pairs {(double) c, (double)(c / t)} of the PLAIN constants, same indexing as bc; used for groups with
//  pad[0] & 2 -- all source moduli fp64 ones -- and fp64 targets)
// (merged_pinv != nullptr: ModDown merged with the rescale; every group carries one extra source row, the inverse-
//  transformed dropped limb of modulus index groups[g].pad[1], and the targets receive V_t P^-1 + (out_l mod t))
// forward pass 2 (row stages) fused with the evaluation-key inner product (a4) over E = L + np target rows.
// tmp_index[j*E + t] = row of tmp holding digit j / target t, or -1 when t lies in digit j (then the row is
// items[b].ks_in[t] itself, read through the Galois gather).  acc[b][c][t][N] canonical.
int k_ntt_rows_keymac(const KCtx &k, const BatchItem *items, int L, int E, int beta, const int *tmp_index, const u64 *tmp,
                      size_t tmp_bstride, u64 *acc, size_t acc_bstride, int n_batch, int n_up, int n_distinct_keys);
// forward pass 2 fused with the divide epilogue (ModDown a5 / rescale a8):
// out[dst_row] = (minuend[aux2] - X) * mul[mod] (+ addend_c[mod] through the gather)
// minuend = from_items ? items[b].sub_in : acc + b*acc_bstride
int k_ntt_rows_divide(const KCtx &k, const BatchItem *items, const u64 *tmp, size_t tmp_bstride, const u64 *acc,
                      size_t acc_bstride, bool minuend_from_items, const ShoupC *mul, const RowDesc *rows, int n_rows,
                      int n_batch, const ShoupC *merged_mul2 = nullptr);
// (merged_mul2 != nullptr: out = ((minuend * merged_mul2[mod] + addend) - X) * mul[mod], the ModDown + rescale merge)
// MAC (a7) over groups of outputs sharing one ciphertext sequence (register tiling, fenc_elem.cu):
// out[out_start+i] = sum_{t<n_terms} ct[ct_start+t] (*) pt[pt_start + i*n_terms + t], i < n_out <= FENC_MAC_GROUP
int k_mac(const KCtx &k, const MacGroup *groups, int n_groups, int max_group, const u64 *const *term_ct, const u64 *const *term_pt,
          u64 *const *outs, int L, int max_lazy, u64 q_max, double alg_bytes);
// scalar MAC of factored weights (R2.9c): a group = up to FENC_SMAC_GROUP outputs sharing one ciphertext sequence and one
// mask segmentation; out[out_start+i] = sum_s M_s (*) ( sum_{t in segment s} k[kidx[k_start + i*n_terms + t]] . ct[ct_start+t] )
#define FENC_SMAC_GROUP 8
struct SmacGroup {
  int n_out, n_terms, ct_start, k_start, out_start, seg_start, n_seg, pad;
};
// kpair: [n_w][L] 16-byte entries: k_mode 0 {k 2^64 mod q, 0}; 1 {(double)(k mod q), (double)((k mod q) / q)};
// 2, 3 {(double) k signed, 0} (fenc_elem.cu: the ciphertext word split in 2 x 25 / 3 x 17 bits; mode 3 groups <= 4 outputs)
int k_smac(const KCtx &k, const SmacGroup *groups, int n_groups, int max_group, const u64 *const *term_ct, const int *kidx,
           const ShoupC *kpair, const int *seg_end, const u64 *const *seg_mask, u64 *const *outs, int L, int k_mode,
           int max_lazy, double alg_bytes, double alg_mulaccs);
// outs[o] = sum of listed [2][L][N] arrays
int k_add_many(const KCtx &k, const u64 *const *term, const int *start, u64 *const *outs, int n_out, int L, int n_terms);
// rows kernels: row r uses modulus row_mod[r] (device array)
// out = x - a * s_mont[mod]   (s_mont: [nmod][N] Montgomery form)
int k_x_minus_as(const KCtx &k, const u64 *a, const u64 *x, const u64 *s_mont, u64 *out, const int *row_mod, int n_rows);
// out[t] = c0[t] + c1[t] * s_mont[t], t < L
int k_dec_combine(const KCtx &k, const u64 *ct, const u64 *s_mont, u64 *out, int L);
// samplers of the counter-based generator (R2.3); coefficient domain, one row per key
int k_sample_uniform(const KCtx &k, const u64 *keys, const int *row_mod, u64 *dst, int n_rows);
// dst[r][n] = (gauss(key)[n] + addend[n]) mod q_{row_mod[r]}; addend may be NULL
int k_sample_gauss(const KCtx &k, u64 key, const i64 *addend, const int *row_mod, u64 *dst, int n_rows);
int k_reduce_signed(const KCtx &k, const i64 *coeffs, const int *row_mod, u64 *dst, int n_rows);
// dst = to ? src 2^64 mod q : src 2^-64 mod q
int k_mont_convert(const KCtx &k, const u64 *src, u64 *dst, const int *row_mod, int n_rows, bool to_mont);
// b = x + f[mod] * sp[mod][gather_g(.)]   (sp Montgomery-form secret; f normal form): evk's "+ f s'" term
int k_add_f_sprime(const KCtx &k, const u64 *x, const u64 *sp_mont, u32 g, const u64 *f, u64 *out, const int *row_mod,
                   int n_rows);
// out[r] = a[r] * b[r] mod q (both normal form, NTT domain)
int k_mul_rows(const KCtx &k, const u64 *a, const u64 *b, u64 *out, const int *row_mod, int n_rows);
// tensor product of n ciphertext pairs: d[b] = (a0 b0, a0 b1 + a1 b0, a1 b1), d: [n][3][L][N]
int k_tensor_product(const KCtx &k, const u64 *const *ina, const u64 *const *inb, u64 *d, int n, int L);
// d[o] = sum_{i < group} (c0 c0, 2 c0 c1, c1 c1) of in[o*group + i]  (R2.12c)
int k_square_sum(const KCtx &k, const u64 *const *in, int group, u64 *d, int n, int L);
// out[b] = in[b] * k (kl: per-limb Montgomery form) or, add_const, c0 += k (kl: per-limb residues)
int k_scalar(const KCtx &k, const u64 *const *in, u64 *const *out, const u64 *kl, int n, int L, bool add_const);
// out[r] = a[r] + b[r] (+ b[r] again when twice)
int k_add_rows(const KCtx &k, const u64 *a, const u64 *b, u64 *out, const int *row_mod, int n_rows, bool twice);

// ---------------------------------------------------------------- host math (fenc_host.cpp)
namespace fh {
u64 mulmod(u64 a, u64 b, u64 q);
u64 powmod(u64 a, u64 e, u64 q);
u64 invmod(u64 a, u64 q);
bool is_prime(u64 n);
bool find_primes(int logN, int bits, int count, std::vector<u64> &out);
u64 find_psi(u64 q, u64 N);
u64 shoup(u64 c, u64 q);    // floor(c 2^64 / q)
u64 to_mont(u64 c, u64 q);  // c 2^64 mod q
u64 neg_qinv(u64 q);        // -q^{-1} mod 2^64
void build_twiddles(u64 q, u64 psi, int logN, ShoupC *fwd, ShoupC *inv);
bool f64_modulus(u64 q, int logN);
bool f64_narrow(u64 q);  // below 2^45: also the base conversions run in fp64
inline u64 double_bits(double d) { u64 b; memcpy(&b, &d, 8); return b; }  // butterflies of this modulus multiply on the FP64 pipe (twiddle tables hold fp64 pairs)
u64 mix64(u64 z);
u64 stream_key(u64 seed, u64 purpose, u64 a, u64 b, u64 c);
void sample_ternary(u64 key, int N, int64_t *out);
// encode / decode (R2.2): fp64 FFT over the 2N-th roots of unity
void encode_slots(int logN, const double *re, const double *im, double scale, int64_t *coeffs);
void decode_coeffs(int logN, const long double *m_over_scale, double *re, double *im);
// Garner mixed-radix lift of [L][N] residues to centred values divided by scale
void crt_centre_scaled(const u64 *q, int L, int N, const u64 *res, long double scale, long double *out);
}  // namespace fh
