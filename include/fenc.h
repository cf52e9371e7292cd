/*
 * fenc.h -- C ABI of libfenc: the B200-native (sm_100a) hot path of FEnc^2 (arxiv/paper_2606_16359):
 * a CKKS homomorphic convolution layer over fragment-encoded ciphertexts.
 *
 * Citations are "PAPER.md:<line>" (the paper) or "DESIGN.md R2.x / A-n" (the readings this build takes
 * where the paper is silent; the paper only names the CKKS primitives).
 *
 * Conventions
 *  - Plain C, no exceptions cross the boundary.  Every function returns fenc_status (0 = OK); outputs are
 *    written only on success.  fenc_last_error(ctx) returns a text for the last failure on that context.
 *  - "host" pointers are ordinary CPU memory owned by the caller; the library copies what it needs before
 *    returning.  "device" pointers are CUDA global memory on the context's device.
 *  - Handles (fenc_ctx, fenc_keys, fenc_pt, fenc_ct, fenc_wts) are opaque, created by the library and
 *    destroyed by the matching *_free (NULL-safe).  A handle must be freed before its context.
 *  - Device memory comes from the allocator callbacks in fenc_params_desc (the Python binding backs them
 *    with torch tensors); if they are NULL the library uses cudaMalloc / cudaFree.
 *  - All GPU work is enqueued on the stream given at init (torch's current stream in the binding) and is
 *    asynchronous; calls that return host-visible data synchronise that stream internally.
 *  - There is NO CPU fallback: without a CUDA device of compute capability 10.x init fails (FENC_ERR_DEVICE).
 *  - Device layout of a ciphertext at L limbs: uint64 [2][L][N], limb-major, NTT ("evaluation") domain,
 *    canonical residues in [0, q_i).  The NTT ordering is private; every export is coefficient domain.
 */
#ifndef FENC_H
#define FENC_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  FENC_OK = 0,
  FENC_ERR_INVALID_ARG = 1,
  FENC_ERR_PARAMS = 2,   /* prime not = 1 mod 2N, not enough primes, P < max digit product, ... */
  FENC_ERR_LAYOUT = 3,   /* S does not divide M, m^2 > N/2, stride does not divide S, ...        */
  FENC_ERR_NO_KEY = 4,   /* rotation amount / relinearisation key not generated                */
  FENC_ERR_LEVEL = 5,    /* not enough limbs left for the requested rescale                    */
  FENC_ERR_MISMATCH = 6, /* operands differ in level / scale / layout                          */
  FENC_ERR_OOM = 7,
  FENC_ERR_DEVICE = 8,
  FENC_ERR_CUDA = 9
} fenc_status;

typedef struct fenc_ctx fenc_ctx;
typedef struct fenc_keys fenc_keys;
typedef struct fenc_pt fenc_pt;
typedef struct fenc_ct fenc_ct;
typedef struct fenc_wts fenc_wts;

/* Parameter set (Table I: N, Q = {q_0..q_L}, Delta; BASELINE.json configs; R1).
 * Ciphertext primes: the n_q largest primes = 1 (mod 2N) below 2^q_bits, descending (q_0 largest);
 * special primes likewise below 2^p_bits.  dlen = ceil(n_q / dnum) limbs per key-switch digit unless
 * dlen_override != 0.  init fails with FENC_ERR_PARAMS when P = prod(p_i) < max digit product unless
 * allow_noisy_ks != 0 (A1: BASELINE config 1's literal dnum=1 is bit-exact-only). */
typedef struct {
  uint32_t log2N;            /* 4..16 */
  uint32_t n_q, q_bits;      /* q_bits <= 60 */
  uint32_t n_p, p_bits;      /* p_bits <= 60 */
  uint32_t dnum;
  uint32_t dlen_override;    /* 0 = derive from dnum */
  uint32_t allow_noisy_ks;
  double log2_scale;         /* default scale Delta = 2^log2_scale */
  const uint64_t *q_override; /* host, n_q entries, or NULL */
  const uint64_t *p_override; /* host, n_p entries, or NULL */
  void *(*dev_alloc)(size_t bytes, void *user); /* returns a device pointer (256-byte aligned) or NULL */
  void (*dev_free)(void *dev_ptr, void *user);
  void *user;
  void *cuda_stream;         /* cudaStream_t; NULL = legacy default stream */
  int device;                /* CUDA device ordinal */
} fenc_params_desc;

/* Convolution shape, Eq. 2 + Algorithm 1. */
typedef struct {
  uint32_t BS, C_in, H, W, C_out, K, stride, pad;
  int32_t depthwise;
  uint32_t S; /* fragment (block) size; 0 = Conv-aware selection (R2.10) */
  uint32_t M; /* square padded frame; 0 = next power of two >= max(H, W) (A4)             */
  /* Segmented layout (R2.11b; the consumer of AAC's output): seg_v = v > 0 means the input
   * AND output ciphertexts hold ch_phys / v segments of v channel positions, segment sg carrying the v channels of batch
   * group bg*seg + sg -- the layout the canonical batch-group compaction (fenc_compress) produces.  Channel diagonal d
   * then wraps inside a segment: two partial sums, rotated by d*cs and (d - v)*cs, masks folded into the weights.
   * 0 (or ch_phys) = the plain layout. */
  uint32_t seg_v;
  /* cap on the samples per ciphertext, B = min(next_pow2(BS), (N/2)/m^2, B_cap); 0 = none ("batch first").
   * With a cap a large batch has several batch groups and several channel positions per ciphertext. */
  uint32_t B_cap;
  /* Baby-step giant-step over the channel diagonals (R2.9d): with bsgs = g > 1 (a power of two
   * dividing ch) a diagonal is d = i g + j and
   *   Y = sum_i Rot( sum_j sum_t Rot(in_t, amt_t + j cs) (*) W'(t, d), i g cs ),  W'(t, d) = Rot(W(t, d), j cs):
   * the baby step is folded into the inner rotation (one rotation of the original input, hoistable), ch/g - 1 outer
   * rotations per output instead of ch - 1.  0 or 1: plain diagonals; FENC_CONV_BSGS_AUTO: the g with the fewest rotations
   * (inner + outer), ties to the smaller g.  On a segmented layout (seg_v = v, g | v) the two parts of diagonal d keep
   * its baby step and rotate by i g cs and (i g - v) cs.  The weight keys stay (.., d, ..); the plaintext of a key is W'. */
  uint32_t bsgs;
} fenc_conv_desc;
#define FENC_CONV_BSGS_AUTO 0xFFFFFFFFu

/* Filled by fenc_layout_plan.  All counts are exact for the operation graph of DESIGN.md R2.9. */
typedef struct {
  uint32_t S, S_out, M, M_out, m, B, ch, cs, G_in, G_out, BG, H_out, W_out;
  uint32_t n_in_ct, n_out_ct, n_inner_rot, n_outer_rot, n_pmult, n_distinct_pt, n_rot_keys;
  uint32_t ch_phys, seg;             /* channel positions of a whole ciphertext; segments (ch_phys = seg * ch)              */
  double S_star_real;                /* (K^2 C_in BS / (alpha C_out))^(1/4): Eq. 8 with BS restored (A5) */
  double paper_rot_count;            /* #Rot as Table IX prints it (A6, A18)           */
  int32_t rot_steps[512];            /* the n_rot_keys distinct rotation amounts the layer needs          */
} fenc_layout;

#define FENC_RELIN_KEY_ID (1ll << 40)

/* ------------------------------------------------------------------ context */
fenc_status fenc_params_init(const fenc_params_desc *desc, fenc_ctx **out);
void fenc_ctx_free(fenc_ctx *ctx);
const char *fenc_last_error(fenc_ctx *ctx);
/* host q[n_q], p[n_p]; dlen_out / beta_max_out may be NULL */
fenc_status fenc_get_primes(fenc_ctx *ctx, uint64_t *q, uint64_t *p, uint32_t *dlen_out, uint32_t *beta_max_out);
fenc_status fenc_sync(fenc_ctx *ctx); /* synchronise the context's stream */

/* ------------------------------------------------------------------ planner (host only) */
fenc_status fenc_layout_plan(fenc_ctx *ctx, const fenc_conv_desc *conv, fenc_layout *out);

/* ------------------------------------------------------------------ keys (R2.3, R2.4)
 * Secret: uniform ternary; errors: discrete Gaussian sigma = 3.2; all from the counter-based generator of
 * DESIGN.md R2.3 keyed by `seed` (evaluated on the device; bit-identical to any host evaluation).
 * rot_steps: host array of n_rot rotation amounts (reduced mod N/2; 0 ignored).  Evaluation keys stay on
 * the device in NTT form. */
fenc_status fenc_keygen(fenc_ctx *ctx, uint64_t seed, const int32_t *rot_steps, size_t n_rot, int want_relin,
                        fenc_keys **out);
void fenc_keys_free(fenc_keys *keys);
/* Key material generated on the HOST and uploaded verbatim (north_star: "all key, encryption and error randomness generated
 * on the host from a seed and uploaded"; R2.4): s[N] the secret's coefficients in {-1,0,1}; for key i
 * (key_ids[i] = rotation amount in [1, N/2) or FENC_RELIN_KEY_ID) b[i] and a[i] are uint64 [beta_max][n_q+n_p][N],
 * coefficient domain, canonical residues -- the format fenc_evk_export writes.  The library only transforms them to its
 * device form (NTT domain, Montgomery); nothing is sampled.  All pointers are host memory, copied before returning. */
typedef struct {
  const int64_t *s;
  size_t n_keys;
  const int64_t *key_ids;
  const uint64_t *const *b;
  const uint64_t *const *a;
} fenc_key_material;
fenc_status fenc_keys_import(fenc_ctx *ctx, const fenc_key_material *mat, fenc_keys **out);
/* host s[N]: the secret's coefficients in {-1,0,1} */
fenc_status fenc_secret_export(fenc_ctx *ctx, const fenc_keys *keys, int64_t *s);
/* key_id = rotation amount in [1, N/2) or FENC_RELIN_KEY_ID.  host b, a: uint64 [beta_max][n_q+n_p][N],
 * coefficient domain, canonical residues (the parity view of a switching key, R2.4). */
fenc_status fenc_evk_export(fenc_ctx *ctx, const fenc_keys *keys, int64_t key_id, uint64_t *b, uint64_t *a);

/* ------------------------------------------------------------------ plaintexts (R2.2, R2.9) */
/* Algorithm 1: gather fragment ciphertext (u, v, group, batch_group) of host x[BS][C][H][W] (fp64) per
 * `layout` (input side of the conv the layout was planned for), then encode at `scale` on n_limbs limbs.
 * scale <= 0 means the context default. */
fenc_status fenc_encode_fragment(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout,
                                 const double *x, uint32_t u, uint32_t v, uint32_t group, uint32_t batch_group,
                                 uint32_t n_limbs, double scale, fenc_pt **out);
/* host re[N/2], im[N/2] (im may be NULL): m_t = round((2 s / N) Re(sum_j z_j conj(zeta_j)^t)) (R2.2) */
fenc_status fenc_encode_slots(fenc_ctx *ctx, const double *re, const double *im, uint32_t n_limbs, double scale,
                              fenc_pt **out);
/* host centred integer coefficients [N]: where bit-exact parity starts (A7) */
fenc_status fenc_pt_from_coeffs(fenc_ctx *ctx, const int64_t *coeffs, uint32_t n_limbs, double scale, fenc_pt **out);
fenc_status fenc_pt_coeffs(fenc_ctx *ctx, const fenc_pt *pt, int64_t *coeffs /* host [N] */);
void fenc_pt_free(fenc_pt *pt);

/* ------------------------------------------------------------------ ciphertexts (R2.5) */
/* Symmetric encryption: c1 = a uniform per limb, c0 = -a s + e + m; randomness from enc_seed (R2.3). */
fenc_status fenc_encrypt(fenc_ctx *ctx, const fenc_keys *keys, const fenc_pt *pt, uint64_t enc_seed, fenc_ct **out);
/* host re[N/2], im[N/2] (im may be NULL): decode(c0 + c1 s) at the ciphertext's scale */
fenc_status fenc_decrypt_slots(fenc_ctx *ctx, const fenc_keys *keys, const fenc_ct *ct, double *re, double *im);
/* decrypt, decode and scatter (inverse of Algorithm 1, output side of `conv`): writes only this ciphertext's
 * entries of host y[BS][C_out][H_out][W_out].  which = 0: input-side layout ([BS][C_in][H][W]), 1: output side. */
fenc_status fenc_decrypt_decode(fenc_ctx *ctx, const fenc_keys *keys, const fenc_ct *ct, const fenc_conv_desc *conv,
                                const fenc_layout *layout, int which, uint32_t u, uint32_t v, uint32_t group,
                                uint32_t batch_group, double *y);
/* host limbs: uint64 [2][L][N], coefficient domain, canonical residues in [0, q_i) */
fenc_status fenc_ct_export(fenc_ctx *ctx, const fenc_ct *ct, uint64_t *limbs);
fenc_status fenc_ct_import(fenc_ctx *ctx, const uint64_t *limbs, uint32_t L, double scale, fenc_ct **out);
/* fenc_ct_import without the host synchronisation: the host->device copy runs on a copy stream of the context's own
 * (overlapping work already enqueued on the context's stream), the NTT follows on the context's stream.  `limbs`
 * (host; page-locked memory for a truly asynchronous copy) stays owned by the caller and must remain valid and
 * unchanged until the next synchronising call on this context returns (fenc_sync, fenc_ct_export, any decrypt).
 * Serving loops use it to upload the next request while the current one computes.  The copies land
 * in a queue of staging buffers that the library grows on demand (while the oldest buffer still waits for its transform)
 * up to 8 GiB of device memory, or FENC_STAGE_MAX_MB MiB if that environment variable is set when the context's first
 * asynchronous import runs; at the cap an upload waits for the transform that frees the oldest buffer. */
fenc_status fenc_ct_import_async(fenc_ctx *ctx, const uint64_t *limbs, uint32_t L, double scale, fenc_ct **out);
/* fenc_ct_export without the host synchronisation: the inverse transform is enqueued on the context's stream, the
 * device->host copy on a second stream of the context's own, so kernels enqueued behind the export do not wait for the
 * bus.  `limbs` (host, page-locked for a truly asynchronous copy; owned by the caller) holds the result once
 * fenc_export_wait or fenc_sync has returned.  fenc_export_wait blocks until every fenc_ct_export_async issued so far has
 * landed; work enqueued on the context after them is not waited for.  The ciphertext may be freed or overwritten right
 * after the call (the transform reads it in stream order).  While in flight an export holds a device buffer of the
 * ciphertext's size. */
fenc_status fenc_ct_export_async(fenc_ctx *ctx, const fenc_ct *ct, uint64_t *limbs);
fenc_status fenc_export_wait(fenc_ctx *ctx);
fenc_status fenc_ct_info(fenc_ctx *ctx, const fenc_ct *ct, uint32_t *L, double *scale, void **device_ptr);
void fenc_ct_free(fenc_ct *ct);

/* ------------------------------------------------------------------ primitives (R2.6-R2.8) */
/* Rot(in[i], steps[i]) for i < n in ONE batched pass (automorphism + hybrid key switch: ModUp, evk inner
 * product, ModDown; Eq. 1).  All inputs must share the level.  steps: host array. */
fenc_status fenc_rotate(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, const int32_t *steps, size_t n,
                        fenc_ct **out);
/* drop the last limb of each input, floor rounding on the canonical representative (A10) */
fenc_status fenc_rescale(fenc_ctx *ctx, fenc_ct *const *in, size_t n, fenc_ct **out);
fenc_status fenc_add(fenc_ctx *ctx, const fenc_ct *a, const fenc_ct *b, fenc_ct **out);
/* out = sum_i in[i] (*) pt[i], one lazy 128-bit accumulation per coefficient (a7); scale multiplies */
fenc_status fenc_pmult_sum(fenc_ctx *ctx, fenc_ct *const *in, fenc_pt *const *pt, size_t n, fenc_ct **out);
/* out[i] = in[i]^2 relinearised and rescaled (a13; R2.12), all n in ONE batched key switch; inputs share the level */
fenc_status fenc_square_relin(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, size_t n, fenc_ct **out);
/* out[i] = a[i] * b[i] relinearised and rescaled (CMult; R2.12); square_relin is the case b = a */
/* Sum of squares with ONE relinearisation (R2.12c; x^2 followed by the 2x2 sum-pool of PAPER.md:284): output o is
 *   rescale( (D0, D1) + KS(D2; relin) ),  (D0, D1, D2) = sum_{i < group} (c0 c0, 2 c0 c1, c1 c1) of in[o*group + i]:
 * the tensor products are added before the key switch, so a pooled output costs one relinearisation instead of `group`.
 * in: n_out*group ciphertexts at one level and scale (host array of handles); out: n_out new ciphertexts at L-1 and
 * scale^2 / q_{L-1}.  group = 1 is fenc_square_relin.  Decrypts to the sum of the squared slot vectors; the limbs
 * differ from the sum of `group` fenc_square_relin results (compare with the oracle's square_sum_relin). */
fenc_status fenc_square_sum_relin(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, size_t n_out, size_t group,
                                  fenc_ct **out);
fenc_status fenc_cmult_relin(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *a, fenc_ct *const *b, size_t n, fenc_ct **out);
/* PMultConst (R2.8): out[i] = in[i] * k for the integer k given by its residues, host k_res[L] with k_res[t] = k mod q_t
 * (the caller rounds c*E exactly, R2.8); the scale is multiplied by scale_factor (= E).  No level is consumed. */
fenc_status fenc_mul_scalar(fenc_ctx *ctx, fenc_ct *const *in, size_t n, const uint64_t *k_res, double scale_factor, fenc_ct **out);
/* out[i] = in[i] + k: the integer k (residues k_res[L]) added to coefficient 0 of c0, i.e. round(scale*c) for a real constant c */
fenc_status fenc_add_const(fenc_ctx *ctx, fenc_ct *const *in, size_t n, const uint64_t *k_res, fenc_ct **out);
/* out[g] = sum_{i < group} in[g*group + i] for g < n_groups: avg-pool by fragment selection (a14; PAPER.md:284;
 * the 1/group^2 factor belongs to the next layer's weights, R2.12).  No rotations, no level consumed. */
fenc_status fenc_sum_groups(fenc_ctx *ctx, fenc_ct *const *in, size_t group, size_t n_groups, fenc_ct **out);

/* 2x2 sum-pool by fragment selection with the fragment order owned by the library (a14; R2.12): in holds
 * n ciphertexts ordered [...][u][v] with S x S fragments per (batch group, channel group), S even; out receives n/4
 * ciphertexts ordered [...][u_o][v_o], out(u_o, v_o) = sum_{a,b in {0,1}} in(2 u_o + a, 2 v_o + b). */
fenc_status fenc_sum_pool(fenc_ctx *ctx, fenc_ct *const *in, size_t n, uint32_t S, fenc_ct **out);
/* x^2 followed by that pool with ONE relinearisation per pooled output (R2.12c): fenc_square_sum_relin over the four
 * fragments of every output, same ordering as fenc_sum_pool. */
fenc_status fenc_square_sum_pool(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, size_t n, uint32_t S, fenc_ct **out);
/* Degree-3 activation a0 + a1 x + a3 x^3 in two levels (a13; R2.12), every step batched over the n
 * inputs (level L, scale s): x2 = Rescale(Relin(x x)); t = Rescale(k3 x) with k3 = round_half_up(a3 q_{L-1});
 * x3 = Rescale(Relin(x2 t)) at scale s3 = s^3 / (q_{L-1} q_{L-2}); u = Rescale(Rescale(k1 x)) with k1 = round_half_up(a1 s^2);
 * out = x3 + u + k0 on coefficient 0 of c0, k0 = round_half_up(a0 s3).  The three integers are rounded exactly by the
 * caller from the exact rational scale (R2.8) and passed as residues: host k3_res[L], k1_res[L], k0_res[L-2];
 * scale_sq = s^2 as a double (bookkeeping of the output scale only).  out: n ciphertexts at L-2. */
fenc_status fenc_poly3(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, size_t n, const uint64_t *k3_res,
                       const uint64_t *k1_res, const uint64_t *k0_res, double scale_sq, fenc_ct **out);

/* ------------------------------------------------------------------ HConv (R2.9) */
/* Number of distinct non-zero weight plaintexts of the layer and their keys (u_o, v_o, g_out, g_in, d, i, j). */
fenc_status fenc_wts_keys(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout, uint32_t *keys7,
                          size_t capacity, size_t *n);
/* Encode every non-zero weight plaintext from host w[C_out][C_in or 1][K][K] at `scale` (<= 0: q_{L-1}, A14). */
fenc_status fenc_conv_weights(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout, const double *w,
                              uint32_t n_limbs, double scale, fenc_wts **out);
/* Same from pre-encoded centred integer coefficients, host coeffs[n][N] in fenc_wts_keys order (A7). */
fenc_status fenc_conv_weights_from_coeffs(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout,
                                          const int64_t *coeffs, size_t n, uint32_t n_limbs, double scale,
                                          fenc_wts **out);
void fenc_wts_free(fenc_wts *w);
/* ---- factored weights for the large-batch case (R2.9c; "Special Case: Large Batch", and the
 * scale split Delta_1 Delta_2 = Delta of PAPER.md:276).  When a ciphertext holds ONE channel (layout ch = 1, or any layer
 * whose weight plaintexts have a single valid channel position) every weight plaintext is a real value v times a 0/1
 * validity mask mu (zero padding, frame padding, stride).  The factored form stores per weight only the integer
 * k = round_half_up(v E1) (one residue per limb) and per DISTINCT mask one plaintext M = encode(mu, E2), E1 E2 = s_w
 * (default s_w = q_{L-1}, E1 = 2^ceil(log2(s_w)/2)), and fenc_hconv evaluates per output and diagonal
 *   P_d = sum_mu M_mu (*) ( sum_{terms t with mask mu} k_t . R_t ):
 * scalar multiply-accumulates of (rotated) input ciphertexts, then one plaintext product per mask.  Same level use and
 * output scale as the plain form; the limbs differ from it (compare with the oracle's hconv_factored).  A layer of C_out x
 * C_in x K^2 weights then needs C_out C_in K^2 L words instead of that many plaintexts of L N words.
 * fenc_wts_factors: mask id of every weight in fenc_wts_keys order (ids in order of first appearance) and the number of
 * distinct masks; FENC_ERR_LAYOUT when some weight plaintext has several valid channel positions.
 * fenc_wts_mask_slots: the 0/1 slot vector of one mask, host slots[N/2]. */
fenc_status fenc_wts_factors(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout, uint32_t *mask_of,
                             size_t capacity, size_t *n, size_t *n_masks);
fenc_status fenc_wts_mask_slots(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout, uint32_t mask_id,
                                double *slots);
/* host w[C_out][C_in or 1][K][K]; scale <= 0: s_w = q_{L-1} (A14) */
fenc_status fenc_conv_weights_factored(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout, const double *w,
                                       uint32_t n_limbs, double scale, fenc_wts **out);
/* the same from integers (A7: parity starts at integer coefficients): host k[n] = the multipliers round_half_up(v E1) in
 * fenc_wts_keys order, host mask_coeffs[n_masks][N] = centred coefficients of the masks encoded at E2, in mask-id order */
fenc_status fenc_conv_weights_factored_from_ints(fenc_ctx *ctx, const fenc_conv_desc *conv, const fenc_layout *layout,
                                                 const int64_t *k, size_t n, const int64_t *mask_coeffs, size_t n_masks,
                                                 uint32_t n_limbs, double E1, double E2, fenc_wts **out);
/* One fragment-encoded conv layer over ALL batch groups.  in: n_in = S^2 G_in BG ciphertexts ordered
 * [bg][g][u][v]; out: n_out = S_out^2 G_out BG ciphertexts ordered [bg][g_out][u_o][v_o].  Inner rotations
 * (batched), MAC, outer rotations (batched), one rescale per output ciphertext when do_rescale != 0 (A13). */
fenc_status fenc_hconv(fenc_ctx *ctx, const fenc_keys *keys, const fenc_conv_desc *conv, const fenc_layout *layout,
                       const fenc_wts *wts, fenc_ct *const *in, size_t n_in, int do_rescale, fenc_ct **out,
                       size_t n_out_capacity, size_t *n_out);

/* ------------------------------------------------------------------ FC by plain diagonals (a15; R2.12)
 * The joint index p = cpos*m^2 + k in [0, P), P = (N/2)/B, is the position inside a ciphertext; input feature
 * <-> (input ct c, p), neuron nu <-> (output ct c', p) with nu = c'*P + p;
 *   out_{c'} = sum_d Rot( sum_c x_c (*) Wd(c',c,d), d*B ),  Wd(c',c,d)[p] = W[nu(c',(p-d) mod P)][feat(c,p)] or 0.
 * Input features: in_C > 0: the S=1 fragment layout of a [BS][in_C][in_H][in_W] tensor in an in_M x in_M frame
 * (PyTorch flatten order feat = channel*H*W + h*W + w); in_C = 0: the output layout of a previous fc (feat = c*P + p).
 * B = min(next_pow2(BS), (N/2)/in_M^2) samples per ciphertext, as in the conv layouts it chains with.
 * Baby-step giant-step ("diagonal-matrix multiplication with BSGS"; R2.12b): with bsgs = g > 1 (a power of
 * two dividing P) a diagonal is d = i g + j and
 *   out_{c'} = sum_i Rot( sum_j sum_c Rot(x_c, j B) (*) W'(c',c,d), i g B ),  W'(c',c,d) = Rot(Wd(c',c,d), j B):
 * (g-1) baby rotations per input ciphertext, shared by every output, and P/g - 1 giant rotations per output ciphertext
 * instead of P - 1.  bsgs = 0 or 1: plain diagonals; FENC_FC_BSGS_AUTO: the g with the fewest rotations
 * n_in_ct (g-1) + n_out_ct (P/g - 1), ties to the smaller g.  The weight calls take the same descriptor (the keys stay
 * (c', c, d); the plaintext of a key is W'). */
#define FENC_FC_BSGS_AUTO 0xFFFFFFFFu
typedef struct {
  uint32_t BS, n_in, n_out;
  uint32_t in_C, in_H, in_W, in_M;
  uint32_t bsgs;
  /* Fragment-encoded embeddings (R2.13, the Transformer extension): BS tokens, a token's
   * embedding split in sub-blocks of S coordinates; coordinate e = p S + u lives in ciphertext u (0 <= u < S) at position
   * p.  frag_in = S > 0: S input ciphertexts per batch group, feat(c, p) = p S + c (needs ceil(n_in / S) <= P and
   * in_C = 0); frag_out = S' > 0: S' output ciphertexts, nu(c', p) = p S' + c'.  X W^T is then the diagonal product above;
   * with n_in = S P it needs P - 1 = n_in / S - 1 rotations per output ciphertext (plain diagonals) instead of n_in - 1.
   * 0: the orders stated above. */
  uint32_t frag_in, frag_out;
} fenc_fc_desc;
typedef struct {
  uint32_t B, P, BG, n_in_ct, n_out_ct, n_rot /* baby + giant */, n_pmult, n_distinct_pt, n_rot_keys, bsgs /* g used */;
  int32_t rot_steps[512];
} fenc_fc_info;
fenc_status fenc_fc_plan(fenc_ctx *ctx, const fenc_fc_desc *fc, fenc_fc_info *out);
/* keys (c_out_ct, c_in_ct, d) of the non-zero weight plaintexts, in the order the weight calls use */
fenc_status fenc_fc_wts_keys(fenc_ctx *ctx, const fenc_fc_desc *fc, uint32_t *keys3, size_t capacity, size_t *n);
/* host w[n_out][n_in] (fp64); scale <= 0: q_{L-1} (A14) */
fenc_status fenc_fc_weights(fenc_ctx *ctx, const fenc_fc_desc *fc, const double *w, uint32_t n_limbs, double scale,
                            fenc_wts **out);
fenc_status fenc_fc_weights_from_coeffs(fenc_ctx *ctx, const fenc_fc_desc *fc, const int64_t *coeffs, size_t n,
                                        uint32_t n_limbs, double scale, fenc_wts **out);
/* Input / output side of a fully connected layer on host arrays (the counterparts of fenc_encode_fragment and
 * fenc_decrypt_decode): slot p B + b of input ciphertext (c, bg) holds x[bg B + b][feat(c, p)], 0 where feat is undefined
 * or the sample index is >= BS.  host x[BS][n_in] (fp64, row-major); scale <= 0: the context default.
 * side = 0 encodes / decodes per the INPUT order (feat), side = 1 per the OUTPUT order (nu) -- the latter to feed a next
 * layer whose input order equals this layer's output order (frag_in' = frag_out), or to read a result. */
fenc_status fenc_fc_encode_input(fenc_ctx *ctx, const fenc_fc_desc *fc, const double *x, uint32_t c, uint32_t batch_group,
                                 uint32_t n_limbs, double scale, fenc_pt **out);
/* decrypt, decode, scatter: writes only this ciphertext's entries of host y[BS][n_out] (side 1) or y[BS][n_in] (side 0) */
fenc_status fenc_fc_decrypt_decode(fenc_ctx *ctx, const fenc_keys *keys, const fenc_ct *ct, const fenc_fc_desc *fc, int side,
                                   uint32_t c, uint32_t batch_group, double *y);
/* in: n_in_ct*BG ciphertexts ordered [bg][c]; out: n_out_ct*BG ordered [bg][c'] */
fenc_status fenc_fc(fenc_ctx *ctx, const fenc_keys *keys, const fenc_fc_desc *fc, const fenc_wts *wts, fenc_ct *const *in,
                    size_t n_in, int do_rescale, fenc_ct **out, size_t n_out_capacity, size_t *n_out);

/* ------------------------------------------------------------------ hoisted inner rotations (R2.7b)
 * The inner rotations of a linear layer (fenc_hconv, fenc_fc) rotate each input ciphertext by several amounts.  With
 * hoisting on, the decomposition of c1 (inverse NTT, ModUp, forward NTT) runs once per input ciphertext and every rotation
 * applies its automorphism to the extended digits: Rot = (sigma_g(c0) + ModDown(sum_j sigma_g(up_j) evk_j.b),
 * ModDown(sum_j sigma_g(up_j) evk_j.a)).  Same keys, same decryption up to key-switch noise of the same size; the limbs
 * differ from the plain form (sigma_g(ModUp_j(c1)) and ModUp_j(sigma_g(c1)) differ by multiples of Q_j), so a run is
 * compared with the oracle's hoisted variant.  Outer rotations, fenc_rotate and fenc_compress are unaffected.
 * Default: off.  Takes effect for the calls that follow. */
fenc_status fenc_set_hoisting(fenc_ctx *ctx, int on);
/* The same form as a primitive: every input (all at one level) rotated by every amount, one decomposition per input.
 * out (capacity n_in * n_steps) receives out[i * n_steps + s] = Rot(in[i], steps[s]); an amount of 0 copies.
 * FENC_ERR_NO_KEY if a rotation key is missing; nothing is written to out on failure. */
fenc_status fenc_rotate_hoisted(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, size_t n_in, const int32_t *steps,
                                size_t n_steps, fenc_ct **out);

/* ------------------------------------------------------------------ AAC compress (R2.11) */
/* out[t] = sum over the terms with term_out[i] == t of Rot(mask (*) in[term_src[i]], term_rot[i]).
 * mask may be NULL (maskless mode, no level consumed); with a mask and do_rescale != 0 this is the paper's
 * split-scale mode (one late rescale).  term_*: host arrays of n_terms entries. */
fenc_status fenc_compress(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, size_t n_in, const fenc_pt *mask,
                          const uint32_t *term_out, const uint32_t *term_src, const int32_t *term_rot, size_t n_terms,
                          int do_rescale, fenc_ct **out, size_t n_out);

/* Repack (R2.11c; "we adapt the pre- or post-processing (rot-mask-add) operations to adjust block
 * size"): the general rot-mask-add with one mask per term,
 *   out[t] = Rescale( sum over the terms i with term_out[i] == t of Rot(masks[i] (*) in[term_src[i]], term_rot[i]) ),
 * terms sharing (output, amount) are summed before their one rotation.  masks: host array of n_terms plaintext handles at
 * the inputs' level, all at one scale (q_{L-1} keeps the ciphertext scale: one level).  It moves a tensor
 * between two layouts (another block size S, another segmentation); the plan is the caller's (oracle/fragment.py
 * repack_plan states the one the tests use).  do_rescale = 0 leaves the sum at scale s_ct * s_mask. */
fenc_status fenc_repack(fenc_ctx *ctx, const fenc_keys *keys, fenc_ct *const *in, size_t n_in, fenc_pt *const *masks,
                        const uint32_t *term_out, const uint32_t *term_src, const int32_t *term_rot, size_t n_terms,
                        int do_rescale, fenc_ct **out, size_t n_out);

/* ------------------------------------------------------------------ allocation-free rescale
 * For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): fenc_rescale (a8; R2.8) with its intermediates in a file-scope device array of FENC_STATIC_SCRATCH_BYTES
 * that every GPU loading the library holds until exit, instead of the context's workspace and descriptor ring.
 * fenc_rescale_static_prepare(ctx, L) is the SET-UP step (it may allocate): builds the tables of level L and resolves the
 * array's device address for the context's device; call it once per (context, level) before the first static call.
 * fenc_rescale_static(ctx, in, out): out := in with its last limb dropped (floor rounding on the canonical representative,
 * A10), bit-identical to fenc_rescale.  `in` is a ciphertext at L >= 2 limbs, `out` an EXISTING ciphertext of the same
 * context at L-1 limbs, owned by the caller (its contents are overwritten, its scale set to in.scale / q_{L-1}); the call
 * makes no cudaMalloc / cudaFree, no allocator callback, and creates no stream or event; work is enqueued on the
 * context's stream.  It needs 256 + (2 + 2(L-1)) * N * 8 bytes of the array: N = 2^16 up to L = 31 (every BASELINE layer
 * configuration: at most 30 limbs), N <= 2^15 at any level this library supports; larger requests fail with FENC_ERR_INVALID_ARG and a message naming both sizes;
 * a level whose tables do not exist yet, a device whose array address has not been resolved (no prepare call yet in this
 * process), or a context with the profiling hooks enabled, fails with FENC_ERR_INVALID_ARG too.
 * Every call on a device shares the array and finds the previous call's contents in it (every word a call reads it has
 * written first, so nothing needs clearing); calls enqueued on one stream are ordered, calls that OVERLAP on the GPU
 * (two contexts or streams on the same device) race -- serialise them. */
#define FENC_STATIC_SCRATCH_BYTES (32u << 20)
fenc_status fenc_rescale_static_prepare(fenc_ctx *ctx, uint32_t L);
fenc_status fenc_rescale_static(fenc_ctx *ctx, const fenc_ct *in, fenc_ct *out);

/* ------------------------------------------------------------------ measurement helpers */
/* Raw batched negacyclic NTT / iNTT (a1) in place on device memory: rows uint64 [n_rows][N]; mod_idx: host
 * array, row r uses modulus mod_idx[r] (0..n_q-1 ciphertext primes, n_q.. special primes). */
fenc_status fenc_ntt_rows(fenc_ctx *ctx, void *device_rows, const int32_t *mod_idx, size_t n_rows, int inverse);
/* Per-kernel-class timing with CUDA events on the context's stream, and the algorithmic bytes each launch moved
 * and the modular butterflies it computed.  Off by default.  ms / launches / alg_bytes /
 * alg_butterflies: host arrays of fenc_profile_kernels() entries. */
fenc_status fenc_profile_enable(fenc_ctx *ctx, int on);
int fenc_profile_kernels(void);
const char *fenc_profile_name(int id);
fenc_status fenc_profile_read(fenc_ctx *ctx, double *ms, uint64_t *launches, double *alg_bytes, double *alg_butterflies,
                              int reset);
/* Measured arithmetic ceilings on this device: dependency-free 32-bit IMAD lane-ops/s, and
 * register-only forward butterflies/s of the library's own butterfly (no memory traffic) -- the integer Shoup butterfly,
 * or, when q_0 is below 2^45 and the context's butterflies run on the FP64 pipe, the faster of that and the fp64 one. */
fenc_status fenc_measure_alu_peak(fenc_ctx *ctx, double *imad_lane_ops_per_s, double *butterflies_per_s);
/* The arithmetic ceiling of the scalar MAC of factored weights (R2.9c): its inner operation in the mode ordinary weights
 * run in (the ciphertext word split in 2 x 25 bits times the small signed multiplier: 2 DFMA per multiply-accumulate plus
 * the shared conversions), registers only, all SMs (q = q_0, below 2^50) -- modular multiply-accumulates per second.
 * For kernel class "smac" the second counter of fenc_profile_read holds multiply-accumulates, not butterflies. */
fenc_status fenc_measure_smac_peak(fenc_ctx *ctx, double *mulaccs_per_s);
/* counters since context creation: kernels launched by this library; optional reset */
uint64_t fenc_launch_count(fenc_ctx *ctx, int reset);
/* bytes currently held through the allocator */
uint64_t fenc_device_bytes(fenc_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* FENC_H */
