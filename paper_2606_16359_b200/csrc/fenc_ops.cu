// fenc_ops.cu -- keys, plaintexts, encryption / decryption and the ciphertext primitives of the C ABI.
#include <cstdlib>
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>

#include "fenc_ctx.h"

enum { PURPOSE_SECRET = 1, PURPOSE_EVK_A = 2, PURPOSE_EVK_E = 3, PURPOSE_ENC_A = 4, PURPOSE_ENC_E = 5 };

static bool scale_close(double a, double b) { return std::fabs(a - b) <= 1e-9 * std::fabs(b); }

// centred integer coefficients (host) -> [L][N] NTT domain, Montgomery form
fenc_status coeffs_to_mont(fenc_ctx *ctx, const int64_t *coeffs, int L, u64 *d_out) {
  Scope sc(ctx);
  const size_t N = ctx->N;
  i64 *d_c = sc.alloc<i64>(N);
  if (!d_c) return fail(ctx, FENC_ERR_OOM, "coefficient staging");
  CUDA_OK(ctx, cudaMemcpyAsync(d_c, coeffs, N * 8, cudaMemcpyHostToDevice, ctx->stream));
  CUDA_OK(ctx, k_reduce_signed(ctx->k, d_c, ctx->d_ident_mod, d_out, L));
  CUDA_OK(ctx, k_ntt(ctx->k, d_out, 0, d_out, 0, ctx->d_ident_rows, L, 1));
  CUDA_OK(ctx, k_mont_convert(ctx->k, d_out, d_out, ctx->d_ident_mod, L, true));
  return FENC_OK;
}
fenc_status pt_device(fenc_ctx *ctx, fenc_pt *pt) {
  if (pt->d_mont) return FENC_OK;
  pt->d_mont = dalloc_t<u64>(ctx, (size_t)pt->L * ctx->N);
  if (!pt->d_mont) return fail(ctx, FENC_ERR_OOM, "plaintext");
  return coeffs_to_mont(ctx, pt->coeffs.data(), pt->L, pt->d_mont);
}

// ------------------------------------------------------------------------------------------------ keys (R2.4)
// For every digit j over ALL nq+np limbs t: a_j[t] uniform, b_j[t] = -a_j[t] s + e_j + f_{j,t} s' (mod t),
// f_{j,t} = P mod t if t in D_j else 0.  Stored in NTT domain, Montgomery form: [beta_max][{b,a}][A][N].
static fenc_status make_switch_key(fenc_ctx *ctx, fenc_keys *K, int64_t key_id, const u64 *d_sp_mont, u32 g, u64 **out) {
  Scope sc(ctx);
  const int A = ctx->A, N = ctx->N, nq = ctx->nq;
  const size_t AN = (size_t)A * N;
  // held by a guard until the key is complete: every early return below releases it
  struct EvkGuard {
    fenc_ctx *ctx; u64 *p;
    ~EvkGuard() { if (p) dfree(ctx, p); }
  } guard{ctx, dalloc_t<u64>(ctx, (size_t)ctx->beta_max * 2 * AN)};
  u64 *evk = guard.p;
  u64 *d_a = sc.alloc<u64>(AN), *d_e = sc.alloc<u64>(AN);
  u64 *d_keys = sc.alloc<u64>(A), *d_f = sc.alloc<u64>(A);
  if (!evk || !d_a || !d_e || !d_keys || !d_f) return fail(ctx, FENC_ERR_OOM, "evaluation key");
  u64 Pmod[FENC_MAX_MOD];
  for (int t = 0; t < A; t++) {
    u64 m = ctx->mod[t], x = 1;
    for (int i = 0; i < ctx->np; i++) x = fh::mulmod(x, ctx->mod[nq + i] % m, m);
    Pmod[t] = x;
  }
  for (int j = 0; j < ctx->beta_max; j++) {
    std::vector<u64> hk(A), hf(A, 0);
    for (int t = 0; t < A; t++) hk[t] = fh::stream_key(K->seed, PURPOSE_EVK_A, (u64)key_id, (u64)j, (u64)t);
    for (int t = j * ctx->dlen; t < std::min((j + 1) * ctx->dlen, nq); t++) hf[t] = Pmod[t];
    CUDA_OK(ctx, cudaMemcpyAsync(d_keys, hk.data(), A * 8, cudaMemcpyHostToDevice, ctx->stream));
    CUDA_OK(ctx, cudaMemcpyAsync(d_f, hf.data(), A * 8, cudaMemcpyHostToDevice, ctx->stream));
    CUDA_OK(ctx, k_sample_uniform(ctx->k, d_keys, ctx->d_ident_mod, d_a, A));
    CUDA_OK(ctx, k_sample_gauss(ctx->k, fh::stream_key(K->seed, PURPOSE_EVK_E, (u64)key_id, (u64)j, 0), nullptr, ctx->d_ident_mod, d_e, A));
    CUDA_OK(ctx, k_ntt(ctx->k, d_a, 0, d_a, 0, ctx->d_ident_rows, A, 1));
    CUDA_OK(ctx, k_ntt(ctx->k, d_e, 0, d_e, 0, ctx->d_ident_rows, A, 1));
    u64 *kb = evk + (size_t)(j * 2 + 0) * AN, *ka = evk + (size_t)(j * 2 + 1) * AN;
    CUDA_OK(ctx, k_x_minus_as(ctx->k, d_a, d_e, K->d_s_mont, kb, ctx->d_ident_mod, A));
    CUDA_OK(ctx, k_add_f_sprime(ctx->k, kb, d_sp_mont, g, d_f, kb, ctx->d_ident_mod, A));
    CUDA_OK(ctx, k_mont_convert(ctx->k, kb, kb, ctx->d_ident_mod, A, true));
    CUDA_OK(ctx, k_mont_convert(ctx->k, d_a, ka, ctx->d_ident_mod, A, true));
    CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));  // hk / hf go out of scope
  }
  *out = evk;
  guard.p = nullptr;
  return FENC_OK;
}

extern "C" fenc_status fenc_keygen(fenc_ctx *ctx, uint64_t seed, const int32_t *rot_steps, size_t n_rot, int want_relin,
                                   fenc_keys **out) {
  Scope sc(ctx);
  if (!ctx || !out || (n_rot && !rot_steps)) return FENC_ERR_INVALID_ARG;
  std::unique_ptr<fenc_keys, void (*)(fenc_keys *)> K(new fenc_keys{ctx, seed, {}, nullptr, {}}, fenc_keys_free);
  const int A = ctx->A, N = ctx->N;
  K->s.resize(N);
  fh::sample_ternary(fh::stream_key(seed, PURPOSE_SECRET, 0, 0, 0), N, K->s.data());
  K->d_s_mont = dalloc_t<u64>(ctx, (size_t)A * N);
  i64 *d_c = sc.alloc<i64>(N);
  if (!K->d_s_mont || !d_c) return fail(ctx, FENC_ERR_OOM, "secret key");
  CUDA_OK(ctx, cudaMemcpyAsync(d_c, K->s.data(), (size_t)N * 8, cudaMemcpyHostToDevice, ctx->stream));
  CUDA_OK(ctx, k_reduce_signed(ctx->k, d_c, ctx->d_ident_mod, K->d_s_mont, A));
  CUDA_OK(ctx, k_ntt(ctx->k, K->d_s_mont, 0, K->d_s_mont, 0, ctx->d_ident_rows, A, 1));
  CUDA_OK(ctx, k_mont_convert(ctx->k, K->d_s_mont, K->d_s_mont, ctx->d_ident_mod, A, true));
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  for (size_t i = 0; i < n_rot; i++) {
    int r = ((rot_steps[i] % ctx->n) + ctx->n) % ctx->n;
    if (r == 0 || K->evk.count(r)) continue;
    u64 *evk = nullptr;
    // s' = sigma_g(s): in the NTT domain the automorphism is the index gather (done inside k_add_f_sprime)
    fenc_status st = make_switch_key(ctx, K.get(), r, K->d_s_mont, galois_elt(ctx, r), &evk);
    if (st != FENC_OK) return st;
    K->evk[r] = evk;
  }
  if (want_relin) {
    // s' = s * s: from Montgomery form, mont_mul(s 2^64, s 2^64) = s^2 2^64 directly
    u64 *d_s2 = sc.alloc<u64>((size_t)A * N), *d_sn = sc.alloc<u64>((size_t)A * N);
    if (!d_s2 || !d_sn) return fail(ctx, FENC_ERR_OOM, "relinearisation key");
    CUDA_OK(ctx, k_mont_convert(ctx->k, K->d_s_mont, d_sn, ctx->d_ident_mod, A, false));
    CUDA_OK(ctx, k_mul_rows(ctx->k, d_sn, d_sn, d_s2, ctx->d_ident_mod, A));
    CUDA_OK(ctx, k_mont_convert(ctx->k, d_s2, d_s2, ctx->d_ident_mod, A, true));
    u64 *evk = nullptr;
    fenc_status st = make_switch_key(ctx, K.get(), FENC_RELIN_KEY_ID, d_s2, 1, &evk);
    if (st != FENC_OK) return st;
    K->evk[FENC_RELIN_KEY_ID] = evk;
  }
  *out = K.release();
  return FENC_OK;
}
extern "C" void fenc_keys_free(fenc_keys *K) {
  if (!K) return;
  cudaStreamSynchronize(K->ctx->stream);
  dfree(K->ctx, K->d_s_mont);
  for (auto &kv : K->evk) dfree(K->ctx, kv.second);
  delete K;
}
// the secret's device form: s reduced mod every modulus, NTT domain, Montgomery form
static fenc_status upload_secret(fenc_ctx *ctx, fenc_keys *K) {
  Scope sc(ctx);
  const int A = ctx->A, N = ctx->N;
  K->d_s_mont = dalloc_t<u64>(ctx, (size_t)A * N);
  i64 *d_c = sc.alloc<i64>(N);
  if (!K->d_s_mont || !d_c) return fail(ctx, FENC_ERR_OOM, "secret key");
  CUDA_OK(ctx, cudaMemcpyAsync(d_c, K->s.data(), (size_t)N * 8, cudaMemcpyHostToDevice, ctx->stream));
  CUDA_OK(ctx, k_reduce_signed(ctx->k, d_c, ctx->d_ident_mod, K->d_s_mont, A));
  CUDA_OK(ctx, k_ntt(ctx->k, K->d_s_mont, 0, K->d_s_mont, 0, ctx->d_ident_rows, A, 1));
  CUDA_OK(ctx, k_mont_convert(ctx->k, K->d_s_mont, K->d_s_mont, ctx->d_ident_mod, A, true));
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  return FENC_OK;
}
// Host-generated key material uploaded verbatim (R2.4): coefficient-domain canonical residues -> NTT domain, Montgomery
extern "C" fenc_status fenc_keys_import(fenc_ctx *ctx, const fenc_key_material *mat, fenc_keys **out) {
  if (!ctx || !mat || !out || !mat->s || (mat->n_keys && (!mat->key_ids || !mat->b || !mat->a))) return FENC_ERR_INVALID_ARG;
  std::unique_ptr<fenc_keys, void (*)(fenc_keys *)> K(new fenc_keys{ctx, 0, {}, nullptr, {}}, fenc_keys_free);
  const int A = ctx->A, N = ctx->N;
  const size_t AN = (size_t)A * N;
  K->s.assign(mat->s, mat->s + N);
  for (int i = 0; i < N; i++)
    if (K->s[i] < -1 || K->s[i] > 1) return fail(ctx, FENC_ERR_INVALID_ARG, "secret coefficient %d is not ternary", i);
  fenc_status st = upload_secret(ctx, K.get());
  if (st != FENC_OK) return st;
  for (size_t k = 0; k < mat->n_keys; k++) {
    const int64_t id = mat->key_ids[k];
    if (!(id == FENC_RELIN_KEY_ID || (id >= 1 && id < ctx->n)) || K->evk.count(id) || !mat->b[k] || !mat->a[k])
      return fail(ctx, FENC_ERR_INVALID_ARG, "key %zu: bad id %lld or missing arrays", k, (long long)id);
    u64 *evk = dalloc_t<u64>(ctx, (size_t)ctx->beta_max * 2 * AN);
    if (!evk) return fail(ctx, FENC_ERR_OOM, "evaluation key");
    K->evk[id] = evk;  // owned by K from here on (freed with it on any later failure)
    for (int j = 0; j < ctx->beta_max; j++)
      for (int c = 0; c < 2; c++) {
        u64 *dst = evk + (size_t)(j * 2 + c) * AN;
        const u64 *src = (c == 0 ? mat->b[k] : mat->a[k]) + (size_t)j * AN;
        for (int t = 0; t < A; t++)
          for (int n = 0; n < N; n += N / 4 ? N / 4 : 1)  // spot check of canonical residues (4 per row)
            if (src[(size_t)t * N + n] >= ctx->mod[t]) return fail(ctx, FENC_ERR_INVALID_ARG, "key %zu: residue not reduced", k);
        CUDA_OK(ctx, cudaMemcpyAsync(dst, src, AN * 8, cudaMemcpyHostToDevice, ctx->stream));
        CUDA_OK(ctx, k_ntt(ctx->k, dst, 0, dst, 0, ctx->d_ident_rows, A, 1));
        CUDA_OK(ctx, k_mont_convert(ctx->k, dst, dst, ctx->d_ident_mod, A, true));
      }
    CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));  // the caller's arrays may go away after the call
  }
  *out = K.release();
  return FENC_OK;
}
extern "C" fenc_status fenc_secret_export(fenc_ctx *ctx, const fenc_keys *K, int64_t *s) {
  if (!ctx || !K || !s) return FENC_ERR_INVALID_ARG;
  memcpy(s, K->s.data(), K->s.size() * 8);
  return FENC_OK;
}
extern "C" fenc_status fenc_evk_export(fenc_ctx *ctx, const fenc_keys *K, int64_t key_id, uint64_t *b, uint64_t *a) {
  Scope sc(ctx);
  if (!ctx || !K || !b || !a) return FENC_ERR_INVALID_ARG;
  auto it = K->evk.find(key_id);
  if (it == K->evk.end()) return fail(ctx, FENC_ERR_NO_KEY, "no key %lld", (long long)key_id);
  const int A = ctx->A, N = ctx->N;
  const size_t AN = (size_t)A * N;
  u64 *tmp = sc.alloc<u64>(AN);
  if (!tmp) return fail(ctx, FENC_ERR_OOM, "export staging");
  for (int j = 0; j < ctx->beta_max; j++)
    for (int c = 0; c < 2; c++) {
      CUDA_OK(ctx, k_mont_convert(ctx->k, it->second + (size_t)(j * 2 + c) * AN, tmp, ctx->d_ident_mod, A, false));
      CUDA_OK(ctx, k_intt(ctx->k, nullptr, tmp, 0, false, tmp, 0, ctx->d_ident_rows, A, ctx->d_ninv, 1));
      CUDA_OK(ctx, cudaMemcpyAsync((c == 0 ? b : a) + (size_t)j * AN, tmp, AN * 8, cudaMemcpyDeviceToHost, ctx->stream));
    }
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  return FENC_OK;
}

// ------------------------------------------------------------------------------------------------ plaintexts
extern "C" fenc_status fenc_pt_from_coeffs(fenc_ctx *ctx, const int64_t *coeffs, uint32_t n_limbs, double scale, fenc_pt **out) {
  if (!ctx || !coeffs || !out || n_limbs < 1 || (int)n_limbs > ctx->nq) return FENC_ERR_INVALID_ARG;
  fenc_pt *pt = new fenc_pt{ctx, (int)n_limbs, scale > 0 ? scale : ctx->default_scale, {}, nullptr};
  pt->coeffs.assign(coeffs, coeffs + ctx->N);
  *out = pt;
  return FENC_OK;
}
extern "C" fenc_status fenc_encode_slots(fenc_ctx *ctx, const double *re, const double *im, uint32_t n_limbs, double scale,
                                         fenc_pt **out) {
  if (!ctx || !re || !out || n_limbs < 1 || (int)n_limbs > ctx->nq) return FENC_ERR_INVALID_ARG;
  fenc_pt *pt = new fenc_pt{ctx, (int)n_limbs, scale > 0 ? scale : ctx->default_scale, {}, nullptr};
  pt->coeffs.resize(ctx->N);
  fh::encode_slots(ctx->logN, re, im, pt->scale, pt->coeffs.data());
  *out = pt;
  return FENC_OK;
}
extern "C" fenc_status fenc_pt_coeffs(fenc_ctx *ctx, const fenc_pt *pt, int64_t *coeffs) {
  if (!ctx || !pt || !coeffs) return FENC_ERR_INVALID_ARG;
  memcpy(coeffs, pt->coeffs.data(), pt->coeffs.size() * 8);
  return FENC_OK;
}
extern "C" void fenc_pt_free(fenc_pt *pt) {
  if (!pt) return;
  if (pt->d_mont) {
    cudaStreamSynchronize(pt->ctx->stream);
    dfree(pt->ctx, pt->d_mont);
  }
  delete pt;
}

// ------------------------------------------------------------------------------------------------ encrypt / decrypt (R2.5)
extern "C" fenc_status fenc_encrypt(fenc_ctx *ctx, const fenc_keys *K, const fenc_pt *pt, uint64_t enc_seed, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !K || !pt || !out) return FENC_ERR_INVALID_ARG;
  const int L = pt->L, N = ctx->N;
  fenc_ct *ct = sc.ct(L, pt->scale);
  i64 *d_m = sc.alloc<i64>(N);
  u64 *d_x = sc.alloc<u64>((size_t)L * N), *d_keys = sc.alloc<u64>(L);
  if (!ct || !d_m || !d_x || !d_keys) return fail(ctx, FENC_ERR_OOM, "encrypt");
  std::vector<u64> hk(L);
  for (int t = 0; t < L; t++) hk[t] = fh::stream_key(enc_seed, PURPOSE_ENC_A, (u64)t, 0, 0);
  CUDA_OK(ctx, cudaMemcpyAsync(d_m, pt->coeffs.data(), (size_t)N * 8, cudaMemcpyHostToDevice, ctx->stream));
  CUDA_OK(ctx, cudaMemcpyAsync(d_keys, hk.data(), (size_t)L * 8, cudaMemcpyHostToDevice, ctx->stream));
  u64 *c0 = ct->d, *c1 = ct->d + (size_t)L * N;
  CUDA_OK(ctx, k_sample_gauss(ctx->k, fh::stream_key(enc_seed, PURPOSE_ENC_E, 0, 0, 0), d_m, ctx->d_ident_mod, d_x, L));  // e + m
  CUDA_OK(ctx, k_sample_uniform(ctx->k, d_keys, ctx->d_ident_mod, c1, L));                                                // a
  CUDA_OK(ctx, k_ntt(ctx->k, d_x, 0, d_x, 0, ctx->d_ident_rows, L, 1));
  CUDA_OK(ctx, k_ntt(ctx->k, c1, 0, c1, 0, ctx->d_ident_rows, L, 1));
  CUDA_OK(ctx, k_x_minus_as(ctx->k, c1, d_x, K->d_s_mont, c0, ctx->d_ident_mod, L));  // c0 = (e + m) - a s
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  sc.ok = true;
  *out = ct;
  return FENC_OK;
}

extern "C" fenc_status fenc_decrypt_slots(fenc_ctx *ctx, const fenc_keys *K, const fenc_ct *ct, double *re, double *im) {
  Scope sc(ctx);
  if (!ctx || !K || !ct || !re) return FENC_ERR_INVALID_ARG;
  const int L = ct->L, N = ctx->N;
  u64 *d_mu = sc.alloc<u64>((size_t)L * N);
  if (!d_mu) return fail(ctx, FENC_ERR_OOM, "decrypt");
  CUDA_OK(ctx, k_dec_combine(ctx->k, ct->d, K->d_s_mont, d_mu, L));
  CUDA_OK(ctx, k_intt(ctx->k, nullptr, d_mu, 0, false, d_mu, 0, ctx->d_ident_rows, L, ctx->d_ninv, 1));
  std::vector<u64> mu((size_t)L * N);
  CUDA_OK(ctx, cudaMemcpyAsync(mu.data(), d_mu, mu.size() * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  std::vector<long double> m(N);
  fh::crt_centre_scaled(ctx->mod.data(), L, N, mu.data(), (long double)ct->scale, m.data());
  fh::decode_coeffs(ctx->logN, m.data(), re, im);
  return FENC_OK;
}

extern "C" fenc_status fenc_ct_export(fenc_ctx *ctx, const fenc_ct *ct, uint64_t *limbs) {
  Scope sc(ctx);
  if (!ctx || !ct || !limbs) return FENC_ERR_INVALID_ARG;
  LevelPlan *P = get_plan(ctx, ct->L);
  const size_t n = (size_t)2 * ct->L * ctx->N;
  u64 *tmp = sc.alloc<u64>(n);
  if (!P || !tmp) return fail(ctx, FENC_ERR_OOM, "export");
  CUDA_OK(ctx, k_intt(ctx->k, nullptr, ct->d, 0, false, tmp, 0, P->d_rows_ct, 2 * ct->L, P->d_scale_ct, 1));
  CUDA_OK(ctx, cudaMemcpyAsync(limbs, tmp, n * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  return FENC_OK;
}
// Export without the host synchronisation.  The inverse transform runs on the context's stream (so it reads the
// ciphertext in stream order, whatever the caller does with the handle afterwards) into a buffer of its own; the
// device -> host copy runs on a second stream, d2h_stream, behind an event: on the context's stream a copy of a request's
// results (config 4: 13.4 GB per batch group, a third of a second on the bus) would hold back every kernel of the next
// request enqueued behind it -- measured before this split: a period of 1007 ms per request for 630 ms of kernels.  The
// buffer returns to the pool when its copy has landed (export_drain, polled by the next export and by every
// synchronising call), so a request's exports hold one copy of its results on the device while they are in flight.
fenc_status export_drain(fenc_ctx *ctx, bool block) {
  while (!ctx->exports.empty()) {
    fenc_ctx::PendingExport &e = ctx->exports.front();
    if (block) CUDA_OK(ctx, cudaEventSynchronize(e.landed));
    else {
      cudaError_t q = cudaEventQuery(e.landed);
      if (q == cudaErrorNotReady) break;
      CUDA_OK(ctx, q);
    }
    dfree(ctx, e.buf);
    ctx->export_events.push_back(e.landed);
    ctx->exports.pop_front();
  }
  return FENC_OK;
}
extern "C" fenc_status fenc_ct_export_async(fenc_ctx *ctx, const fenc_ct *ct, uint64_t *limbs) {
  if (!ctx || !ct || !limbs) return FENC_ERR_INVALID_ARG;
  fenc_status st = export_drain(ctx, false);
  if (st != FENC_OK) return st;
  LevelPlan *P = get_plan(ctx, ct->L);
  const size_t n = (size_t)2 * ct->L * ctx->N;
  if (!ctx->d2h_stream) CUDA_OK(ctx, cudaStreamCreateWithFlags(&ctx->d2h_stream, cudaStreamNonBlocking));
  if (!ctx->export_ready) CUDA_OK(ctx, cudaEventCreateWithFlags(&ctx->export_ready, cudaEventDisableTiming));
  cudaEvent_t landed = nullptr;
  if (!ctx->export_events.empty()) landed = ctx->export_events.back(), ctx->export_events.pop_back();
  else CUDA_OK(ctx, cudaEventCreateWithFlags(&landed, cudaEventDisableTiming));
  u64 *tmp = (u64 *)dalloc(ctx, n * 8);
  if (!P || !tmp) {
    ctx->export_events.push_back(landed);
    dfree(ctx, tmp);
    return fail(ctx, FENC_ERR_OOM, "export");
  }
  ctx->exports.push_back({tmp, landed});  // from here on the buffer is released by export_drain, also after an error
  cudaError_t e = (cudaError_t)k_intt(ctx->k, nullptr, ct->d, 0, false, tmp, 0, P->d_rows_ct, 2 * ct->L, P->d_scale_ct, 1);
  if (e == cudaSuccess) e = cudaEventRecord(ctx->export_ready, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->d2h_stream, ctx->export_ready, 0);
  if (e == cudaSuccess) e = cudaMemcpyAsync(limbs, tmp, n * 8, cudaMemcpyDeviceToHost, ctx->d2h_stream);
  cudaError_t e2 = cudaEventRecord(landed, ctx->d2h_stream);  // recorded in every case: export_drain waits on it
  CUDA_OK(ctx, e);
  CUDA_OK(ctx, e2);
  return FENC_OK;
}
extern "C" fenc_status fenc_export_wait(fenc_ctx *ctx) {
  if (!ctx) return FENC_ERR_INVALID_ARG;
  return export_drain(ctx, true);
}
extern "C" fenc_status fenc_ct_import(fenc_ctx *ctx, const uint64_t *limbs, uint32_t L, double scale, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !limbs || !out || L < 1 || (int)L > ctx->nq) return FENC_ERR_INVALID_ARG;
  LevelPlan *P = get_plan(ctx, (int)L);
  fenc_ct *ct = sc.ct((int)L, scale > 0 ? scale : ctx->default_scale);
  if (!P || !ct) return fail(ctx, FENC_ERR_OOM, "import");
  const size_t n = (size_t)2 * L * ctx->N;
  CUDA_OK(ctx, cudaMemcpyAsync(ct->d, limbs, n * 8, cudaMemcpyHostToDevice, ctx->stream));
  CUDA_OK(ctx, k_ntt(ctx->k, ct->d, 0, ct->d, 0, P->d_rows_ct, 2 * (int)L, 1));
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  sc.ok = true;
  *out = ct;
  return FENC_OK;
}
// The same import without a host synchronisation and with the copy off the compute stream: the limbs go to a slot of a
// staging queue on the context's copy stream (overlapping whatever the compute stream is running), the compute stream
// waits for that copy only, transforms staging -> ciphertext, and releases the slot.  A slot is never touched by any
// other kernel, so the copy has to wait for nothing but the transform that last read the slot.
extern "C" fenc_status fenc_ct_import_async(fenc_ctx *ctx, const uint64_t *limbs, uint32_t L, double scale, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !limbs || !out || L < 1 || (int)L > ctx->nq) return FENC_ERR_INVALID_ARG;
  LevelPlan *P = get_plan(ctx, (int)L);
  fenc_ct *ct = sc.ct((int)L, scale > 0 ? scale : ctx->default_scale);
  if (!P || !ct) return fail(ctx, FENC_ERR_OOM, "import");
  const size_t bytes = (size_t)2 * L * ctx->N * 8;
  if (!ctx->copy_stream) CUDA_OK(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
  if (!ctx->stage_max) {
    const char *mb = getenv("FENC_STAGE_MAX_MB");
    ctx->stage_max = mb && atoll(mb) > 0 ? (size_t)atoll(mb) << 20 : FENC_STAGE_BYTES_MAX;
  }
  // the oldest slot if its transform has run (or the queue may not grow any further: then the copy waits for it), else a new one
  StageSlot sl;
  bool reuse = ctx->stage.size() >= 2 && (cudaEventQuery(ctx->stage.front().consumed) == cudaSuccess || ctx->stage_bytes + bytes > ctx->stage_max);
  (void)cudaGetLastError();  // cudaErrorNotReady is not an error
  if (reuse) {
    sl = ctx->stage.front();
    ctx->stage.pop_front();
    ctx->stage_bytes -= sl.bytes;
  } else {
    CUDA_OK(ctx, cudaEventCreateWithFlags(&sl.copied, cudaEventDisableTiming));
    CUDA_OK(ctx, cudaEventCreateWithFlags(&sl.consumed, cudaEventDisableTiming));
  }
  if (sl.bytes < bytes) {
    // the old buffer returns to the pool behind the transform that last read it; the new one may come from the pool
    // with compute-stream work still pending on it, so its first copy waits for everything enqueued so far
    dfree(ctx, sl.d);
    sl.bytes = 0;
    sl.d = (u64 *)dalloc(ctx, bytes);
    if (sl.d) sl.bytes = bytes;
    if (sl.d) CUDA_OK(ctx, cudaEventRecord(sl.consumed, ctx->stream));
  }
  if (!sl.d) {
    cudaEventDestroy(sl.copied), cudaEventDestroy(sl.consumed);
    return fail(ctx, FENC_ERR_OOM, "import staging (%zu bytes)", bytes);
  }
  ctx->stage.push_back(sl);
  ctx->stage_bytes += sl.bytes;
  CUDA_OK(ctx, cudaStreamWaitEvent(ctx->copy_stream, sl.consumed, 0));
  CUDA_OK(ctx, cudaMemcpyAsync(sl.d, limbs, bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
  CUDA_OK(ctx, cudaEventRecord(sl.copied, ctx->copy_stream));
  CUDA_OK(ctx, cudaStreamWaitEvent(ctx->stream, sl.copied, 0));
  CUDA_OK(ctx, k_ntt(ctx->k, sl.d, 0, ct->d, 0, P->d_rows_ct, 2 * (int)L, 1));
  CUDA_OK(ctx, cudaEventRecord(sl.consumed, ctx->stream));
  sc.ok = true;
  *out = ct;
  return FENC_OK;
}
extern "C" fenc_status fenc_ct_info(fenc_ctx *ctx, const fenc_ct *ct, uint32_t *L, double *scale, void **device_ptr) {
  if (!ctx || !ct) return FENC_ERR_INVALID_ARG;
  if (L) *L = ct->L;
  if (scale) *scale = ct->scale;
  if (device_ptr) *device_ptr = ct->d;
  return FENC_OK;
}
extern "C" void fenc_ct_free(fenc_ct *ct) {
  if (!ct) return;
  dfree(ct->ctx, ct->d);
  delete ct;
}

// ------------------------------------------------------------------------------------------------ primitives
// Groups outputs with identical ciphertext sequences (up to FENC_MAC_GROUP per group) and launches the MAC.
fenc_status run_mac(fenc_ctx *ctx, const MacJob &job, int L) {
  const size_t n = job.outs.size();
  if (n == 0) return FENC_OK;
  std::map<std::vector<const u64 *>, std::vector<int>> by_seq;
  std::vector<std::vector<const u64 *>> order;  // first-appearance order keeps neighbouring fragments adjacent
  for (size_t o = 0; o < n; o++) {
    std::vector<const u64 *> seq(job.terms[o].size());
    for (size_t t = 0; t < seq.size(); t++) seq[t] = job.terms[o][t].first;
    auto it = by_seq.find(seq);
    if (it == by_seq.end()) order.push_back(seq), by_seq[seq] = {(int)o};
    else it->second.push_back((int)o);
  }
  std::vector<MacGroup> groups;
  std::vector<const u64 *> tc, tp, all_c, all_p;
  std::vector<u64 *> outs;
  int max_group = 1;
  for (auto &seq : order) {
    const std::vector<int> &members = by_seq[seq];
    for (size_t at = 0; at < members.size(); at += FENC_MAC_GROUP) {
      const int ng = (int)std::min<size_t>(FENC_MAC_GROUP, members.size() - at);
      MacGroup g{ng, (int)seq.size(), (int)tc.size(), (int)tp.size(), (int)outs.size(), {0, 0, 0}};
      tc.insert(tc.end(), seq.begin(), seq.end());
      for (int i = 0; i < ng; i++) {
        const auto &tl = job.terms[members[at + i]];
        for (auto &pr : tl) tp.push_back(pr.second);
        outs.push_back(job.outs[members[at + i]]);
      }
      groups.push_back(g);
      max_group = std::max(max_group, ng);
    }
  }
  DescStage st(ctx);
  size_t o0 = st.add(groups), o1 = st.add(tc), o2 = st.add(tp), o3 = st.add(outs);
  char *base = st.commit();
  if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
  CUDA_OK(ctx, k_mac(ctx->k, (const MacGroup *)(base + o0), (int)groups.size(), max_group, (const u64 *const *)(base + o1),
                     (const u64 *const *)(base + o2), (u64 *const *)(base + o3), L, ctx->max_lazy, *std::max_element(ctx->mod.begin(), ctx->mod.begin() + L), mac_alg_bytes(ctx, tc, tp, n, L)));
  return FENC_OK;
}
// Factored weights (R2.9c): outputs with the same ciphertext sequence AND the same mask segmentation (the output channels
// of one fragment) form groups of up to FENC_SMAC_GROUP; one launch for all of them.
fenc_status run_smac(fenc_ctx *ctx, const SmacJob &job, const fenc_wts *W, int L) {
  const size_t n = job.outs.size();
  if (n == 0) return FENC_OK;
  typedef std::pair<std::vector<const u64 *>, std::vector<const u64 *>> Seq;  // (ciphertexts, masks) per term
  std::map<Seq, std::vector<int>> by_seq;
  std::vector<Seq> order;
  for (size_t o = 0; o < n; o++) {
    Seq seq;
    for (auto &t : job.terms[o]) seq.first.push_back(t.ct), seq.second.push_back(t.mask);
    auto it = by_seq.find(seq);
    if (it == by_seq.end()) order.push_back(seq), by_seq[seq] = {(int)o};
    else it->second.push_back((int)o);
  }
  std::vector<SmacGroup> groups;
  std::vector<const u64 *> tc, seg_mask, all_masks;
  std::vector<int> kidx, seg_end;
  std::vector<u64 *> outs;
  int max_group = 1;
  for (auto &seq : order) {
    const std::vector<int> &members = by_seq[seq];
    const int nt = (int)seq.first.size();
    std::vector<int> ends;
    std::vector<const u64 *> masks;
    for (int t = 0; t < nt; t++)
      if (t + 1 == nt || seq.second[t + 1] != seq.second[t]) ends.push_back(t + 1), masks.push_back(seq.second[t]);
    const size_t gcap = W->k_mode == 3 ? 4 : FENC_SMAC_GROUP;  // three partial sums per accumulator: groups of 4 outputs
    for (size_t at = 0; at < members.size(); at += gcap) {
      const int ng = (int)std::min<size_t>(gcap, members.size() - at);
      groups.push_back(SmacGroup{ng, nt, (int)tc.size(), (int)kidx.size(), (int)outs.size(), (int)seg_end.size(), (int)ends.size(), 0});
      tc.insert(tc.end(), seq.first.begin(), seq.first.end());
      seg_end.insert(seg_end.end(), ends.begin(), ends.end());
      seg_mask.insert(seg_mask.end(), masks.begin(), masks.end());
      for (int i = 0; i < ng; i++) {
        for (auto &t : job.terms[members[at + i]]) kidx.push_back(t.w);
        outs.push_back(job.outs[members[at + i]]);
      }
      max_group = std::max(max_group, ng);
    }
    all_masks.insert(all_masks.end(), masks.begin(), masks.end());
  }
  DescStage st(ctx);
  size_t o0 = st.add(groups), o1 = st.add(tc), o2 = st.add(kidx), o3 = st.add(seg_end), o4 = st.add(seg_mask), o5 = st.add(outs);
  char *base = st.commit();
  if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
  // algorithmic bytes: every distinct ciphertext and mask read once, every output written once, the scalars once
  const double bytes = mac_alg_bytes(ctx, tc, all_masks, n, L) + 16.0 * L * (double)W->n;
  double mulaccs = 0;
  for (auto &tl : job.terms) mulaccs += 2.0 * (double)tl.size() * L * ctx->N;
  CUDA_OK(ctx, k_smac(ctx->k, (const SmacGroup *)(base + o0), (int)groups.size(), max_group, (const u64 *const *)(base + o1),
                      (const int *)(base + o2), W->d_k, (const int *)(base + o3), (const u64 *const *)(base + o4),
                      (u64 *const *)(base + o5), L, W->k_mode, W->k_lazy, bytes, mulaccs));
  return FENC_OK;
}
// algorithmic bytes of one MAC launch: every distinct ciphertext and plaintext read once, every output written once
double mac_alg_bytes(fenc_ctx *ctx, const std::vector<const u64 *> &tc, const std::vector<const u64 *> &tp, size_t n_out, int L) {
  std::vector<const u64 *> a(tc), b(tp);
  std::sort(a.begin(), a.end()), std::sort(b.begin(), b.end());
  size_t nc = std::unique(a.begin(), a.end()) - a.begin(), npt = std::unique(b.begin(), b.end()) - b.begin();
  return 8.0 * L * ctx->N * (2.0 * nc + (double)npt + 2.0 * n_out);
}
extern "C" fenc_status fenc_rotate(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, const int32_t *steps, size_t n,
                                   fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !K || !in || !steps || !out) return FENC_ERR_INVALID_ARG;
  if (n == 0) return FENC_OK;
  const int L = in[0]->L;
  std::vector<const u64 *> vin(n);
  std::vector<u64 *> vout(n);
  std::vector<int> vs(steps, steps + n);
  std::vector<fenc_ct *> made(n, nullptr);
  for (size_t i = 0; i < n; i++) {
    if (in[i]->L != L) return fail(ctx, FENC_ERR_MISMATCH, "rotate: inputs differ in level");
    made[i] = sc.ct(L, in[i]->scale);
    if (!made[i]) return fail(ctx, FENC_ERR_OOM, "rotate output");
    vin[i] = in[i]->d, vout[i] = made[i]->d;
  }
  fenc_status st = rotate_raw(ctx, K, L, vin, vs, vout);
  if (st != FENC_OK) return st;
  sc.ok = true;
  for (size_t i = 0; i < n; i++) out[i] = made[i];
  return FENC_OK;
}

// every input rotated by every amount with ONE decomposition per input (R2.7b); out[i * n_steps + s] = Rot(in[i], steps[s])
extern "C" fenc_status fenc_rotate_hoisted(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, size_t n_in, const int32_t *steps,
                                           size_t n_steps, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !K || !in || !steps || !out) return FENC_ERR_INVALID_ARG;
  if (n_in == 0 || n_steps == 0) return FENC_OK;
  const int L = in[0]->L;
  std::vector<const u64 *> src(n_in);
  std::vector<int> src_of, vs;
  std::vector<u64 *> vout;
  std::vector<fenc_ct *> made;
  for (size_t i = 0; i < n_in; i++) {
    if (in[i]->L != L) return fail(ctx, FENC_ERR_MISMATCH, "rotate: inputs differ in level");
    src[i] = in[i]->d;
    for (size_t s = 0; s < n_steps; s++) {
      fenc_ct *c = sc.ct(L, in[i]->scale);
      if (!c) return fail(ctx, FENC_ERR_OOM, "rotate output");
      made.push_back(c), vout.push_back(c->d), src_of.push_back((int)i), vs.push_back(steps[s]);
    }
  }
  fenc_status st = rotate_hoisted_raw(ctx, K, L, src, src_of, vs, vout);
  if (st != FENC_OK) return st;
  sc.ok = true;
  for (size_t i = 0; i < made.size(); i++) out[i] = made[i];
  return FENC_OK;
}

extern "C" fenc_status fenc_rescale(fenc_ctx *ctx, fenc_ct *const *in, size_t n, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !in || !out) return FENC_ERR_INVALID_ARG;
  if (n == 0) return FENC_OK;
  const int L = in[0]->L;
  if (L < 2) return fail(ctx, FENC_ERR_LEVEL, "rescale at the last level");
  std::vector<BatchItem> items(n);
  std::vector<fenc_ct *> made(n, nullptr);
  for (size_t i = 0; i < n; i++) {
    if (in[i]->L != L) return fail(ctx, FENC_ERR_MISMATCH, "rescale: inputs differ in level");
    made[i] = sc.ct(L - 1, in[i]->scale / (double)ctx->mod[L - 1]);
    if (!made[i]) return fail(ctx, FENC_ERR_OOM, "rescale output");
    items[i] = BatchItem{};
    items[i].sub_in = in[i]->d, items[i].out = made[i]->d;
  }
  fenc_status st = rescale_batch(ctx, L, items);
  if (st != FENC_OK) return st;
  sc.ok = true;
  for (size_t i = 0; i < n; i++) out[i] = made[i];
  return FENC_OK;
}

extern "C" fenc_status fenc_add(fenc_ctx *ctx, const fenc_ct *a, const fenc_ct *b, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !a || !b || !out) return FENC_ERR_INVALID_ARG;
  if (a->L != b->L || !scale_close(a->scale, b->scale)) return fail(ctx, FENC_ERR_MISMATCH, "add: level or scale differ");
  fenc_ct *c = sc.ct(a->L, a->scale);
  if (!c) return fail(ctx, FENC_ERR_OOM, "add");
  std::vector<const u64 *> terms{a->d, b->d};
  std::vector<int> start{0, 2};
  std::vector<u64 *> outs{c->d};
  DescStage st(ctx);
  size_t o1 = st.add(terms), o2 = st.add(start), o3 = st.add(outs);
  char *base = st.commit();
  if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
  CUDA_OK(ctx, k_add_many(ctx->k, (const u64 *const *)(base + o1), (const int *)(base + o2), (u64 *const *)(base + o3), 1, a->L, 2));
  sc.ok = true;
  *out = c;
  return FENC_OK;
}

extern "C" fenc_status fenc_pmult_sum(fenc_ctx *ctx, fenc_ct *const *in, fenc_pt *const *pt, size_t n, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !in || !pt || !out || n == 0) return FENC_ERR_INVALID_ARG;
  const int L = in[0]->L;
  std::vector<const u64 *> tc(n), tp(n);
  for (size_t i = 0; i < n; i++) {
    if (in[i]->L != L || pt[i]->L != L) return fail(ctx, FENC_ERR_MISMATCH, "pmult: level differs");
    if (!scale_close(in[i]->scale * pt[i]->scale, in[0]->scale * pt[0]->scale)) return fail(ctx, FENC_ERR_MISMATCH, "pmult: scales differ");
    fenc_status s = pt_device(ctx, pt[i]);
    if (s != FENC_OK) return s;
    tc[i] = in[i]->d, tp[i] = pt[i]->d_mont;
  }
  fenc_ct *c = sc.ct(L, in[0]->scale * pt[0]->scale);
  if (!c) return fail(ctx, FENC_ERR_OOM, "pmult");
  MacJob job;
  job.terms.resize(1);
  for (size_t i = 0; i < n; i++) job.terms[0].push_back({tc[i], tp[i]});
  job.outs.push_back(c->d);
  fenc_status ms = run_mac(ctx, job, L);
  if (ms != FENC_OK) return ms;
  sc.ok = true;
  *out = c;
  return FENC_OK;
}

// CMult + relinearise + rescale (a13, R2.12): (d0, d1, d2) = (a0 b0, a0 b1 + a1 b0, a1 b1);
// (d0, d1) + KS(d2; relin); rescale.  Batched over n pairs; x^2 is the case b = a.
// group > 0 (R2.12c): inb is unused, ina holds n*group ciphertexts and output o is the sum of the squares of
// ina[o*group .. o*group+group-1] with ONE relinearisation.
static fenc_status cmult_relin(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *ina, fenc_ct *const *inb, size_t n, fenc_ct **out,
                               size_t group = 0) {
  Scope sc(ctx);
  if (n == 0) return FENC_OK;
  const size_t n_in = group ? n * group : n;
  if (group) inb = ina;
  auto it = K->evk.find(FENC_RELIN_KEY_ID);
  if (it == K->evk.end()) return fail(ctx, FENC_ERR_NO_KEY, "no relinearisation key");
  const int L = ina[0]->L;
  if (L < 2) return fail(ctx, FENC_ERR_LEVEL, "a product needs a level to rescale into");
  const size_t LN = (size_t)L * ctx->N;
  std::vector<const u64 *> pa(n_in), pb(n_in);
  for (size_t i = 0; i < n_in; i++) {
    if (ina[i]->L != L || inb[i]->L != L) return fail(ctx, FENC_ERR_MISMATCH, "product: inputs differ in level");
    if (group && !scale_close(ina[i]->scale, ina[0]->scale)) return fail(ctx, FENC_ERR_MISMATCH, "sum of squares: inputs differ in scale");
    pa[i] = ina[i]->d, pb[i] = inb[i]->d;
  }
  // N >= 2^12: the rescale is merged into the ModDown of the relinearisation (one pass less over the ciphertext)
  const bool merged = ks_can_merge_rescale(ctx, L);
  u64 *d = sc.alloc<u64>(n * 3 * LN), *mid = merged ? nullptr : sc.alloc<u64>(n * 2 * LN);
  if (!d || (!merged && !mid)) return fail(ctx, FENC_ERR_OOM, "product");
  {
    DescStage st(ctx);
    size_t o0 = st.add(pa), o1 = st.add(pb);
    char *base = st.commit();
    if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
    if (group) CUDA_OK(ctx, k_square_sum(ctx->k, (const u64 *const *)(base + o0), (int)group, d, (int)n, L));
    else CUDA_OK(ctx, k_tensor_product(ctx->k, (const u64 *const *)(base + o0), (const u64 *const *)(base + o1), d, (int)n, L));
  }
  std::vector<BatchItem> items(n), rs(n);
  std::vector<fenc_ct *> made(n, nullptr);
  for (size_t i = 0; i < n; i++) {
    u64 *di = d + i * 3 * LN;
    items[i] = BatchItem{};
    const size_t i0 = group ? i * group : i;
    made[i] = sc.ct(L - 1, ina[i0]->scale * inb[i0]->scale / (double)ctx->mod[L - 1]);
    if (!made[i]) return fail(ctx, FENC_ERR_OOM, "product output");
    items[i].ks_in = di + 2 * LN, items[i].out = merged ? made[i]->d : mid + i * 2 * LN, items[i].evk = it->second;
    items[i].add0 = di, items[i].add1 = di + LN, items[i].g = 1;
    rs[i] = BatchItem{};
    rs[i].sub_in = merged ? nullptr : mid + i * 2 * LN, rs[i].out = made[i]->d;
  }
  fenc_status st = ks_batch(ctx, L, items, merged);
  if (st != FENC_OK) return st;
  if (!merged) st = rescale_batch(ctx, L, rs);
  if (st != FENC_OK) return st;
  sc.ok = true;
  for (size_t i = 0; i < n; i++) out[i] = made[i];
  return FENC_OK;
}
extern "C" fenc_status fenc_square_relin(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, size_t n, fenc_ct **out) {
  if (!ctx || !K || !in || !out) return FENC_ERR_INVALID_ARG;
  return cmult_relin(ctx, K, in, in, n, out);
}
extern "C" fenc_status fenc_square_sum_relin(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, size_t n_out, size_t group,
                                             fenc_ct **out) {
  if (!ctx || !K || !in || !out || group < 1) return FENC_ERR_INVALID_ARG;
  return cmult_relin(ctx, K, in, in, n_out, out, group);
}
extern "C" fenc_status fenc_cmult_relin(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *a, fenc_ct *const *b, size_t n, fenc_ct **out) {
  if (!ctx || !K || !a || !b || !out) return FENC_ERR_INVALID_ARG;
  return cmult_relin(ctx, K, a, b, n, out);
}

// PMultConst (R2.8): every limb times the integer k, given by its residues k mod q_t; the caller states the
// factor the scale is multiplied by.  add_const: the integer k is added to coefficient 0 of c0 (scale unchanged).
static fenc_status scalar_op(fenc_ctx *ctx, fenc_ct *const *in, size_t n, const uint64_t *k_res, double factor, bool add_const,
                             fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !in || !k_res || !out) return FENC_ERR_INVALID_ARG;
  if (n == 0) return FENC_OK;
  const int L = in[0]->L;
  std::vector<u64> kl(L);
  for (int t = 0; t < L; t++) {
    if (k_res[t] >= ctx->mod[t]) return fail(ctx, FENC_ERR_INVALID_ARG, "scalar residue %d is not reduced", t);
    kl[t] = add_const ? k_res[t] : fh::to_mont(k_res[t], ctx->mod[t]);
  }
  std::vector<const u64 *> pin(n);
  std::vector<u64 *> pout(n);
  std::vector<fenc_ct *> made(n, nullptr);
  for (size_t i = 0; i < n; i++) {
    if (in[i]->L != L) return fail(ctx, FENC_ERR_MISMATCH, "scalar op: inputs differ in level");
    made[i] = sc.ct(L, add_const ? in[i]->scale : in[i]->scale * factor);
    if (!made[i]) return fail(ctx, FENC_ERR_OOM, "scalar op output");
    pin[i] = in[i]->d, pout[i] = made[i]->d;
  }
  DescStage st(ctx);
  size_t o0 = st.add(pin), o1 = st.add(pout), o2 = st.add(kl);
  char *base = st.commit();
  if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
  CUDA_OK(ctx, k_scalar(ctx->k, (const u64 *const *)(base + o0), (u64 *const *)(base + o1), (const u64 *)(base + o2), (int)n, L, add_const));
  sc.ok = true;
  for (size_t i = 0; i < n; i++) out[i] = made[i];
  return FENC_OK;
}
extern "C" fenc_status fenc_mul_scalar(fenc_ctx *ctx, fenc_ct *const *in, size_t n, const uint64_t *k_res, double scale_factor,
                                       fenc_ct **out) {
  return scalar_op(ctx, in, n, k_res, scale_factor, false, out);
}
extern "C" fenc_status fenc_add_const(fenc_ctx *ctx, fenc_ct *const *in, size_t n, const uint64_t *k_res, fenc_ct **out) {
  return scalar_op(ctx, in, n, k_res, 1.0, true, out);
}

extern "C" fenc_status fenc_sum_groups(fenc_ctx *ctx, fenc_ct *const *in, size_t group, size_t n_groups, fenc_ct **out) {
  Scope sc(ctx);
  if (!ctx || !in || !out || group == 0) return FENC_ERR_INVALID_ARG;
  if (n_groups == 0) return FENC_OK;
  const int L = in[0]->L;
  std::vector<const u64 *> terms(group * n_groups);
  std::vector<int> start(n_groups + 1);
  std::vector<u64 *> outs(n_groups);
  std::vector<fenc_ct *> made(n_groups, nullptr);
  for (size_t i = 0; i < group * n_groups; i++) {
    if (in[i]->L != L || !scale_close(in[i]->scale, in[0]->scale)) return fail(ctx, FENC_ERR_MISMATCH, "sum: level or scale differ");
    terms[i] = in[i]->d;
  }
  for (size_t g = 0; g < n_groups; g++) {
    made[g] = sc.ct(L, in[0]->scale);
    if (!made[g]) return fail(ctx, FENC_ERR_OOM, "sum output");
    start[g] = (int)(g * group), outs[g] = made[g]->d;
  }
  start[n_groups] = (int)(group * n_groups);
  DescStage st(ctx);
  size_t o0 = st.add(terms), o1 = st.add(start), o2 = st.add(outs);
  char *base = st.commit();
  if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
  CUDA_OK(ctx, k_add_many(ctx->k, (const u64 *const *)(base + o0), (const int *)(base + o1), (u64 *const *)(base + o2), (int)n_groups, L,
                          (int)terms.size()));
  sc.ok = true;
  for (size_t g = 0; g < n_groups; g++) out[g] = made[g];
  return FENC_OK;
}

// ------------------------------------------------------------------------------------------------ pooling order, activation
// indices such that consecutive groups of four are the fragments (2u_o + a, 2v_o + b) of output fragment (u_o, v_o);
// ciphertext order [...][u][v] (pooling keeps or combines whole fragment ciphertexts)
static fenc_status pool_gather(fenc_ctx *ctx, fenc_ct *const *in, size_t n, uint32_t S, std::vector<fenc_ct *> &ordered) {
  if (S < 2 || (S & 1) || n % ((size_t)S * S)) return fail(ctx, FENC_ERR_LAYOUT, "pool needs an even S and a multiple of S^2 ciphertexts");
  ordered.clear();
  for (size_t base = 0; base < n; base += (size_t)S * S)
    for (uint32_t uo = 0; uo < S / 2; uo++)
      for (uint32_t vo = 0; vo < S / 2; vo++)
        for (int a = 0; a < 2; a++)
          for (int b = 0; b < 2; b++) ordered.push_back(in[base + (2 * uo + a) * S + (2 * vo + b)]);
  return FENC_OK;
}
extern "C" fenc_status fenc_sum_pool(fenc_ctx *ctx, fenc_ct *const *in, size_t n, uint32_t S, fenc_ct **out) {
  if (!ctx || !in || !out) return FENC_ERR_INVALID_ARG;
  std::vector<fenc_ct *> ord;
  fenc_status st = pool_gather(ctx, in, n, S, ord);
  if (st != FENC_OK) return st;
  return fenc_sum_groups(ctx, ord.data(), 4, n / 4, out);
}
extern "C" fenc_status fenc_square_sum_pool(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, size_t n, uint32_t S, fenc_ct **out) {
  if (!ctx || !K || !in || !out) return FENC_ERR_INVALID_ARG;
  std::vector<fenc_ct *> ord;
  fenc_status st = pool_gather(ctx, in, n, S, ord);
  if (st != FENC_OK) return st;
  return cmult_relin(ctx, K, ord.data(), ord.data(), n / 4, out, 4);
}

// Degree-3 activation (R2.12): the library owns the order of the steps, the caller the three exactly rounded integers.
extern "C" fenc_status fenc_poly3(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, size_t n, const uint64_t *k3_res,
                                  const uint64_t *k1_res, const uint64_t *k0_res, double scale_sq, fenc_ct **out) {
  if (!ctx || !K || !in || !k3_res || !k1_res || !k0_res || !out) return FENC_ERR_INVALID_ARG;
  if (n == 0) return FENC_OK;
  const int L = in[0]->L;
  if (L < 3) return fail(ctx, FENC_ERR_LEVEL, "the degree-3 activation needs two levels");
  struct Tmp {  // intermediate ciphertexts of this call
    std::vector<fenc_ct *> v;
    ~Tmp() { for (fenc_ct *c : v) fenc_ct_free(c); }
    fenc_ct **fresh(size_t n) { size_t at = v.size(); v.resize(at + n, nullptr); return v.data() + at; }
  } tmp;
  tmp.v.reserve(8 * n);  // no reallocation: the pointers handed out stay valid
  fenc_status st;
  fenc_ct **x2 = tmp.fresh(n), **t0 = tmp.fresh(n), **t = tmp.fresh(n), **x3 = tmp.fresh(n), **u0 = tmp.fresh(n), **u1 = tmp.fresh(n),
          **u = tmp.fresh(n), **y = tmp.fresh(n);
  if ((st = cmult_relin(ctx, K, in, in, n, x2)) != FENC_OK) return st;                                  // x^2 at L-1
  if ((st = scalar_op(ctx, in, n, k3_res, (double)ctx->mod[L - 1], false, t0)) != FENC_OK) return st;    // a3 q_{L-1} x
  if ((st = fenc_rescale(ctx, t0, n, t)) != FENC_OK) return st;                                          // a3 x at L-1
  if ((st = cmult_relin(ctx, K, x2, t, n, x3)) != FENC_OK) return st;                                    // a3 x^3 at L-2
  if ((st = scalar_op(ctx, in, n, k1_res, scale_sq, false, u0)) != FENC_OK) return st;                   // a1 s^2 x
  if ((st = fenc_rescale(ctx, u0, n, u1)) != FENC_OK) return st;
  if ((st = fenc_rescale(ctx, u1, n, u)) != FENC_OK) return st;                                          // a1 x at L-2, scale s3
  for (size_t i = 0; i < n; i++)
    if ((st = fenc_add(ctx, x3[i], u[i], &y[i])) != FENC_OK) return st;
  return scalar_op(ctx, y, n, k0_res, 1.0, true, out);
}

// ------------------------------------------------------------------------------------------------ raw NTT (a1)
extern "C" fenc_status fenc_ntt_rows(fenc_ctx *ctx, void *device_rows, const int32_t *mod_idx, size_t n_rows, int inverse) {
  if (!ctx || !device_rows || !mod_idx) return FENC_ERR_INVALID_ARG;
  std::vector<RowDesc> rows(n_rows);
  std::vector<ShoupC> sc(n_rows);
  for (size_t r = 0; r < n_rows; r++) {
    if (mod_idx[r] < 0 || mod_idx[r] >= ctx->A) return FENC_ERR_INVALID_ARG;
    u64 m = ctx->mod[mod_idx[r]];
    u64 ni = fh::invmod((u64)ctx->N % m, m);
    rows[r] = RowDesc{mod_idx[r], (int)r, (int)r, 0, 0, {0, 0, 0}};
    sc[r] = ShoupC{ni, fh::shoup(ni, m)};
  }
  DescStage st(ctx);
  size_t o0 = st.add(rows), o1 = st.add(sc);
  char *base = st.commit();
  if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
  u64 *p = (u64 *)device_rows;
  if (inverse) CUDA_OK(ctx, k_intt(ctx->k, nullptr, p, 0, false, p, 0, (const RowDesc *)(base + o0), (int)n_rows, (const ShoupC *)(base + o1), 1));
  else CUDA_OK(ctx, k_ntt(ctx->k, p, 0, p, 0, (const RowDesc *)(base + o0), (int)n_rows, 1));
  return FENC_OK;
}
