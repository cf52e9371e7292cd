// fenc_ctx.cu -- context, per-level key-switch tables, workspace, and the batched key-switch / rescale drivers.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "fenc_ctx.h"

fenc_status fail(fenc_ctx *ctx, fenc_status st, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (ctx) ctx->err = buf;
  return st;
}

// Device memory comes from the caller's allocator (a callback into the host framework) or cudaMalloc.  Blocks up to
// POOL_BLOCK_MAX are kept in per-size free lists when released and handed out again without leaving the library: a
// layer creates and drops hundreds of ciphertext-sized buffers per call, the same sizes every step, and the callbacks
// alone made the FC layers host-bound.  Everything the library enqueues runs on the context's stream, so a block reused
// by a later call is ordered after the work that last touched it.
static const size_t POOL_BLOCK_MAX = (size_t)64 << 20, POOL_BYTES_MAX = (size_t)4 << 30;
static void *raw_alloc(fenc_ctx *ctx, size_t bytes) {
  void *p = nullptr;
  if (ctx->dev_alloc) p = ctx->dev_alloc(bytes, ctx->user);
  else if (cudaMalloc(&p, bytes) != cudaSuccess) p = nullptr;
  if (!p) (void)cudaGetLastError();
  return p;
}
static void raw_free(fenc_ctx *ctx, void *p) {
  if (ctx->dev_free) ctx->dev_free(p, ctx->user);
  else cudaFree(p);
}
void pool_release(fenc_ctx *ctx) {
  for (auto &kv : ctx->pool)
    for (void *p : kv.second) raw_free(ctx, p);
  ctx->pool.clear();
  ctx->pool_bytes = 0;
}
void *dalloc(fenc_ctx *ctx, size_t bytes) {
  if (bytes == 0) bytes = 256;
  void *p = nullptr;
  if (bytes <= POOL_BLOCK_MAX) {
    auto it = ctx->pool.find(bytes);
    if (it != ctx->pool.end() && !it->second.empty()) {
      p = it->second.back();
      it->second.pop_back();
      ctx->pool_bytes -= bytes;
    }
  }
  if (!p) p = raw_alloc(ctx, bytes);
  if (!p && ctx->pool_bytes) {  // out of memory with blocks parked in the pool: give them back and retry
    pool_release(ctx);
    p = raw_alloc(ctx, bytes);
  }
  if (p) {
    ctx->live[p] = bytes;
    ctx->dev_bytes += bytes;
  }
  return p;
}
void dfree(fenc_ctx *ctx, void *p) {
  if (!p) return;
  size_t bytes = 0;
  auto it = ctx->live.find(p);
  if (it != ctx->live.end()) {
    bytes = it->second;
    ctx->dev_bytes -= bytes;
    ctx->live.erase(it);
  }
  if (bytes && bytes <= POOL_BLOCK_MAX && ctx->pool_bytes + bytes <= POOL_BYTES_MAX) {
    ctx->pool[bytes].push_back(p);
    ctx->pool_bytes += bytes;
    return;
  }
  raw_free(ctx, p);
}
void *workspace(fenc_ctx *ctx, size_t bytes) {
  if (bytes > ctx->ws_bytes) {
    dfree(ctx, ctx->ws);
    ctx->ws_bytes = 0;
    ctx->ws = dalloc(ctx, bytes);
    if (ctx->ws) ctx->ws_bytes = bytes;
  }
  return ctx->ws;
}
// Descriptor arrays go through a ring of pinned host slots: a copy from pageable memory would synchronise the stream
// before every batch (and stall the host-side enqueue of the next kernels behind all queued GPU work).
// The slot reaches the device through a small kernel that reads the page-locked slot over the bus (pinned allocations
// are device-addressable under unified addressing), not through the copy engine: a descriptor copy queued behind the bulk
// uploads of fenc_ct_import_async would hold the compute stream back for as long as those take (measured: the whole
// 1.3 ms of a LeNet-5 request's upload, once per step).
__global__ void desc_copy_kernel(uint4 *dst, const uint4 *src, size_t n16) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}
static const size_t DESC_SLOT = (size_t)1 << 20;
static const int DESC_SLOTS = FENC_DESC_SLOTS;
char *DescStage::commit() {
  size_t need = (host.size() + 255) & ~(size_t)255;
  if (need > ctx->desc_bytes) {
    dfree(ctx, ctx->desc_buf);
    size_t cap = need < DESC_SLOT ? DESC_SLOT : need * 2;
    ctx->desc_buf = dalloc(ctx, cap);
    ctx->desc_bytes = ctx->desc_buf ? cap : 0;
    if (!ctx->desc_buf) return nullptr;
  }
  if (host.empty()) return (char *)ctx->desc_buf;
  if (host.size() <= DESC_SLOT) {
    if (!ctx->desc_pinned) {
      if (cudaHostAlloc(&ctx->desc_pinned, DESC_SLOT * DESC_SLOTS, cudaHostAllocDefault) != cudaSuccess) ctx->desc_pinned = nullptr;
      for (int i = 0; i < DESC_SLOTS && ctx->desc_pinned; i++) cudaEventCreateWithFlags(&ctx->desc_ev[i], cudaEventDisableTiming);
    }
    if (ctx->desc_pinned) {
      const int slot = ctx->desc_next++ % DESC_SLOTS;
      if (ctx->desc_used[slot]) cudaEventSynchronize(ctx->desc_ev[slot]);  // the copy that last read this slot is done
      char *h = (char *)ctx->desc_pinned + (size_t)slot * DESC_SLOT;
      memcpy(h, host.data(), host.size());
      const size_t n16 = (host.size() + 15) / 16;
      const unsigned blocks = (unsigned)std::min<size_t>((n16 + 255) / 256, 128);
      desc_copy_kernel<<<blocks, 256, 0, ctx->stream>>>((uint4 *)ctx->desc_buf, (const uint4 *)h, n16);
      ctx->launches++;
      if (cudaGetLastError() != cudaSuccess) return nullptr;
      cudaEventRecord(ctx->desc_ev[slot], ctx->stream);
      ctx->desc_used[slot] = true;
      return (char *)ctx->desc_buf;
    }
  }
  if (cudaMemcpyAsync(ctx->desc_buf, host.data(), host.size(), cudaMemcpyHostToDevice, ctx->stream) != cudaSuccess) return nullptr;
  return (char *)ctx->desc_buf;
}
fenc_ct *new_ct(fenc_ctx *ctx, int L, double scale) {
  u64 *d = dalloc_t<u64>(ctx, (size_t)2 * L * ctx->N);
  if (!d) return nullptr;
  return new fenc_ct{ctx, L, scale, d};
}
u32 galois_elt(const fenc_ctx *ctx, int step) {
  int r = ((step % ctx->n) + ctx->n) % ctx->n;
  return (u32)fh::powmod(5, (u64)r, 2ull * ctx->N);
}

// ------------------------------------------------------------------------------------------------ context
extern "C" fenc_status fenc_params_init(const fenc_params_desc *d, fenc_ctx **out) {
  if (!d || !out) return FENC_ERR_INVALID_ARG;
  std::unique_ptr<fenc_ctx, void (*)(fenc_ctx *)> c(new fenc_ctx(), fenc_ctx_free);
  fenc_ctx *ctx = c.get();
  if (d->log2N < 4 || d->log2N > 16 || d->n_q < 1 || d->n_p < 1 || d->n_q + d->n_p > FENC_MAX_MOD || d->q_bits > 60 ||
      d->p_bits > 60 || (d->dnum < 1 && !d->dlen_override))
    return FENC_ERR_PARAMS;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || d->device < 0 || d->device >= ndev) {
    (void)cudaGetLastError();
    return FENC_ERR_DEVICE;  // no CPU fallback
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, d->device) != cudaSuccess || prop.major != 10) return FENC_ERR_DEVICE;
  if (cudaSetDevice(d->device) != cudaSuccess) return FENC_ERR_DEVICE;
  ctx->device = d->device;
  ctx->stream = (cudaStream_t)d->cuda_stream;
  ctx->dev_alloc = d->dev_alloc, ctx->dev_free = d->dev_free, ctx->user = d->user;
  ctx->logN = d->log2N, ctx->N = 1 << d->log2N, ctx->n = ctx->N / 2;
  ctx->nq = d->n_q, ctx->np = d->n_p, ctx->A = ctx->nq + ctx->np;
  std::vector<u64> q, p;
  if (d->q_override) q.assign(d->q_override, d->q_override + d->n_q);
  else if (!fh::find_primes(ctx->logN, d->q_bits, d->n_q, q)) return FENC_ERR_PARAMS;
  if (d->p_override) p.assign(d->p_override, d->p_override + d->n_p);
  else if (!fh::find_primes(ctx->logN, d->p_bits, d->n_p, p)) return FENC_ERR_PARAMS;
  ctx->mod = q;
  ctx->mod.insert(ctx->mod.end(), p.begin(), p.end());
  for (size_t i = 0; i < ctx->mod.size(); i++) {
    u64 m = ctx->mod[i];
    if (m >= (1ull << 61) || m % (2ull * ctx->N) != 1 || !fh::is_prime(m)) return FENC_ERR_PARAMS;
    for (size_t k = 0; k < i; k++)
      if (ctx->mod[k] == m) return FENC_ERR_PARAMS;
  }
  ctx->dlen = d->dlen_override ? (int)d->dlen_override : (ctx->nq + (int)d->dnum - 1) / (int)d->dnum;
  if (ctx->dlen < 1 || ctx->dlen > ctx->nq) return FENC_ERR_PARAMS;
  ctx->beta_max = (ctx->nq + ctx->dlen - 1) / ctx->dlen;
  // key-switch noise condition P >= max_j Q_j (A1)
  long double logP = 0, logQj = 0;
  for (u64 m : p) logP += log2l((long double)m);
  for (int i = 0; i < ctx->dlen; i++) logQj += log2l((long double)q[i]);
  if (logP < logQj && !d->allow_noisy_ks) return FENC_ERR_PARAMS;
  // lazy 128-bit accumulation bounds (fenc_device.cuh): sums must stay below t 2^64
  u64 qmax = 0, pmax = 0;
  for (u64 m : q) qmax = m > qmax ? m : qmax;
  for (u64 m : p) pmax = m > pmax ? m : pmax;
  u64 allmax = qmax > pmax ? qmax : pmax;
  if ((u64)ctx->beta_max > ~0ull / allmax) return FENC_ERR_PARAMS;
  ctx->lazy_q = (int)std::min<u64>(~0ull / qmax, 1u << 20);  // base-conversion terms per Montgomery reduction
  ctx->lazy_p = (int)std::min<u64>(~0ull / pmax, 1u << 20);
  u64 ml = ~0ull / qmax;
  ctx->max_lazy = ml > (1u << 20) ? (1 << 20) : (int)ml;
  ctx->default_scale = std::ldexp(1.0, (int)d->log2_scale);
  // device tables
  const int A = ctx->A, N = ctx->N;
  std::vector<ModConst> mods(A);
  std::vector<ShoupC> fwd((size_t)A * N), inv((size_t)A * N), ninv(A);
  std::vector<RowDesc> ident(A);
  std::vector<int> imod(2 * A);
  ctx->psi.resize(A);
  for (int i = 0; i < A; i++) {
    u64 m = ctx->mod[i];
    ctx->psi[i] = fh::find_psi(m, N);
    int bits = 64 - __builtin_clzll(m - 1);
    mods[i] = ModConst{m, fh::neg_qinv(m), fh::to_mont(fh::to_mont(1, m), m), (bits >= 64 ? ~0ull : (1ull << bits) - 1), (u64)((((u128)1) << 64) / m), fh::f64_modulus(m, ctx->logN) ? fh::double_bits(1.0 / (double)m) : 0ull, {0, 0}};
    fh::build_twiddles(m, ctx->psi[i], ctx->logN, &fwd[(size_t)i * N], &inv[(size_t)i * N]);
    u64 ni = fh::invmod((u64)N % m, m);
    ninv[i] = ShoupC{ni, fh::shoup(ni, m)};
    ident[i] = RowDesc{i, i, i, 0, 0, {0, 0, 0}};
    imod[i] = imod[A + i] = i;
  }
  ctx->d_mods = dalloc_t<ModConst>(ctx, A);
  ctx->d_tw_fwd = dalloc_t<ShoupC>(ctx, (size_t)A * N);
  ctx->d_tw_inv = dalloc_t<ShoupC>(ctx, (size_t)A * N);
  ctx->d_ident_rows = dalloc_t<RowDesc>(ctx, A);
  ctx->d_ninv = dalloc_t<ShoupC>(ctx, A);
  ctx->d_ident_mod = dalloc_t<int>(ctx, 2 * A);
  if (!ctx->d_mods || !ctx->d_tw_fwd || !ctx->d_tw_inv || !ctx->d_ident_rows || !ctx->d_ninv || !ctx->d_ident_mod) return FENC_ERR_OOM;
  cudaMemcpy(ctx->d_mods, mods.data(), A * sizeof(ModConst), cudaMemcpyHostToDevice);
  cudaMemcpy(ctx->d_tw_fwd, fwd.data(), fwd.size() * sizeof(ShoupC), cudaMemcpyHostToDevice);
  cudaMemcpy(ctx->d_tw_inv, inv.data(), inv.size() * sizeof(ShoupC), cudaMemcpyHostToDevice);
  cudaMemcpy(ctx->d_ident_rows, ident.data(), A * sizeof(RowDesc), cudaMemcpyHostToDevice);
  cudaMemcpy(ctx->d_ninv, ninv.data(), A * sizeof(ShoupC), cudaMemcpyHostToDevice);
  if (cudaMemcpy(ctx->d_ident_mod, imod.data(), 2 * A * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) return FENC_ERR_CUDA;
  // 2-pass NTT geometry
  NttGeom g{};
  g.logN = ctx->logN;
  if (ctx->logN <= 11) {
    g.brow = ctx->logN, g.bcol = 0, g.lt_row = ctx->logN, g.lt_col = ctx->logN, g.lc_col = ctx->logN;
  } else {
    g.brow = 8, g.bcol = ctx->logN - 8, g.lt_row = FENC_ROW_LT, g.lc_col = 4, g.lt_col = g.bcol + 4;
  }
  ctx->k = KCtx{(void *)ctx->stream, g, ctx->d_mods, ctx->d_tw_fwd, ctx->d_tw_inv, &ctx->launches, N, ctx->nq, ctx->np, nullptr};
  *out = c.release();
  return FENC_OK;
}

extern "C" void fenc_ctx_free(fenc_ctx *ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
  for (auto &kv : ctx->plans)
    for (void *p : kv.second->owned) dfree(ctx, p);
  if (ctx->copy_stream) cudaStreamSynchronize(ctx->copy_stream);
  for (StageSlot &sl : ctx->stage) {
    dfree(ctx, sl.d);
    if (sl.copied) cudaEventDestroy(sl.copied);
    if (sl.consumed) cudaEventDestroy(sl.consumed);
  }
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  export_drain(ctx, true);
  for (cudaEvent_t e : ctx->export_events) cudaEventDestroy(e);
  if (ctx->export_ready) cudaEventDestroy(ctx->export_ready);
  if (ctx->d2h_stream) cudaStreamDestroy(ctx->d2h_stream);
  dfree(ctx, ctx->ws), dfree(ctx, ctx->desc_buf);
  if (ctx->desc_pinned) {
    for (int i = 0; i < FENC_DESC_SLOTS; i++) cudaEventDestroy(ctx->desc_ev[i]);
    cudaFreeHost(ctx->desc_pinned);
  }
  dfree(ctx, ctx->d_mods), dfree(ctx, ctx->d_tw_fwd), dfree(ctx, ctx->d_tw_inv);
  dfree(ctx, ctx->d_ident_rows), dfree(ctx, ctx->d_ninv), dfree(ctx, ctx->d_ident_mod);
  pool_release(ctx);
  delete ctx;
}
extern "C" const char *fenc_last_error(fenc_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }
extern "C" fenc_status fenc_get_primes(fenc_ctx *ctx, uint64_t *q, uint64_t *p, uint32_t *dlen, uint32_t *beta_max) {
  if (!ctx) return FENC_ERR_INVALID_ARG;
  if (q) memcpy(q, ctx->mod.data(), ctx->nq * sizeof(u64));
  if (p) memcpy(p, ctx->mod.data() + ctx->nq, ctx->np * sizeof(u64));
  if (dlen) *dlen = ctx->dlen;
  if (beta_max) *beta_max = ctx->beta_max;
  return FENC_OK;
}
extern "C" fenc_status fenc_set_hoisting(fenc_ctx *ctx, int on) {
  if (!ctx) return FENC_ERR_INVALID_ARG;
  ctx->hoist_inner = on != 0;
  return FENC_OK;
}
extern "C" fenc_status fenc_sync(fenc_ctx *ctx) {
  if (!ctx) return FENC_ERR_INVALID_ARG;
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  return export_drain(ctx, true);  // results of fenc_ct_export_async have landed once a synchronising call returns
}
extern "C" uint64_t fenc_launch_count(fenc_ctx *ctx, int reset) {
  if (!ctx) return 0;
  u64 v = ctx->launches;
  if (reset) ctx->launches = 0;
  return v;
}
extern "C" uint64_t fenc_device_bytes(fenc_ctx *ctx) { return ctx ? ctx->dev_bytes : 0; }

// ------------------------------------------------------------------------------------------------ per-level tables
// DESIGN.md R2.6: digit j = limbs [j dlen, min((j+1) dlen, L)), Q_j its product;
//   ModUp:   y_i = d[q_i] [(Q_j/q_i)^-1]_{q_i},   up_j[t] = sum_i y_i ((Q_j/q_i) mod t)          (no correction)
//   ModDown: y_i = acc[p_i] [(P/p_i)^-1]_{p_i},   out[t] = (acc[t] - sum_i y_i ((P/p_i) mod t)) [P^-1]_t
// DESIGN.md R2.8: rescale c'[t] = (c[t] - (c[q_{L-1}] mod t)) [q_{L-1}^-1]_t.
LevelPlan *get_plan(fenc_ctx *ctx, int L) {
  auto it = ctx->plans.find(L);
  if (it != ctx->plans.end()) return it->second.get();
  std::unique_ptr<LevelPlan> pl(new LevelPlan());
  LevelPlan &P = *pl;
  const int np = ctx->np, nq = ctx->nq, dlen = ctx->dlen, A = ctx->A;
  const std::vector<u64> &mod = ctx->mod;
  P.L = L, P.E = L + np, P.beta = (L + dlen - 1) / dlen;
  const int E = P.E;
  auto emod = [&](int row) { return row < L ? row : nq + (row - L); };
  auto shoupc = [&](u64 c, u64 m) { return ShoupC{c, fh::shoup(c, m)}; };
  std::vector<RowDesc> rows_in(L), rows_up, rows_p(2 * np), rows_down(2 * L), rows_div(2 * L), rows_ct(2 * L);
  std::vector<ShoupC> scale_in(L), scale_p(2 * np), mul_pinv(A, ShoupC{0, 0}), scale_ct(2 * L);
  std::vector<u64> bc_up, bc_down((size_t)L * np);
  std::vector<ShoupC> bc_up_f64, bc_rs_f64;
  std::vector<int> tmp_index((size_t)P.beta * E, -1);
  std::vector<ConvGroup> groups_up, groups_down, groups_rs;
  for (int j = 0; j < P.beta; j++) {
    const int lo = j * dlen, hi = std::min(lo + dlen, L);
    for (int i = lo; i < hi; i++) {
      u64 qi = mod[i], qhat = 1;
      for (int i2 = lo; i2 < hi; i2++)
        if (i2 != i) qhat = fh::mulmod(qhat, mod[i2] % qi, qi);
      u64 ninv = fh::invmod((u64)ctx->N % qi, qi);
      rows_in[i] = RowDesc{i, i, i, 0, 0, {0, 0, 0}};
      scale_in[i] = shoupc(fh::mulmod(ninv, fh::invmod(qhat, qi), qi), qi);
    }
    bool src_f64 = true;
    for (int i = lo; i < hi; i++) src_f64 = src_f64 && fh::f64_modulus(mod[i], ctx->logN);  // below 2^50: conv_dot_f64
    groups_up.push_back(ConvGroup{lo, lo, hi - lo, lo, (int)rows_up.size(), E - (hi - lo), {src_f64 ? 2 : 0, 0}});
    P.n_src_up = std::max(P.n_src_up, hi - lo);
    for (int t = 0; t < E; t++) {
      if (t >= lo && t < hi) continue;
      const u64 T = mod[emod(t)];
      RowDesc rd{emod(t), lo, (int)rows_up.size(), hi - lo, (int)bc_up.size(), {0, 0, 0}};
      for (int i = lo; i < hi; i++) {
        u64 c = 1;
        for (int i2 = lo; i2 < hi; i2++)
          if (i2 != i) c = fh::mulmod(c, mod[i2] % T, T);
        bc_up.push_back(fh::to_mont(c, T));
        bc_up_f64.push_back(ShoupC{fh::double_bits((double)c), fh::double_bits((double)((long double)c / (long double)T))});
      }
      tmp_index[(size_t)j * E + t] = rd.dst_row;
      rows_up.push_back(rd);
    }
  }
  P.n_up = (int)rows_up.size();
  for (int c = 0; c < 2; c++)
    for (int i = 0; i < np; i++) {
      u64 pi = mod[nq + i], phat = 1;
      for (int i2 = 0; i2 < np; i2++)
        if (i2 != i) phat = fh::mulmod(phat, mod[nq + i2] % pi, pi);
      u64 ninv = fh::invmod((u64)ctx->N % pi, pi);
      rows_p[c * np + i] = RowDesc{nq + i, c * E + L + i, c * np + i, 0, 0, {0, 0, 0}};
      scale_p[c * np + i] = shoupc(fh::mulmod(ninv, fh::invmod(phat, pi), pi), pi);
    }
  for (int t = 0; t < L; t++) {
    const u64 T = mod[t];
    u64 Pm = 1;
    for (int i = 0; i < np; i++) {
      Pm = fh::mulmod(Pm, mod[nq + i] % T, T);
      u64 c = 1;
      for (int i2 = 0; i2 < np; i2++)
        if (i2 != i) c = fh::mulmod(c, mod[nq + i2] % T, T);
      bc_down[(size_t)t * np + i] = fh::to_mont(c, T);
    }
    mul_pinv[t] = shoupc(fh::invmod(Pm, T), T);
    u64 ninv = fh::invmod((u64)ctx->N % T, T);
    for (int c = 0; c < 2; c++) {
      rows_down[c * L + t] = RowDesc{t, c * np, c * L + t, np, t * np, {0, 0, 0}};
      rows_div[c * L + t] = RowDesc{t, c * L + t, c * L + t, c, c * E + t, {0, 0, 0}};
      rows_ct[c * L + t] = RowDesc{t, c * L + t, c * L + t, 0, 0, {0, 0, 0}};
      scale_ct[c * L + t] = shoupc(ninv, T);
    }
  }
  for (int c = 0; c < 2; c++) {
    groups_down.push_back(ConvGroup{c * np, nq, np, c * np, c * L, L, {0, 0}});
    groups_rs.push_back(ConvGroup{c, L - 1, 1, c, c * (L - 1), L - 1, {(L >= 2 && fh::f64_modulus(mod[L - 1], ctx->logN)) ? 2 : 0, 0}});
  }
  P.d_groups_up = upload_owned(ctx, P.owned, groups_up);
  P.d_groups_down = upload_owned(ctx, P.owned, groups_down);
  P.d_groups_rs = upload_owned(ctx, P.owned, groups_rs);
  P.d_rows_in = upload_owned(ctx, P.owned, rows_in);
  P.d_scale_in = upload_owned(ctx, P.owned, scale_in);
  P.d_rows_up = upload_owned(ctx, P.owned, rows_up);
  P.d_bc_up = upload_owned(ctx, P.owned, bc_up);
  P.d_bc_up_f64 = upload_owned(ctx, P.owned, bc_up_f64);
  P.d_tmp_index = upload_owned(ctx, P.owned, tmp_index);
  P.d_rows_p = upload_owned(ctx, P.owned, rows_p);
  P.d_scale_p = upload_owned(ctx, P.owned, scale_p);
  P.d_rows_down = upload_owned(ctx, P.owned, rows_down);
  P.d_bc_down = upload_owned(ctx, P.owned, bc_down);
  P.d_rows_div = upload_owned(ctx, P.owned, rows_div);
  P.d_mul_pinv = upload_owned(ctx, P.owned, mul_pinv);
  P.d_rows_ct = upload_owned(ctx, P.owned, rows_ct);
  P.d_scale_ct = upload_owned(ctx, P.owned, scale_ct);
  // rescale tables
  const int L1 = L - 1;
  std::vector<RowDesc> rs_in(2), rs_up, rs_div;
  std::vector<ShoupC> rs_scale(2), mul_ql(A, ShoupC{0, 0});
  std::vector<u64> bc_rs;
  if (L >= 2) {
    const u64 ql = mod[L1];
    u64 ninv = fh::invmod((u64)ctx->N % ql, ql);
    for (int c = 0; c < 2; c++) {
      rs_in[c] = RowDesc{L1, c * L + L1, c, 0, 0, {0, 0, 0}};
      rs_scale[c] = shoupc(ninv, ql);
    }
    for (int t = 0; t < L1; t++) {
      bc_rs.push_back(fh::to_mont(1, mod[t]));
      bc_rs_f64.push_back(ShoupC{fh::double_bits(1.0), fh::double_bits(1.0 / (double)mod[t])});
      mul_ql[t] = shoupc(fh::invmod(ql % mod[t], mod[t]), mod[t]);
    }
    for (int c = 0; c < 2; c++)
      for (int t = 0; t < L1; t++) {
        rs_up.push_back(RowDesc{t, c, c * L1 + t, 1, t, {0, 0, 0}});
        rs_div.push_back(RowDesc{t, c * L1 + t, c * L1 + t, c, c * L + t, {0, 0, 0}});
      }
  }
  if (L >= 2) {
    std::vector<RowDesc> rows_p2, rows_down2, rows_div2;
    std::vector<ShoupC> scale_p2;
    std::vector<ConvGroup> groups_down2;
    for (int c = 0; c < 2; c++) {
      for (int i = 0; i < np; i++) {
        RowDesc rd = rows_p[c * np + i];
        rd.dst_row = c * (np + 1) + i;
        rows_p2.push_back(rd);
        scale_p2.push_back(scale_p[c * np + i]);
      }
      rows_p2.push_back(RowDesc{L1, c * E + L1, c * (np + 1) + np, 1, c, {0, 0, 0}});
      scale_p2.push_back(rs_scale[c]);
      groups_down2.push_back(ConvGroup{c * (np + 1), nq, np + 1, c * (np + 1), c * L1, L1, {1, L1}});
      for (int t = 0; t < L1; t++) {
        rows_down2.push_back(RowDesc{t, c * (np + 1), c * L1 + t, np, t * np, {0, 0, 0}});
        rows_div2.push_back(RowDesc{t, c * L1 + t, c * L1 + t, c, c * E + t, {0, 0, 0}});
      }
    }
    P.d_rows_p2 = upload_owned(ctx, P.owned, rows_p2);
    P.d_scale_p2 = upload_owned(ctx, P.owned, scale_p2);
    P.d_groups_down2 = upload_owned(ctx, P.owned, groups_down2);
    P.d_rows_down2 = upload_owned(ctx, P.owned, rows_down2);
    P.d_rows_div2 = upload_owned(ctx, P.owned, rows_div2);
  }
  P.d_rows_rs_in = upload_owned(ctx, P.owned, rs_in);
  P.d_scale_rs = upload_owned(ctx, P.owned, rs_scale);
  P.d_rows_rs_up = upload_owned(ctx, P.owned, rs_up);
  P.d_bc_rs = upload_owned(ctx, P.owned, bc_rs);
  P.d_bc_rs_f64 = upload_owned(ctx, P.owned, bc_rs_f64);
  P.d_rows_rs_div = upload_owned(ctx, P.owned, rs_div);
  P.d_mul_qlinv = upload_owned(ctx, P.owned, mul_ql);
  cudaStreamSynchronize(ctx->stream);  // host vectors go out of scope
  for (void *p : P.owned)
    if (!p) return nullptr;
  LevelPlan *ret = pl.get();
  ctx->plans[L] = std::move(pl);
  return ret;
}

// ------------------------------------------------------------------------------------------------ batched key switch
static const size_t WS_CAP = (size_t)6 << 30;  // workspace budget for one chunk of a batch
static const size_t GRID_Z_MAX = 65535;          // CUDA's limit on gridDim.z (small rings reach it before WS_CAP)

bool ks_can_merge_rescale(const fenc_ctx *ctx, int L) {
  return L >= 2 && convert_cols_fits(ctx->logN, ctx->np + 1, true);
}

fenc_status ks_batch(fenc_ctx *ctx, int L, std::vector<BatchItem> &items, bool rescale_after, const HoistUp *hoist) {
  if (items.empty()) return FENC_OK;
  if (rescale_after && !ks_can_merge_rescale(ctx, L)) return fail(ctx, FENC_ERR_INVALID_ARG, "merged rescale unavailable here");
  LevelPlan *P = get_plan(ctx, L);
  if (!P) return fail(ctx, FENC_ERR_OOM, "level plan");
  const size_t N = ctx->N;
  const int E = P->E, np = ctx->np, npy = rescale_after ? ctx->np + 1 : ctx->np;
  const size_t per = ((size_t)L + P->n_up + 2 * E + 2 * npy + 2 * L) * N;  // u64 per item
  size_t chunk = WS_CAP / (per * 8);
  if (chunk < 1) chunk = 1;
  if (chunk > GRID_Z_MAX) chunk = GRID_Z_MAX;  // the batch index is blockIdx.z in the transform kernels
  if (chunk > items.size()) chunk = items.size();
  u64 *ws = (u64 *)workspace(ctx, chunk * per * 8);
  if (!ws) return fail(ctx, FENC_ERR_OOM, "key-switch workspace (%zu bytes)", chunk * per * 8);
  u64 *y = ws, *tmp = y + chunk * L * N, *acc = tmp + chunk * P->n_up * N, *yP = acc + chunk * 2 * E * N,
      *tmp2 = yP + chunk * 2 * npy * N;
  const KCtx &k = ctx->k;
  for (size_t at = 0; at < items.size(); at += chunk) {
    const int nb = (int)std::min(chunk, items.size() - at);
    DescStage st(ctx);
    std::vector<BatchItem> part(items.begin() + at, items.begin() + at + nb);
    // items sharing a key run as neighbouring blocks (L2 reuse of the key tile)
    std::stable_sort(part.begin(), part.end(), [](const BatchItem &a, const BatchItem &b) { return a.evk < b.evk; });
    int n_keys = 0;
    for (int i = 0; i < nb; i++) n_keys += (i == 0 || part[i].evk != part[i - 1].evk);
    st.add(part);
    const BatchItem *d_items = (const BatchItem *)st.commit();
    if (!d_items) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
    // a2 + a1 + a3: inverse row pass of sigma_g(d); then ONE fused column kernel per digit group: inverse column
    // stages + ModUp scaling of the digit's limbs in shared memory, base conversion and forward column stages per target
    const bool fused_up = convert_cols_fits(ctx->logN, P->n_src_up, false);
    if (hoist) {
      // R2.7b: the decomposition was done once per source (rotate_hoisted_raw); a1 + a4 reduce to a gathered inner product
      CUDA_OK(ctx, k_hoisted_keymac(k, d_items, L, E, P->beta, P->d_tmp_index, hoist->up, hoist->sstride, acc, (size_t)2 * E * N, nb,
                                    n_keys, hoist->n_sources, P->n_up));
    } else {
    if (fused_up) {
      CUDA_OK(ctx, k_intt_rows_only(k, d_items, nullptr, 0, true, y, (size_t)L * N, P->d_rows_in, L, nb));
      CUDA_OK(ctx, k_convert_cols(k, y, (size_t)L * N, P->d_groups_up, P->beta, P->n_src_up, P->d_scale_in, P->d_bc_up, P->d_rows_up,
                                  P->n_up, tmp, (size_t)P->n_up * N, nb, ctx->lazy_q, nullptr, P->d_bc_up_f64));
    } else {
      CUDA_OK(ctx, k_intt(k, d_items, nullptr, 0, true, y, (size_t)L * N, P->d_rows_in, L, P->d_scale_in, nb));
      CUDA_OK(ctx, k_ntt_cols_bconv(k, y, (size_t)L * N, P->d_bc_up, tmp, (size_t)P->n_up * N, P->d_rows_up, P->n_up, nb, L, ctx->lazy_q));
    }
    // a1 (pass 2) + a4: evk inner product
    CUDA_OK(ctx, k_ntt_rows_keymac(k, d_items, L, E, P->beta, P->d_tmp_index, tmp, (size_t)P->n_up * N, acc, (size_t)2 * E * N, nb, P->n_up, n_keys));
    }
    if (rescale_after) {
      // a5 + a8 merged: the limb the rescale drops is inverse-transformed with the special limbs; one column kernel and
      // one divide epilogue produce the rescaled ciphertext directly
      const int L1 = L - 1;
      CUDA_OK(ctx, k_intt_rows_only(k, d_items, acc, (size_t)2 * E * N, false, yP, (size_t)2 * npy * N, P->d_rows_p2, 2 * npy, nb,
                                    P->d_mul_pinv));
      CUDA_OK(ctx, k_convert_cols(k, yP, (size_t)2 * npy * N, P->d_groups_down2, 2, npy, P->d_scale_p2, P->d_bc_down, P->d_rows_down2,
                                  2 * L1, tmp2, (size_t)2 * L1 * N, nb, ctx->lazy_p, P->d_mul_pinv));
      CUDA_OK(ctx, k_ntt_rows_divide(k, d_items, tmp2, (size_t)2 * L1 * N, acc, (size_t)2 * E * N, false, P->d_mul_qlinv,
                                     P->d_rows_div2, 2 * L1, nb, P->d_mul_pinv));
      continue;
    }
    // a5: ModDown = inverse row pass of the special limbs, fused column kernel per component, divide epilogue in pass 2
    const bool fused_down = convert_cols_fits(ctx->logN, np, false);
    if (fused_down) {
      CUDA_OK(ctx, k_intt_rows_only(k, nullptr, acc, (size_t)2 * E * N, false, yP, (size_t)2 * np * N, P->d_rows_p, 2 * np, nb));
      CUDA_OK(ctx, k_convert_cols(k, yP, (size_t)2 * np * N, P->d_groups_down, 2, np, P->d_scale_p, P->d_bc_down, P->d_rows_down, 2 * L,
                                  tmp2, (size_t)2 * L * N, nb, ctx->lazy_p));
    } else {
      CUDA_OK(ctx, k_intt(k, nullptr, acc, (size_t)2 * E * N, false, yP, (size_t)2 * np * N, P->d_rows_p, 2 * np, P->d_scale_p, nb));
      CUDA_OK(ctx, k_ntt_cols_bconv(k, yP, (size_t)2 * np * N, P->d_bc_down, tmp2, (size_t)2 * L * N, P->d_rows_down, 2 * L, nb, 2 * np, ctx->lazy_p));
    }
    CUDA_OK(ctx, k_ntt_rows_divide(k, d_items, tmp2, (size_t)2 * L * N, acc, (size_t)2 * E * N, false, P->d_mul_pinv, P->d_rows_div, 2 * L, nb));
  }
  return FENC_OK;
}

fenc_status rescale_batch(fenc_ctx *ctx, int L, std::vector<BatchItem> &items) {
  if (items.empty()) return FENC_OK;
  if (L < 2) return fail(ctx, FENC_ERR_LEVEL, "rescale needs at least 2 limbs");
  LevelPlan *P = get_plan(ctx, L);
  if (!P) return fail(ctx, FENC_ERR_OOM, "level plan");
  const size_t N = ctx->N;
  const int L1 = L - 1;
  const size_t per = ((size_t)2 + 2 * L1) * N;
  size_t chunk = std::min(std::min(items.size(), GRID_Z_MAX), std::max<size_t>(1, WS_CAP / (per * 8)));
  u64 *ws = (u64 *)workspace(ctx, chunk * per * 8);
  if (!ws) return fail(ctx, FENC_ERR_OOM, "rescale workspace");
  u64 *yR = ws, *tmp2 = yR + chunk * 2 * N;
  const KCtx &k = ctx->k;
  for (size_t at = 0; at < items.size(); at += chunk) {
    const int nb = (int)std::min(chunk, items.size() - at);
    DescStage st(ctx);
    std::vector<BatchItem> part(items.begin() + at, items.begin() + at + nb);
    for (auto &it : part) it.ks_in = it.sub_in, it.add0 = it.add1 = nullptr, it.g = 1;
    st.add(part);
    const BatchItem *d_items = (const BatchItem *)st.commit();
    if (!d_items) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
    if (ctx->logN >= 12) {
      CUDA_OK(ctx, k_intt_rows_only(k, d_items, nullptr, 0, false, yR, 2 * N, P->d_rows_rs_in, 2, nb));
      CUDA_OK(ctx, k_convert_cols(k, yR, 2 * N, P->d_groups_rs, 2, 1, P->d_scale_rs, P->d_bc_rs, P->d_rows_rs_up, 2 * L1, tmp2,
                                  (size_t)2 * L1 * N, nb, ctx->lazy_q, nullptr, P->d_bc_rs_f64));
    } else {
      CUDA_OK(ctx, k_intt(k, d_items, nullptr, 0, false, yR, 2 * N, P->d_rows_rs_in, 2, P->d_scale_rs, nb));
      CUDA_OK(ctx, k_ntt_cols_bconv(k, yR, 2 * N, P->d_bc_rs, tmp2, (size_t)2 * L1 * N, P->d_rows_rs_up, 2 * L1, nb, 2, ctx->lazy_q));
    }
    CUDA_OK(ctx, k_ntt_rows_divide(k, d_items, tmp2, (size_t)2 * L1 * N, nullptr, 0, true, P->d_mul_qlinv, P->d_rows_rs_div, 2 * L1, nb));
  }
  return FENC_OK;
}

// Hoisted rotations (R2.7b): per source one inverse transform of c1 (no gather), ModUp with the forward column stages,
// and the forward row stages -> extended digits in NTT form; then per rotation the gathered inner product and ModDown.
fenc_status rotate_hoisted_raw(fenc_ctx *ctx, const fenc_keys *keys, int L, const std::vector<const u64 *> &src,
                               const std::vector<int> &src_of, const std::vector<int> &steps, const std::vector<u64 *> &out) {
  if (steps.empty()) return FENC_OK;
  LevelPlan *P = get_plan(ctx, L);
  if (!P) return fail(ctx, FENC_ERR_OOM, "level plan");
  const size_t N = ctx->N, LN = (size_t)L * N;
  // every key is looked up before anything is enqueued: nothing is written on FENC_ERR_NO_KEY
  std::vector<const u64 *> evk(steps.size(), nullptr);
  std::vector<int> red(steps.size());
  for (size_t i = 0; i < steps.size(); i++) {
    red[i] = ((steps[i] % ctx->n) + ctx->n) % ctx->n;
    if (red[i] == 0) continue;
    auto it = keys->evk.find(red[i]);
    if (it == keys->evk.end()) return fail(ctx, FENC_ERR_NO_KEY, "no rotation key for step %d", red[i]);
    evk[i] = it->second;
  }
  // sources are processed in chunks whose decompositions (y + extended digits) stay under the workspace budget, so a
  // large layer or batch costs more launches instead of FENC_ERR_OOM (the plain path chunks the same way in ks_batch)
  const size_t per_src = (LN + (size_t)P->n_up * N) * 8;
  const size_t ns_all = src.size();
  const size_t chunk = std::min<size_t>(std::min(ns_all, GRID_Z_MAX), std::max<size_t>(1, WS_CAP / per_src));
  std::vector<std::vector<size_t>> rots_of(ns_all);
  for (size_t i = 0; i < steps.size(); i++) rots_of[src_of[i]].push_back(i);
  for (size_t s0 = 0; s0 < ns_all; s0 += chunk) {
    Scope sc(ctx);
    const int ns = (int)std::min(chunk, ns_all - s0);
    u64 *y = sc.alloc<u64>((size_t)ns * LN), *up = sc.alloc<u64>((size_t)ns * P->n_up * N);
    if (!y || !up) return fail(ctx, FENC_ERR_OOM, "hoisted decomposition (%d sources)", ns);
    {
      DescStage st(ctx);
      std::vector<BatchItem> sitems(ns);
      for (int i = 0; i < ns; i++) sitems[i] = BatchItem{}, sitems[i].ks_in = src[s0 + i] + LN, sitems[i].g = 1;
      st.add(sitems);
      const BatchItem *d_src = (const BatchItem *)st.commit();
      if (!d_src) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
      const KCtx &k = ctx->k;
      if (convert_cols_fits(ctx->logN, P->n_src_up, false)) {
        CUDA_OK(ctx, k_intt_rows_only(k, d_src, nullptr, 0, true, y, LN, P->d_rows_in, L, ns));
        CUDA_OK(ctx, k_convert_cols(k, y, LN, P->d_groups_up, P->beta, P->n_src_up, P->d_scale_in, P->d_bc_up, P->d_rows_up, P->n_up, up,
                                    (size_t)P->n_up * N, ns, ctx->lazy_q, nullptr, P->d_bc_up_f64));
      } else {
        CUDA_OK(ctx, k_intt(k, d_src, nullptr, 0, true, y, LN, P->d_rows_in, L, P->d_scale_in, ns));
        CUDA_OK(ctx, k_ntt_cols_bconv(k, y, LN, P->d_bc_up, up, (size_t)P->n_up * N, P->d_rows_up, P->n_up, ns, L, ctx->lazy_q));
      }
      CUDA_OK(ctx, k_ntt_rows_only(k, up, (size_t)P->n_up * N, P->d_rows_up, P->n_up, ns));
    }
    std::vector<BatchItem> items;
    for (int si = 0; si < ns; si++)
      for (size_t i : rots_of[s0 + si]) {
        const u64 *in = src[s0 + si];
        if (red[i] == 0) {
          CUDA_OK(ctx, cudaMemcpyAsync(out[i], in, 2 * LN * 8, cudaMemcpyDeviceToDevice, ctx->stream));
          continue;
        }
        BatchItem b{};
        b.ks_in = in + LN, b.out = out[i], b.evk = evk[i], b.add0 = in, b.g = galois_elt(ctx, red[i]), b.pad = (u32)si;
        items.push_back(b);
      }
    HoistUp h{up, (size_t)P->n_up * N, ns};
    fenc_status st = ks_batch(ctx, L, items, false, &h);
    if (st != FENC_OK) return st;
  }
  return FENC_OK;
}

// Rot(in[i], steps[i]) -> out[i]; all at level L (Eq. 1; R2.7: automorphism first)
fenc_status rotate_raw(fenc_ctx *ctx, const fenc_keys *keys, int L, const std::vector<const u64 *> &in,
                       const std::vector<int> &steps, const std::vector<u64 *> &out) {
  std::vector<BatchItem> items;
  const size_t LN = (size_t)L * ctx->N;
  for (size_t i = 0; i < in.size(); i++) {
    int r = ((steps[i] % ctx->n) + ctx->n) % ctx->n;
    if (r == 0) {
      CUDA_OK(ctx, cudaMemcpyAsync(out[i], in[i], 2 * LN * 8, cudaMemcpyDeviceToDevice, ctx->stream));
      continue;
    }
    auto it = keys->evk.find(r);
    if (it == keys->evk.end()) return fail(ctx, FENC_ERR_NO_KEY, "no rotation key for step %d", r);
    BatchItem b{};
    b.ks_in = in[i] + LN, b.sub_in = nullptr, b.out = out[i], b.evk = it->second, b.add0 = in[i], b.add1 = nullptr;
    b.g = galois_elt(ctx, r);
    items.push_back(b);
  }
  return ks_batch(ctx, L, items);
}
