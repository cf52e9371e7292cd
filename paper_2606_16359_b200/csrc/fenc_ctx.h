// fenc_ctx.h -- host-side objects behind the opaque handles of include/fenc.h (library private).
#pragma once
#include <cuda_runtime.h>

#include <array>
#include <deque>
#include <map>
#include <memory>
#include <string>
#include <vector>

#include "fenc_internal.h"

#define FENC_DESC_SLOTS 32  // pinned 1 MiB slots feeding the descriptor buffer: how many batches the host may run ahead

// Per-level (number of ciphertext limbs L) tables of the hybrid key switch and of the rescale (R2.6, R2.8).
struct LevelPlan {
  int L, E, beta, n_up;      // E = L + np target rows; n_up = rows of the ModUp temp = beta*E - L
  // key switch
  RowDesc *d_rows_in;        // [L] iNTT of the polynomial to switch (row t, modulus t)
  ShoupC *d_scale_in;        // [L] N^-1 * Qhat_{j,t}^-1 mod q_t (the ModUp pre-scaling folded into the iNTT)
  RowDesc *d_rows_up;        // [n_up] ModUp + forward pass 1 job rows
  u64 *d_bc_up;              // Montgomery-form (Q_j / q_i mod t) constants, indexed by RowDesc.aux2 + s
  ShoupC *d_bc_up_f64 = nullptr, *d_bc_rs_f64 = nullptr;  // the same constants (plain) as fp64 pairs {c, c/t}
  int *d_tmp_index;          // [beta*E] -> row of the ModUp temp or -1
  RowDesc *d_rows_p;         // [2 np] iNTT of the special limbs of both accumulators
  ShoupC *d_scale_p;         // [2 np] N^-1 * Phat_i^-1 mod p_i
  RowDesc *d_rows_down;      // [2L] ModDown conversion + forward pass 1
  u64 *d_bc_down;            // [L*np] (P / p_i mod q_t) Montgomery form
  RowDesc *d_rows_div;       // [2L] forward pass 2 + divide epilogue
  ShoupC *d_mul_pinv;        // [A] P^-1 mod q_t
  // rescale (drop limb L-1)
  RowDesc *d_rows_rs_in;     // [2]
  ShoupC *d_scale_rs;        // [2] N^-1 mod q_{L-1}
  RowDesc *d_rows_rs_up;     // [2(L-1)]
  u64 *d_bc_rs;              // [L-1] 2^64 mod q_t (i.e. "mod t")
  RowDesc *d_rows_rs_div;    // [2(L-1)]
  ShoupC *d_mul_qlinv;       // [A] q_{L-1}^-1 mod q_t
  // ModDown merged with the rescale that follows a relinearisation (bit-identical to the two in turn):
  // the dropped limb l = L-1 joins the special limbs in the inverse pass and the column kernel, targets are t < L-1
  RowDesc *d_rows_p2 = nullptr;     // [2 (np+1)] special limbs + the combined limb l (aux = 1, aux2 = component)
  ShoupC *d_scale_p2 = nullptr;     // [2 (np+1)]
  ConvGroup *d_groups_down2 = nullptr;  // [2], pad = {1, l}
  RowDesc *d_rows_down2 = nullptr;  // [2 (L-1)]
  RowDesc *d_rows_div2 = nullptr;   // [2 (L-1)]
  // fused column kernel (fenc_ntt.cu convert_cols_kernel): conversion groups per digit / per component
  ConvGroup *d_groups_up = nullptr, *d_groups_down = nullptr, *d_groups_rs = nullptr;
  int n_src_up = 0;          // longest digit in use
  // plain transforms of a whole ciphertext [2][L][N]
  RowDesc *d_rows_ct;        // [2L]
  ShoupC *d_scale_ct;        // [2L] N^-1 mod q_t
  std::vector<void *> owned;
};

struct LinGraph;  // fenc_conv.cu: operation graph of a linear layer (conv or fc)

// one slot of the staging queue behind fenc_ct_import_async: the copy stream fills it, the context's stream transforms it.
// The queue is first-in first-out and GROWS while its oldest slot is still waiting for its transform, up to
// FENC_STAGE_BYTES_MAX (environment FENC_STAGE_MAX_MB): a serving loop uploads request i+2 while request i+1 computes, and
// the transforms of those uploads are enqueued BEHIND request i+1's kernels, so a queue shorter than one request's inputs
// stalls the bus until request i+1 has finished (measured on config 4: 8 slots of 31 MB for 6 GB of inputs left the
// compute stream idle for about 100 ms per request).
#define FENC_STAGE_BYTES_MAX ((size_t)8 << 30)
struct StageSlot {
  u64 *d = nullptr;
  size_t bytes = 0;
  cudaEvent_t copied = nullptr, consumed = nullptr;
};

struct fenc_ctx {
  int logN = 0, N = 0, n = 0, nq = 0, np = 0, A = 0, dlen = 0, beta_max = 0;
  std::vector<u64> mod, psi;  // q_0..q_{nq-1}, p_0..p_{np-1}
  double default_scale = 0;
  int device = 0;
  cudaStream_t stream = nullptr;
  void *(*dev_alloc)(size_t, void *) = nullptr;
  void (*dev_free)(void *, void *) = nullptr;
  void *user = nullptr;
  ModConst *d_mods = nullptr;
  ShoupC *d_tw_fwd = nullptr, *d_tw_inv = nullptr;
  RowDesc *d_ident_rows = nullptr;  // [A] row r <-> modulus r
  ShoupC *d_ninv = nullptr;         // [A] N^-1 mod each modulus
  int *d_ident_mod = nullptr;       // [2A] 0..A-1, 0..A-1
  KCtx k{};
  u64 launches = 0, dev_bytes = 0;
  int max_lazy = 1;                 // floor(2^64 / max ciphertext modulus): terms per lazy 128-bit accumulation
  int lazy_q = 1, lazy_p = 1;       // the same for base conversions out of the q limbs / the p limbs
  std::string err;
  std::map<int, std::unique_ptr<LevelPlan>> plans;
  std::map<void *, size_t> live;    // device pointer -> bytes (accounting)
  std::map<size_t, std::vector<void *>> pool;  // released blocks by size, reused by dalloc (fenc_ctx.cu)
  size_t pool_bytes = 0;
  void *ws = nullptr;               // grow-only key-switch workspace
  size_t ws_bytes = 0;
  void *desc_buf = nullptr;         // device staging for per-call descriptor arrays
  size_t desc_bytes = 0;
  void *desc_pinned = nullptr;      // ring of pinned host slots feeding desc_buf
  cudaEvent_t desc_ev[FENC_DESC_SLOTS] = {};
  bool desc_used[FENC_DESC_SLOTS] = {};
  unsigned desc_next = 0;
  std::map<std::string, std::shared_ptr<LinGraph>> graphs;
  cudaStream_t copy_stream = nullptr;  // host -> staging copies of fenc_ct_import_async (created on first use)
  std::deque<StageSlot> stage;         // oldest use first
  size_t stage_bytes = 0, stage_max = 0;
  // fenc_ct_export_async: the inverse transform runs on the context's stream into a buffer of its own, the device -> host
  // copy on d2h_stream; the buffer returns to the pool once its copy has landed (export_drain)
  cudaStream_t d2h_stream = nullptr;
  cudaEvent_t export_ready = nullptr;  // re-recorded behind every export's transform; the copy stream waits for it
  struct PendingExport { void *buf; cudaEvent_t landed; };
  std::deque<PendingExport> exports;   // in issue order
  std::vector<cudaEvent_t> export_events;  // recycled `landed` events
  bool hoist_inner = false;            // fenc_set_hoisting: inner rotations of linear layers in the hoisted form (R2.7b)
};

// returns the staging buffers of exports whose copies have landed to the pool; block: wait for all of them
fenc_status export_drain(fenc_ctx *ctx, bool block);

struct fenc_keys {
  fenc_ctx *ctx;
  u64 seed;
  std::vector<int64_t> s;        // secret coefficients
  u64 *d_s_mont = nullptr;       // [A][N] NTT domain, Montgomery form
  std::map<int64_t, u64 *> evk;  // key id -> [beta_max][2][A][N] NTT domain, Montgomery form
};

struct fenc_pt {
  fenc_ctx *ctx;
  int L;
  double scale;
  std::vector<int64_t> coeffs;  // centred integer coefficients (A7: parity starts here)
  u64 *d_mont = nullptr;        // [L][N] NTT domain, Montgomery form (built on first use)
};

struct fenc_ct {
  fenc_ctx *ctx;
  int L;
  double scale;
  u64 *d;  // [2][L][N] NTT domain, canonical
};

struct fenc_wts {
  fenc_ctx *ctx;
  int L;
  double scale;
  size_t n;
  size_t n_unique = 0;
  std::vector<int> slot;  // weight index (fenc_wts_keys order) -> storage slot; identical plaintexts share one
  u64 *d_all = nullptr;  // [n_unique][L][N] NTT domain, Montgomery form
  // factored form (R2.9c): d_all holds the n_unique distinct MASK plaintexts, slot[i] the mask of weight i, and
  // d_k the per-weight integer multipliers, [n][L] 16-byte entries (fenc_internal.h k_smac)
  bool factored = false, k_fp64 = false;
  int k_mode = 0;        // fenc_internal.h k_smac: 0 integer, 1 fp64 residues, 2 / 3 signed multipliers (split modes)
  int k_lazy = 1;        // terms per exact partial sum in that mode
  ShoupC *d_k = nullptr;
};

// ---------------------------------------------------------------- helpers (fenc_ctx.cu)
fenc_status fail(fenc_ctx *ctx, fenc_status st, const char *fmt, ...);
#define CUDA_OK(ctx, expr)                                                                              \
  do {                                                                                                  \
    cudaError_t e__ = (cudaError_t)(expr);                                                              \
    if (e__ != cudaSuccess) return fail(ctx, FENC_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e__)); \
  } while (0)
void *dalloc(fenc_ctx *ctx, size_t bytes);
void dfree(fenc_ctx *ctx, void *p);
template <class T>
T *dalloc_t(fenc_ctx *ctx, size_t count) { return (T *)dalloc(ctx, count * sizeof(T)); }
// upload a host vector into plan-owned device memory
template <class T>
T *upload_owned(fenc_ctx *ctx, std::vector<void *> &owned, const std::vector<T> &v) {
  T *d = dalloc_t<T>(ctx, v.size() ? v.size() : 1);
  if (!d) return nullptr;
  if (!v.empty()) cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, ctx->stream);
  owned.push_back(d);
  return d;
}
LevelPlan *get_plan(fenc_ctx *ctx, int L);
void *workspace(fenc_ctx *ctx, size_t bytes);
// stage small host arrays into the context's descriptor buffer (one region per call site per batch)
struct DescStage {
  fenc_ctx *ctx;
  size_t off = 0;
  std::vector<char> host;
  explicit DescStage(fenc_ctx *c) : ctx(c) {}
  template <class T>
  size_t add(const std::vector<T> &v) {
    size_t o = (host.size() + 255) & ~(size_t)255;
    host.resize(o + v.size() * sizeof(T));
    if (!v.empty()) memcpy(host.data() + o, v.data(), v.size() * sizeof(T));
    return o;
  }
  // uploads; returns device base or nullptr
  char *commit();
};
fenc_ct *new_ct(fenc_ctx *ctx, int L, double scale);
extern "C" void fenc_ct_free(fenc_ct *ct);
// Scope-bound temporaries of one API call: device buffers are released when the call returns (the allocator is
// stream-ordered: torch's caching allocator on the context's stream, or cudaFree), and ciphertexts created for the
// outputs are released too unless the call succeeded (ok = true).
struct Scope {
  fenc_ctx *ctx;
  std::vector<void *> bufs;
  std::vector<fenc_ct *> cts;
  bool ok = false;
  explicit Scope(fenc_ctx *c) : ctx(c) {}
  Scope(const Scope &) = delete;
  ~Scope() {
    for (void *b : bufs) dfree(ctx, b);
    if (!ok)
      for (fenc_ct *c : cts) fenc_ct_free(c);
  }
  template <class T>
  T *alloc(size_t count) {
    T *p = dalloc_t<T>(ctx, count);
    if (p) bufs.push_back(p);
    return p;
  }
  fenc_ct *ct(int L, double scale) {
    fenc_ct *c = new_ct(ctx, L, scale);
    if (c) cts.push_back(c);
    return c;
  }
};
// batched key switch over items (all at level L): out = (ModDown(acc_0) + add0, ModDown(acc_1) + add1)
// rescale_after: the rescale is merged into the ModDown (needs both addends, g = 1, N >= 2^12): out is [2][L-1][N]
// hoisted rotations (R2.7b): the extended digits of the sources' c1 in NTT form, [n_sources][n_up][N]; items[i].pad = source
struct HoistUp {
  const u64 *up;
  size_t sstride;
  int n_sources;
};
fenc_status ks_batch(fenc_ctx *ctx, int L, std::vector<BatchItem> &items, bool rescale_after = false, const HoistUp *hoist = nullptr);
// Rot(src[src_of[i]], steps[i]) -> out[i] with ONE decomposition (inverse NTT, ModUp, forward NTT) per source
fenc_status rotate_hoisted_raw(fenc_ctx *ctx, const fenc_keys *keys, int L, const std::vector<const u64 *> &src,
                               const std::vector<int> &src_of, const std::vector<int> &steps, const std::vector<u64 *> &out);
bool ks_can_merge_rescale(const fenc_ctx *ctx, int L);
// batched rescale: items[i].sub_in = input ct [2][L][N], items[i].out = [2][L-1][N]
fenc_status rescale_batch(fenc_ctx *ctx, int L, std::vector<BatchItem> &items);
// rotation items for (in, step) pairs; step 0 handled by a device copy
fenc_status rotate_raw(fenc_ctx *ctx, const fenc_keys *keys, int L, const std::vector<const u64 *> &in,
                       const std::vector<int> &steps, const std::vector<u64 *> &out);
u32 galois_elt(const fenc_ctx *ctx, int step);
fenc_status pt_device(fenc_ctx *ctx, fenc_pt *pt);  // ensure pt->d_mont
// Builds the grouped MAC launch from per-output term lists (ct pointer, pt pointer) and enqueues it.
struct MacJob {
  std::vector<std::vector<std::pair<const u64 *, const u64 *>>> terms;  // per output
  std::vector<u64 *> outs;
};
fenc_status run_mac(fenc_ctx *ctx, const MacJob &job, int L);
// the same for factored weights: per output a list of (ciphertext, weight index, mask plaintext), mask-major
struct SmacTerm {
  const u64 *ct;
  int w;
  const u64 *mask;
};
struct SmacJob {
  std::vector<std::vector<SmacTerm>> terms;  // per output, sorted so that equal masks are consecutive
  std::vector<u64 *> outs;
};
fenc_status run_smac(fenc_ctx *ctx, const SmacJob &job, const fenc_wts *W, int L);
double mac_alg_bytes(fenc_ctx *ctx, const std::vector<const u64 *> &tc, const std::vector<const u64 *> &tp, size_t n_out, int L);
fenc_status coeffs_to_mont(fenc_ctx *ctx, const int64_t *coeffs_host, int L, u64 *d_out);
