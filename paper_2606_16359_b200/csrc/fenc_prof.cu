// fenc_prof.cu -- optional per-kernel-class timing (CUDA events on the launching stream) and algorithmic-byte
// accounting, read by bench.py for the roofline object.  Off by default: no events are recorded unless enabled.
#include <cuda_runtime.h>

#include <vector>

#include "fenc_ctx.h"

struct ProfRec { int id; cudaEvent_t a, b; };
struct Prof {
  std::vector<ProfRec> recs;
  std::vector<cudaEvent_t> pool;
  double ms[K_COUNT] = {0}, bytes[K_COUNT] = {0};
  u64 count[K_COUNT] = {0};
  cudaEvent_t get() {
    if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
    cudaEvent_t e; cudaEventCreate(&e); return e;
  }
};
void prof_begin(Prof *p, void *stream, int id, double alg_bytes) {
  ProfRec r{id, p->get(), p->get()};
  p->bytes[id] += alg_bytes, p->count[id]++;
  cudaEventRecord(r.a, (cudaStream_t)stream);
  p->recs.push_back(r);
}
void prof_end(Prof *p, void *stream) { cudaEventRecord(p->recs.back().b, (cudaStream_t)stream); }

static const char *kNames[K_COUNT] = {"intt_rowpass", "intt_colpass", "ntt_colpass", "ntt_colpass_bconv", "ntt_rowpass",
                                      "ntt_rows_keymac", "ntt_rows_divide", "mac", "add_many", "rowop", "sample"};

extern "C" fenc_status fenc_profile_enable(fenc_ctx *ctx, int on) {
  if (!ctx) return FENC_ERR_INVALID_ARG;
  cudaStreamSynchronize(ctx->stream);
  if (on && !ctx->k.prof) ctx->k.prof = new Prof();
  if (!on && ctx->k.prof) {
    for (auto &r : ctx->k.prof->recs) cudaEventDestroy(r.a), cudaEventDestroy(r.b);
    for (auto e : ctx->k.prof->pool) cudaEventDestroy(e);
    delete ctx->k.prof;
    ctx->k.prof = nullptr;
  }
  return FENC_OK;
}
extern "C" int fenc_profile_kernels(void) { return K_COUNT; }
extern "C" const char *fenc_profile_name(int id) { return id >= 0 && id < K_COUNT ? kNames[id] : ""; }
extern "C" fenc_status fenc_profile_read(fenc_ctx *ctx, double *ms, uint64_t *launches, double *alg_bytes, int reset) {
  if (!ctx || !ctx->k.prof) return FENC_ERR_INVALID_ARG;
  Prof *p = ctx->k.prof;
  CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  for (auto &r : p->recs) {
    float t = 0;
    cudaEventElapsedTime(&t, r.a, r.b);
    p->ms[r.id] += t;
    p->pool.push_back(r.a), p->pool.push_back(r.b);
  }
  p->recs.clear();
  for (int i = 0; i < K_COUNT; i++) {
    if (ms) ms[i] = p->ms[i];
    if (launches) launches[i] = p->count[i];
    if (alg_bytes) alg_bytes[i] = p->bytes[i];
    if (reset) p->ms[i] = p->bytes[i] = 0, p->count[i] = 0;
  }
  return FENC_OK;
}
