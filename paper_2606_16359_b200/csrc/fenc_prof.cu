// fenc_prof.cu -- optional per-kernel-class timing (CUDA events on the launching stream) and algorithmic-byte
// accounting, read by bench.py for the roofline object.  Off by default: no events are recorded unless enabled.
#include <cuda_runtime.h>

#include <vector>

#include "fenc_ctx.h"
#include "fenc_device.cuh"

struct ProfRec { int id; cudaEvent_t a, b; };
struct Prof {
  std::vector<ProfRec> recs;
  std::vector<cudaEvent_t> pool;
  double ms[K_COUNT] = {0}, bytes[K_COUNT] = {0}, ops[K_COUNT] = {0};
  u64 count[K_COUNT] = {0};
  cudaEvent_t get() {
    if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
    cudaEvent_t e; cudaEventCreate(&e); return e;
  }
};
void prof_begin(Prof *p, void *stream, int id, double alg_bytes, double alg_butterflies) {
  ProfRec r{id, p->get(), p->get()};
  p->bytes[id] += alg_bytes, p->ops[id] += alg_butterflies, p->count[id]++;
  cudaEventRecord(r.a, (cudaStream_t)stream);
  p->recs.push_back(r);
}
void prof_end(Prof *p, void *stream) { cudaEventRecord(p->recs.back().b, (cudaStream_t)stream); }

static const char *kNames[K_COUNT] = {"intt_rowpass", "intt_colpass", "ntt_colpass", "ntt_colpass_bconv", "ntt_rowpass",
                                      "ntt_rows_keymac", "ntt_rows_divide", "mac", "add_many", "rowop", "sample", "smac"};

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
extern "C" fenc_status fenc_profile_read(fenc_ctx *ctx, double *ms, uint64_t *launches, double *alg_bytes, double *alg_butterflies,
                                         int reset) {
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
    if (alg_butterflies) alg_butterflies[i] = p->ops[i];
    if (reset) p->ms[i] = p->bytes[i] = p->ops[i] = 0, p->count[i] = 0;
  }
  return FENC_OK;
}

// ------------------------------------------------------------------------------------------------ integer-pipe peaks
// Measured denominators for the "alu" roofline: (1) dependency-free 32-bit IMAD chains, all SMs;
// (2) the forward lazy Shoup butterfly of fenc_device.cuh on registers only (no memory traffic): the ceiling of any NTT
// kernel built from this butterfly.
__global__ void __launch_bounds__(256) imad_peak_kernel(u32 *out, int iters) {
  u32 x[8];
#pragma unroll
  for (int k = 0; k < 8; k++) x[k] = threadIdx.x + k;
  const u32 a = 2654435761u + blockIdx.x, b = 40503u;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int k = 0; k < 8; k++) x[k] = x[k] * a + b;
  }
  u32 s = 0;
#pragma unroll
  for (int k = 0; k < 8; k++) s ^= x[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(256) butterfly_peak_kernel(u64 *out, u64 q, u64 w, u64 ws, int iters) {
  u64 x[8];
#pragma unroll
  for (int k = 0; k < 8; k++) x[k] = (threadIdx.x * 8 + k + blockIdx.x) % q;
  const u64 q2 = q + q;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int s = 2; s >= 0; s--) {
#pragma unroll
      for (int k = 0; k < 8; k++) {
        if (k & (1 << s)) continue;
        const int k2 = k | (1 << s);
        const u64 T = shoup_lazy(x[k2], w, ws, q);
        const u64 X = x[k];
        x[k] = X + T;
        x[k2] = X - T + q2;
      }
    }
#pragma unroll
    for (int k = 0; k < 8; k++) x[k] = csub(x[k] & ((1ull << 58) - 1), q2);  // keep the lazy values bounded between rounds
  }
  u64 s = 0;
#pragma unroll
  for (int k = 0; k < 8; k++) s ^= x[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
// the fp64 register round of fenc_device.cuh (moduli below 2^45): convert in, 12 butterflies, convert out
__global__ void __launch_bounds__(256) butterfly_f64_peak_kernel(u64 *out, u64 q, u64 qinv_bits, u64 c_bits, u64 cq_bits, int iters) {
  u64 y[8];
#pragma unroll
  for (int k = 0; k < 8; k++) y[k] = (threadIdx.x * 8 + k + blockIdx.x) % q;
  const F64Mod fm = f64mod(q, qinv_bits);
  const double c = __longlong_as_double((long long)c_bits), cq = __longlong_as_double((long long)cq_bits);
  const double off = __dadd_rn(fm.q, 4503599627370496.0);
  for (int it = 0; it < iters; it++) {
    double x[8];
#pragma unroll
    for (int k = 0; k < 8; k++) x[k] = u2d52(y[k]);
#pragma unroll
    for (int s = 2; s >= 0; s--) {
#pragma unroll
      for (int k = 0; k < 8; k++) {
        if (k & (1 << s)) continue;
        const int k2 = k | (1 << s);
        const double X = x[k], T = mulmod_dd(x[k2], c, cq, fm);
        x[k] = __dadd_rn(X, T);
        x[k2] = __dadd_rn(X, -T);
      }
    }
#pragma unroll
    for (int k = 0; k < 8; k++) y[k] = d2u_off(reduce_dd(x[k], fm), off);  // bounded between rounds, like the inverse round
  }
  u64 s = 0;
#pragma unroll
  for (int k = 0; k < 8; k++) s ^= y[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
// the scalar MAC's inner operation (fenc_elem.cu smac_kernel, the 2 x 25-bit split mode ordinary weights run in) on
// registers only: per term two ciphertext words are split in two pieces each (4 conversions) and multiplied into 8 x 2 x 2
// partial sums by DFMA -- 16 multiply-accumulates for 32 DFMA --, the sums reduced every 32 terms
__global__ void __launch_bounds__(256, 2) smac_peak_kernel(u64 *out, u64 q, u64 qinv_bits, u64 c_bits, u64 cq_bits, int iters) {
  const F64Mod fm = f64mod(q, qinv_bits);
  double sp[8][2][2], kd[8];
  u64 x0 = (threadIdx.x * 7919u + blockIdx.x) % q, x1 = (threadIdx.x * 104729u + blockIdx.x) % q;
#pragma unroll
  for (int i = 0; i < 8; i++) {
    kd[i] = 1048573.0 - 37.0 * i;  // eight small multipliers, as round(v 2^25) of ordinary weights
    sp[i][0][0] = sp[i][0][1] = sp[i][1][0] = sp[i][1][1] = 0.0;
  }
  for (int it = 0; it < iters; it++) {
#pragma unroll 4
    for (int u = 0; u < 32; u++) {
      const double a0 = __hiloint2double(0x43300000, (int)((u32)x0 & 0x1FFFFFFu)) - 4503599627370496.0;
      const double a1 = __hiloint2double(0x43300000, (int)(u32)(x0 >> 25)) - 4503599627370496.0;
      const double b0 = __hiloint2double(0x43300000, (int)((u32)x1 & 0x1FFFFFFu)) - 4503599627370496.0;
      const double b1 = __hiloint2double(0x43300000, (int)(u32)(x1 >> 25)) - 4503599627370496.0;
#pragma unroll
      for (int i = 0; i < 8; i++) {
        sp[i][0][0] = __fma_rn(a0, kd[i], sp[i][0][0]), sp[i][0][1] = __fma_rn(a1, kd[i], sp[i][0][1]);
        sp[i][1][0] = __fma_rn(b0, kd[i], sp[i][1][0]), sp[i][1][1] = __fma_rn(b1, kd[i], sp[i][1][1]);
      }
      x0 += 0x9E3779B1ull, x1 += 0x85EBCA77ull;  // a new ciphertext word per term
      x0 &= 0x3FFFFFFFFFFFFull, x1 &= 0x3FFFFFFFFFFFFull;  // below 2^50
    }
#pragma unroll
    for (int i = 0; i < 8; i++)
      sp[i][0][0] = reduce_dd(sp[i][0][0], fm), sp[i][0][1] = reduce_dd(sp[i][0][1], fm), sp[i][1][0] = reduce_dd(sp[i][1][0], fm),
      sp[i][1][1] = reduce_dd(sp[i][1][1], fm);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += sp[i][0][0] + sp[i][0][1] + sp[i][1][0] + sp[i][1][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = (u64)__double_as_longlong(s) ^ c_bits ^ cq_bits;
}
extern "C" fenc_status fenc_measure_smac_peak(fenc_ctx *ctx, double *mulaccs_per_s) {
  if (!ctx || !mulaccs_per_s) return FENC_ERR_INVALID_ARG;
  const int blocks = 148 * 8, iters = 256;
  u64 *buf = dalloc_t<u64>(ctx, (size_t)blocks * 256);
  if (!buf) return fail(ctx, FENC_ERR_OOM, "peak buffer");
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0), cudaEventCreate(&e1);
  float ms = 0;
  const u64 q = ctx->mod[0], w = ctx->psi[0];
  const u64 qinv = fh::double_bits(1.0 / (double)q), cb = fh::double_bits((double)w), cqb = fh::double_bits((double)((long double)w / (long double)q));
  for (int rep = 0; rep < 2; rep++) {
    cudaEventRecord(e0, ctx->stream);
    smac_peak_kernel<<<blocks, 256, 0, ctx->stream>>>(buf, q, qinv, cb, cqb, iters);
    (void)cqb;
    cudaEventRecord(e1, ctx->stream);
    CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    cudaEventElapsedTime(&ms, e0, e1);
  }
  *mulaccs_per_s = (double)blocks * 256 * 16.0 * 32.0 * iters / (ms * 1e-3);
  cudaEventDestroy(e0), cudaEventDestroy(e1);
  dfree(ctx, buf);
  ctx->launches += 2;
  return FENC_OK;
}
extern "C" fenc_status fenc_measure_alu_peak(fenc_ctx *ctx, double *imad_lane_ops_per_s, double *butterflies_per_s) {
  if (!ctx || !imad_lane_ops_per_s || !butterflies_per_s) return FENC_ERR_INVALID_ARG;
  const int blocks = 148 * 8, iters = 4096;
  u64 *buf = dalloc_t<u64>(ctx, (size_t)blocks * 256);
  if (!buf) return fail(ctx, FENC_ERR_OOM, "peak buffer");
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0), cudaEventCreate(&e1);
  float ms = 0;
  const u64 q = ctx->mod[0], w = ctx->psi[0], ws = fh::shoup(w, q);
  for (int rep = 0; rep < 2; rep++) {  // first repetition warms up
    cudaEventRecord(e0, ctx->stream);
    imad_peak_kernel<<<blocks, 256, 0, ctx->stream>>>((u32 *)buf, iters);
    cudaEventRecord(e1, ctx->stream);
    CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    cudaEventElapsedTime(&ms, e0, e1);
  }
  *imad_lane_ops_per_s = (double)blocks * 256 * 8.0 * iters / (ms * 1e-3);
  for (int rep = 0; rep < 2; rep++) {
    cudaEventRecord(e0, ctx->stream);
    butterfly_peak_kernel<<<blocks, 256, 0, ctx->stream>>>(buf, q, w, ws, iters / 8);
    cudaEventRecord(e1, ctx->stream);
    CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    cudaEventElapsedTime(&ms, e0, e1);
  }
  *butterflies_per_s = (double)blocks * 256 * 12.0 * (iters / 8) / (ms * 1e-3);
  if (fh::f64_modulus(q, ctx->logN)) {  // this context's butterflies of q_0 run on the FP64 pipe: report the faster of the two ceilings
    const u64 qinv = fh::double_bits(1.0 / (double)q), cb = fh::double_bits((double)w), cqb = fh::double_bits((double)((long double)w / (long double)q));
    for (int rep = 0; rep < 2; rep++) {
      cudaEventRecord(e0, ctx->stream);
      butterfly_f64_peak_kernel<<<blocks, 256, 0, ctx->stream>>>(buf, q, qinv, cb, cqb, iters / 8);
      cudaEventRecord(e1, ctx->stream);
      CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
      cudaEventElapsedTime(&ms, e0, e1);
    }
    const double f = (double)blocks * 256 * 12.0 * (iters / 8) / (ms * 1e-3);
    if (f > *butterflies_per_s) *butterflies_per_s = f;
    ctx->launches += 2;
  }
  cudaEventDestroy(e0), cudaEventDestroy(e1);
  dfree(ctx, buf);
  ctx->launches += 4;
  return FENC_OK;
}
