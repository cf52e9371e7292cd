// fenc_static.cu -- fenc_rescale_static: the rescale (a8) for callers that cannot allocate (CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc).  Same three kernels and the same per-level tables as fenc_rescale
// (rescale_batch in fenc_ctx.cu); what differs is where the intermediates and the one-item descriptor live: in a
// file-scope device array of FENC_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit, instead of the
// context's grow-only workspace and descriptor ring.
//
// The array's NAME is only a host-side stand-in in host code: its device address comes from cudaGetSymbolAddress, taken
// once per device at set-up (fenc_rescale_static_prepare) with that device current, and that address is what the kernels
// of the other translation units receive.  Device code in THIS file names the array directly (write_item_kernel).
//
// Sharing: every call on a device uses the same array and finds the previous call's contents in it.  Nothing has to start
// at zero: the descriptor is rewritten by every call, the inverse row pass writes all 2 N words of yR before the column
// kernel reads them, and the column kernel writes all 2 (L-1) N words of tmp before the divide pass reads them.  Calls
// enqueued on one stream are ordered; calls that overlap on the GPU (two contexts or streams on one device) RACE.
#include <cstdio>

#include "fenc_ctx.h"

#define STATIC_HDR_BYTES 256  // the BatchItem of the call
static __device__ __align__(256) unsigned char g_static_scratch[FENC_STATIC_SCRATCH_BYTES];

#define FENC_MAX_DEVICES 64
static u64 *g_scratch_addr[FENC_MAX_DEVICES];  // device address of g_static_scratch per device ordinal (0 = not resolved)

// the call's descriptor, from kernel arguments into the header of the array (no host-to-device copy, no staging buffer)
__global__ void write_item_kernel(BatchItem it) { *reinterpret_cast<BatchItem *>(g_static_scratch) = it; }

static size_t static_need_bytes(const fenc_ctx *ctx, int L) {
  return (size_t)STATIC_HDR_BYTES + ((size_t)2 + 2 * (size_t)(L - 1)) * (size_t)ctx->N * sizeof(u64);
}

// Set-up (may allocate: the per-level tables).  Resolves the array's device address for the context's device.
extern "C" fenc_status fenc_rescale_static_prepare(fenc_ctx *ctx, uint32_t L) {
  if (!ctx) return FENC_ERR_INVALID_ARG;
  if (L < 2 || (int)L > ctx->nq) return fail(ctx, FENC_ERR_LEVEL, "rescale needs 2 <= L <= %d limbs, got %u", ctx->nq, L);
  if (ctx->device < 0 || ctx->device >= FENC_MAX_DEVICES) return fail(ctx, FENC_ERR_DEVICE, "device ordinal %d", ctx->device);
  if (static_need_bytes(ctx, (int)L) > FENC_STATIC_SCRATCH_BYTES)
    return fail(ctx, FENC_ERR_INVALID_ARG, "fenc_rescale_static needs %zu bytes of scratch at N=%d, L=%u; the static array holds %zu",
                static_need_bytes(ctx, (int)L), ctx->N, L, (size_t)FENC_STATIC_SCRATCH_BYTES);
  if (!g_scratch_addr[ctx->device]) {
    int cur = -1;
    CUDA_OK(ctx, cudaGetDevice(&cur));
    if (cur != ctx->device) CUDA_OK(ctx, cudaSetDevice(ctx->device));  // the symbol is looked up with ITS device current
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (cur != ctx->device) cudaSetDevice(cur);
    if (e != cudaSuccess || !p) return fail(ctx, FENC_ERR_CUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
    g_scratch_addr[ctx->device] = (u64 *)p;
  }
  if (!get_plan(ctx, (int)L)) return fail(ctx, FENC_ERR_OOM, "level plan");
  return FENC_OK;
}

// The allocation-free call: out := rescale(in).  No cudaMalloc / cudaFree / allocator callback / event or stream creation.
extern "C" fenc_status fenc_rescale_static(fenc_ctx *ctx, const fenc_ct *in, fenc_ct *out) {
  if (!ctx || !in || !out) return FENC_ERR_INVALID_ARG;
  const int L = in->L, L1 = L - 1;
  if (L < 2) return fail(ctx, FENC_ERR_LEVEL, "rescale at the last level");
  if (in->ctx != ctx || out->ctx != ctx || out->L != L1 || out->d == in->d)
    return fail(ctx, FENC_ERR_MISMATCH, "fenc_rescale_static: out must be another ciphertext of this context at %d limbs (it has %d)", L1, out->L);
  const size_t need = static_need_bytes(ctx, L);
  if (need > FENC_STATIC_SCRATCH_BYTES)
    return fail(ctx, FENC_ERR_INVALID_ARG, "fenc_rescale_static needs %zu bytes of scratch at N=%d, L=%d; the static array holds %zu",
                need, ctx->N, L, (size_t)FENC_STATIC_SCRATCH_BYTES);
  if (ctx->k.prof) return fail(ctx, FENC_ERR_INVALID_ARG, "fenc_rescale_static: the profiling hooks create events; disable fenc_profile_enable");
  u64 *base = (ctx->device >= 0 && ctx->device < FENC_MAX_DEVICES) ? g_scratch_addr[ctx->device] : nullptr;
  auto pit = ctx->plans.find(L);
  if (!base || pit == ctx->plans.end())
    return fail(ctx, FENC_ERR_INVALID_ARG, "fenc_rescale_static: call fenc_rescale_static_prepare(ctx, %d) at set-up", L);
  const LevelPlan *P = pit->second.get();
  const size_t N = ctx->N;
  const BatchItem *d_item = (const BatchItem *)base;
  u64 *yR = base + STATIC_HDR_BYTES / sizeof(u64), *tmp = yR + 2 * N;
  BatchItem it{};
  it.ks_in = in->d, it.sub_in = in->d, it.out = out->d, it.g = 1;
  write_item_kernel<<<1, 1, 0, ctx->stream>>>(it);
  ctx->launches++;
  CUDA_OK(ctx, cudaGetLastError());
  const KCtx &k = ctx->k;
  if (ctx->logN >= 12) {
    CUDA_OK(ctx, k_intt_rows_only(k, d_item, nullptr, 0, false, yR, 2 * N, P->d_rows_rs_in, 2, 1));
    CUDA_OK(ctx, k_convert_cols(k, yR, 2 * N, P->d_groups_rs, 2, 1, P->d_scale_rs, P->d_bc_rs, P->d_rows_rs_up, 2 * L1, tmp,
                                (size_t)2 * L1 * N, 1, ctx->lazy_q, nullptr, P->d_bc_rs_f64));
  } else {
    CUDA_OK(ctx, k_intt(k, d_item, nullptr, 0, false, yR, 2 * N, P->d_rows_rs_in, 2, P->d_scale_rs, 1));
    CUDA_OK(ctx, k_ntt_cols_bconv(k, yR, 2 * N, P->d_bc_rs, tmp, (size_t)2 * L1 * N, P->d_rows_rs_up, 2 * L1, 1, 2, ctx->lazy_q));
  }
  CUDA_OK(ctx, k_ntt_rows_divide(k, d_item, tmp, (size_t)2 * L1 * N, nullptr, 0, true, P->d_mul_qlinv, P->d_rows_rs_div, 2 * L1, 1));
  out->scale = in->scale / (double)ctx->mod[L1];
  return FENC_OK;
}
