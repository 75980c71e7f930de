// C ABI of libsw (include/sw.h): host-side validation and dispatch.  Nothing here computes.
#include <stdarg.h>

#include <atomic>
#include <string.h>

#include "common.cuh"

namespace sw {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

int32_t fail(int32_t code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

static std::atomic<int> g_sms{0};

int32_t check_arch() {
  // per-thread cache keyed by the current device: no shared mutable state between host threads
  static thread_local int cached_dev = -1;
  static thread_local int32_t cached = SW_ERR_ARCH;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return fail(SW_ERR_ARCH, "no CUDA device is available (libsw has no CPU fallback)");
  }
  if (dev == cached_dev) return cached;
  int major = 0, minor = 0, sms = 0;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cached_dev = dev;
  g_sms.store(sms, std::memory_order_relaxed);
  cached = (major == 10) ? SW_OK : SW_ERR_ARCH;
  if (cached != SW_OK) set_error("device %d is sm_%d%d; libsw is built for sm_100a only", dev, major, minor);
  return cached;
}

int num_sms() { const int n = g_sms.load(std::memory_order_relaxed); return n > 0 ? n : 148; }

static std::atomic<uint64_t> g_launches{0};
void count_launch(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }
uint64_t launches() { return g_launches.load(std::memory_order_relaxed); }

int32_t check_launch(const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(SW_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
  return SW_OK;
}

int32_t validate_layout(const sw_layout* L) {
  SW_REQUIRE(L != nullptr, SW_ERR_INVALID_ARG, "layout is NULL");
  SW_REQUIRE(L->batch >= 0 && L->total_tokens >= 0 && L->total_blocks >= 0 && L->max_blocks >= 0,
             SW_ERR_INVALID_ARG, "layout: negative size");
  SW_REQUIRE(L->block == 64 || L->block == 128, SW_ERR_UNSUPPORTED, "layout: block size %d not in {64,128}",
             L->block);
  if (L->batch > 0) {
    SW_REQUIRE(L->cu_seqlens && L->cu_blocks && L->cu_sq, SW_ERR_INVALID_ARG, "layout: NULL cu_* array");
    SW_REQUIRE(L->max_blocks <= L->total_blocks, SW_ERR_INVALID_ARG, "layout: max_blocks > total_blocks");
    SW_REQUIRE((int64_t)L->total_blocks * L->block >= L->total_tokens, SW_ERR_INVALID_ARG,
               "layout: total_blocks*block < total_tokens");
  }
  return SW_OK;
}

int32_t validate_tensor(const sw_tensor* t, const char* name) {
  SW_REQUIRE(t != nullptr, SW_ERR_INVALID_ARG, "%s is NULL", name);
  SW_REQUIRE(t->ptr != nullptr, SW_ERR_INVALID_ARG, "%s.ptr is NULL", name);
  SW_REQUIRE(aligned16(t->ptr), SW_ERR_INVALID_ARG, "%s.ptr is not 16-byte aligned", name);
  SW_REQUIRE(t->dtype == SW_BF16 || t->dtype == SW_F32, SW_ERR_UNSUPPORTED, "%s.dtype %d", name, t->dtype);
  SW_REQUIRE(t->d == 64 || t->d == 128, SW_ERR_UNSUPPORTED, "%s.d = %d not in {64,128}", name, t->d);
  SW_REQUIRE(t->heads >= 1, SW_ERR_INVALID_ARG, "%s.heads = %d", name, t->heads);
  SW_REQUIRE(t->stride_tok % 8 == 0 && t->stride_head % 8 == 0 && t->stride_head >= t->d,
             SW_ERR_INVALID_ARG, "%s: strides must be multiples of 8 elements and stride_head >= d", name);
  return SW_OK;
}

static int32_t validate_sketch_params(const sw_tensor* x, const int32_t* cols, int r) {
  SW_REQUIRE(cols != nullptr, SW_ERR_INVALID_ARG, "cols is NULL");
  SW_REQUIRE(is_pow2(r) && r <= x->d, SW_ERR_INVALID_ARG, "r = %d must be a power of two <= d = %d", r, x->d);
  return SW_OK;
}

}  // namespace sw

using namespace sw;

#define SW_TRY(expr)                  \
  do {                                \
    int32_t _s = (expr);              \
    if (_s != SW_OK) return _s;       \
  } while (0)

static std::atomic<int32_t> g_prefill_kernel{SW_PREFILL_AUTO};   // process-wide test / benchmark switch
static thread_local int32_t g_prefill_used = 0;

extern "C" {

SW_API const char* sw_last_error(void) { return g_err; }
SW_API int32_t sw_version(void) { return SW_VERSION; }
SW_API uint64_t sw_launch_count(void) { return sw::launches(); }

SW_API int32_t sw_sketch(const sw_layout* L, const sw_tensor* x, const int8_t* signs, const int32_t* cols,
                  int32_t r, float scale, float* sketch, float* mean, sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_TRY(validate_tensor(x, "x"));
  SW_TRY(validate_sketch_params(x, cols, r));
  SW_REQUIRE(sketch != nullptr, SW_ERR_INVALID_ARG, "sketch is NULL");
  SW_TRY(check_arch());
  return launch_sketch(*L, *x, signs, cols, r, scale, sketch, mean, (cudaStream_t)stream);
}

SW_API int32_t sw_sketch_qk(const sw_layout* L, const sw_tensor* q, const sw_tensor* k, const int8_t* signs,
                     const int32_t* cols, int32_t r, float scale, float* qs, float* ks, float* qbar, float* kbar,
                     sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_TRY(validate_tensor(q, "q"));
  SW_TRY(validate_tensor(k, "k"));
  SW_REQUIRE(q->dtype == k->dtype && q->d == k->d, SW_ERR_UNSUPPORTED, "q / k dtype or head_dim differ");
  SW_TRY(validate_sketch_params(q, cols, r));
  SW_REQUIRE(qs != nullptr && ks != nullptr, SW_ERR_INVALID_ARG, "qs / ks is NULL");
  SW_TRY(check_arch());
  return launch_sketch_qk(*L, *q, *k, signs, cols, r, scale, qs, ks, qbar, kbar, (cudaStream_t)stream);
}

SW_API int32_t sw_copy_pool(const sw_layout* L, const sw_tensor* x, void* dst, float* sums, sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_TRY(validate_tensor(x, "x"));
  SW_REQUIRE(dst != nullptr && sums != nullptr, SW_ERR_INVALID_ARG, "dst / sums is NULL");
  SW_REQUIRE(aligned16(dst) && dst != x->ptr, SW_ERR_INVALID_ARG, "dst must be 16-byte aligned and not alias x");
  SW_TRY(check_arch());
  return launch_copy_pool(*L, *x, reinterpret_cast<__nv_bfloat16*>(dst), sums, (cudaStream_t)stream);
}

SW_API int32_t sw_sketch_from_pooled(const sw_layout* L, const float* sums, int32_t heads, int32_t d,
                              const int8_t* signs, const int32_t* cols, int32_t r, float scale, float* sketch,
                              float* mean, sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_REQUIRE(sums != nullptr && sketch != nullptr && cols != nullptr, SW_ERR_INVALID_ARG, "sums / sketch / cols is NULL");
  SW_REQUIRE(d == 64 || d == 128, SW_ERR_UNSUPPORTED, "d = %d not in {64,128}", d);
  SW_REQUIRE(heads >= 1, SW_ERR_INVALID_ARG, "heads = %d", heads);
  SW_REQUIRE(is_pow2(r) && r <= d, SW_ERR_INVALID_ARG, "r = %d must be a power of two <= d = %d", r, d);
  SW_TRY(check_arch());
  return launch_sketch_from_pooled(*L, sums, heads, d, signs, cols, r, scale, sketch, mean, (cudaStream_t)stream);
}

SW_API int32_t sw_sketch_append(int32_t batch, int32_t block, int32_t max_blocks, const sw_tensor* x,
                         const int32_t* seqlens, const int8_t* signs, const int32_t* cols, int32_t r,
                         float scale, float* mean, float* sketch, float* tok_sketch, sw_stream_t stream) {
  SW_REQUIRE(batch >= 0 && max_blocks >= 1, SW_ERR_INVALID_ARG, "batch %d / max_blocks %d", batch, max_blocks);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  SW_TRY(validate_tensor(x, "x"));
  SW_TRY(validate_sketch_params(x, cols, r));
  SW_REQUIRE(seqlens != nullptr, SW_ERR_INVALID_ARG, "seqlens is NULL");
  SW_REQUIRE((mean && sketch) || tok_sketch, SW_ERR_INVALID_ARG, "nothing to write");
  SW_REQUIRE((mean != nullptr) == (sketch != nullptr), SW_ERR_INVALID_ARG, "mean and sketch go together");
  SW_TRY(check_arch());
  return launch_sketch_append(batch, block, max_blocks, *x, seqlens, signs, cols, r, scale, mean, sketch,
                              tok_sketch, (cudaStream_t)stream);
}

SW_API int32_t sw_block_scores(const sw_layout* L, const float* qs, const float* ks, int32_t r, int32_t s,
                        uint32_t flags, float* W, float* A, sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_REQUIRE(qs && ks && W, SW_ERR_INVALID_ARG, "qs / ks / W is NULL");
  SW_REQUIRE(aligned16(qs) && aligned16(ks), SW_ERR_INVALID_ARG, "qs / ks must be 16-byte aligned");
  SW_REQUIRE(r >= 1 && r <= 128, SW_ERR_INVALID_ARG, "r = %d out of [1,128]", r);
  SW_REQUIRE(s >= 1, SW_ERR_INVALID_ARG, "s = %d must be >= 1", s);
  SW_TRY(check_arch());
  return launch_block_scores(*L, qs, ks, r, s, flags, W, A, (cudaStream_t)stream);
}

SW_API int32_t sw_block_scores_row(int32_t batch, int32_t block, int32_t max_blocks, const float* q_tok,
                            const float* ks, const int32_t* seqlens, int32_t r, int32_t s, uint32_t flags,
                            float* w_row, sw_stream_t stream) {
  SW_REQUIRE(batch >= 0 && max_blocks >= 1, SW_ERR_INVALID_ARG, "batch %d / max_blocks %d", batch, max_blocks);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  SW_REQUIRE(q_tok && ks && seqlens && w_row, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(r >= 1 && r <= 128 && s >= 1, SW_ERR_INVALID_ARG, "r = %d / s = %d", r, s);
  SW_REQUIRE(!(flags & SW_POW_MATRIX), SW_ERR_UNSUPPORTED, "row mode needs the element-wise power (P4)");
  SW_REQUIRE(flags & SW_CAUSAL, SW_ERR_UNSUPPORTED,
             "decode row mode needs SW_CAUSAL: without the block-causal mask Alg. 2 Step 4(ii) (PAPER.md:822-824) "
             "rewrites a column of the cached scores, which the row-vector form does not carry (P11)");
  SW_TRY(check_arch());
  return launch_block_scores_row(batch, block, max_blocks, q_tok, ks, seqlens, r, s, flags, w_row,
                                 (cudaStream_t)stream);
}

SW_API int32_t sw_walk_update(const sw_layout* L, const float* R_prev, const float* W, int32_t s, uint32_t flags,
                       float* R_out, void* ws, size_t ws_bytes, sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_REQUIRE(W && R_out, SW_ERR_INVALID_ARG, "W / R_out is NULL");
  SW_REQUIRE(R_out != R_prev && R_out != W, SW_ERR_INVALID_ARG, "R_out must not alias its inputs");
  SW_REQUIRE(s >= 1, SW_ERR_INVALID_ARG, "s = %d must be >= 1", s);
  if ((flags & SW_POW_MATRIX) && s > 1) {
    const size_t need = (size_t)L->batch * L->max_blocks * L->max_blocks * sizeof(float);
    SW_REQUIRE(ws != nullptr && ws_bytes >= need, SW_ERR_WORKSPACE,
               "sw_walk_update: workspace %zu < %zu bytes", ws_bytes, need);
  }
  SW_TRY(check_arch());
  return launch_walk(*L, R_prev, W, s, flags, R_out, ws, ws_bytes, (cudaStream_t)stream);
}

SW_API int32_t sw_walk_update_row(int32_t batch, int32_t block, int32_t max_blocks, const float* r_prev,
                           float* W_cache, int64_t stride_seq, const float* w_row,
                           const int32_t* seqlens, uint32_t flags, float* r_out, sw_stream_t stream) {
  SW_REQUIRE(batch >= 0 && max_blocks >= 1, SW_ERR_INVALID_ARG, "batch %d / max_blocks %d", batch, max_blocks);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  SW_REQUIRE(W_cache && w_row && seqlens && r_out, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(r_out != r_prev, SW_ERR_INVALID_ARG, "r_out must not alias r_prev");
  SW_REQUIRE(flags & SW_CAUSAL, SW_ERR_UNSUPPORTED,
             "decode row mode needs SW_CAUSAL: without the block-causal mask Alg. 2 Step 4(ii) (PAPER.md:822-824) "
             "rewrites a column of the cached scores, which the row-vector form does not carry (P11)");
  SW_TRY(check_arch());
  return launch_walk_row(batch, block, max_blocks, r_prev, W_cache, stride_seq, w_row, seqlens, flags,
                         r_out, (cudaStream_t)stream);
}

SW_API int32_t sw_select_topk(const sw_layout* L, const float* R, const int32_t* tau, int32_t tau_max,
                       uint32_t flags, int32_t* idx, int32_t* count, sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_REQUIRE(R && tau && idx && count, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(tau_max >= 1, SW_ERR_INVALID_ARG, "tau_max = %d", tau_max);
  SW_TRY(check_arch());
  return launch_select(*L, R, tau, tau_max, flags, idx, count, (cudaStream_t)stream);
}

SW_API int32_t sw_prefill_select(const sw_layout* L, const float* qs, const float* ks, int32_t r, int32_t s,
                          uint32_t flags, const float* R_prev, float* R_out, float* W, float* A,
                          const int32_t* tau, int32_t tau_max, int32_t* idx, int32_t* count, void* ws,
                          size_t ws_bytes, sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_REQUIRE(qs && ks && R_out && W && tau && idx && count, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(aligned16(qs) && aligned16(ks), SW_ERR_INVALID_ARG, "qs / ks must be 16-byte aligned");
  SW_REQUIRE(R_out != R_prev && R_out != W, SW_ERR_INVALID_ARG, "R_out must not alias its inputs");
  SW_REQUIRE(r >= 1 && r <= 128, SW_ERR_INVALID_ARG, "r = %d out of [1,128]", r);
  SW_REQUIRE(s >= 1 && tau_max >= 1, SW_ERR_INVALID_ARG, "s = %d / tau_max = %d", s, tau_max);
  const size_t pp_bytes = walk_pp_bytes(*L);
  const bool products = (flags & SW_POW_MATRIX) && s > 1;
  if (products)
    SW_REQUIRE(ws != nullptr && ws_bytes >= pp_bytes, SW_ERR_WORKSPACE, "sw_prefill_select: workspace %zu < %zu bytes",
               ws_bytes, pp_bytes);
  SW_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;
  if (L->total_blocks == 0) return SW_OK;
  if (products || !scores_fused_supported(*L, r)) {
    // s successive products (P4 matrix reading) or a sketch the fused score kernel does not take: the plain chain
    SW_TRY(launch_block_scores(*L, qs, ks, r, s, flags, W, A, st));
    SW_TRY(launch_walk(*L, R_prev, W, s, flags, R_out, ws, ws_bytes, st));
    return launch_select(*L, R_out, tau, tau_max, flags, idx, count, st);
  }
  const int causal = (flags & SW_CAUSAL) ? 1 : 0;
  int32_t which = SW_WALK_SIMT;
  if (R_prev != nullptr) {
    const bool have_ws = ws != nullptr && (reinterpret_cast<uintptr_t>(ws) & 127u) == 0 && ws_bytes > pp_bytes;
    which = choose_walk_kernel(*L, have_ws ? ws_bytes - pp_bytes : 0);
    if (which < 0) return which;
  }
  WalkImages im = {};
  const bool tc = which == SW_WALK_TCGEN05;
  if (tc) im = walk_images(*L, reinterpret_cast<uint8_t*>(ws) + pp_bytes);
  note_walk_kernel(which);
  // launch 1: W = A^s (+ R^0 = W^0 for the first layer, + the operand images of W and R_prev for the GEMM)
  SW_TRY(launch_scores_fused(*L, qs, ks, r, s, flags, W, A, R_prev ? nullptr : R_out, tc ? &im : nullptr, R_prev, st));
  // launch 2: the raw product R_prev W
  if (R_prev != nullptr)
    SW_TRY(tc ? launch_walk_tc(*L, im, R_out, causal, /*zero_upper=*/false, st)
              : launch_walk_simt(*L, R_prev, W, R_out, causal, st));
  // launch 3: row rescale (P9) + top-tau, in place
  return launch_rescale_select(*L, R_out, tau, tau_max, flags, idx, count, st);
}

SW_API int32_t sw_select_topk_row(int32_t batch, int32_t block, int32_t max_blocks, const float* r,
                           const int32_t* seqlens, const int32_t* tau, int32_t tau_max, uint32_t flags,
                           int32_t* idx, int32_t* count, sw_stream_t stream) {
  SW_REQUIRE(batch >= 0 && max_blocks >= 1, SW_ERR_INVALID_ARG, "batch %d / max_blocks %d", batch, max_blocks);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  SW_REQUIRE(r && seqlens && tau && idx && count, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(tau_max >= 1, SW_ERR_INVALID_ARG, "tau_max = %d", tau_max);
  SW_TRY(check_arch());
  return launch_select_row(batch, block, max_blocks, r, seqlens, tau, tau_max, flags, idx, count,
                           (cudaStream_t)stream);
}

SW_API int32_t sw_decode_select(int32_t batch, int32_t block, int32_t max_blocks, const sw_tensor* q,
                         const sw_tensor* k_new, const int32_t* seqlens, const int8_t* signs,
                         const int32_t* cols, int32_t r, float scale, int32_t s, uint32_t flags, float* kbar,
                         float* ks, float* W_cache, int64_t stride_seq, const float* r_prev,
                         float* r_out, const int32_t* tau, int32_t tau_max, int32_t* idx, int32_t* count,
                         void* ws, size_t ws_bytes, sw_stream_t stream) {
  SW_REQUIRE(batch >= 0 && max_blocks >= 1, SW_ERR_INVALID_ARG, "batch %d / max_blocks %d", batch, max_blocks);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  SW_TRY(validate_tensor(q, "q"));
  SW_TRY(validate_tensor(k_new, "k_new"));
  SW_REQUIRE(q->dtype == k_new->dtype && q->d == k_new->d, SW_ERR_UNSUPPORTED, "q / k_new dtype or head_dim differ");
  SW_TRY(validate_sketch_params(q, cols, r));
  SW_REQUIRE(seqlens && kbar && ks && W_cache && r_out && tau && idx && count, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(r_out != r_prev, SW_ERR_INVALID_ARG, "r_out must not alias r_prev");
  SW_REQUIRE(s >= 1 && tau_max >= 1, SW_ERR_INVALID_ARG, "s = %d / tau_max = %d", s, tau_max);
  SW_REQUIRE(!(flags & SW_POW_MATRIX), SW_ERR_UNSUPPORTED, "row mode needs the element-wise power (P4)");
  SW_REQUIRE(flags & SW_CAUSAL, SW_ERR_UNSUPPORTED,
             "decode row mode needs SW_CAUSAL: without the block-causal mask Alg. 2 Step 4(ii) (PAPER.md:822-824) "
             "rewrites a column of the cached scores, which the row-vector form does not carry (P11)");
  SW_TRY(check_arch());
  DecodeSelectArgs a;
  a.batch = batch; a.block = block; a.max_blocks = max_blocks; a.q = *q; a.k = *k_new; a.seqlens = seqlens;
  a.signs = signs; a.cols = cols; a.r = r; a.scale = scale; a.s = s; a.flags = flags; a.kbar = kbar; a.ks = ks;
  a.W_cache = W_cache; a.stride_seq = stride_seq; a.r_prev = r_prev; a.r_out = r_out; a.tau = tau;
  a.tau_max = tau_max; a.idx = idx; a.count = count; a.ws = ws; a.ws_bytes = ws_bytes;
  return launch_decode_select(a, (cudaStream_t)stream);
}

static size_t cast_bytes(int64_t tokens, int heads, int d) {
  return ((size_t)tokens * heads * d * 2 + 255) & ~(size_t)255;
}

SW_API size_t sw_workspace_bytes(int32_t op, const sw_layout* L, int32_t h_q, int32_t h_kv, int32_t d,
                          int32_t tau_max, int32_t dtype) {
  switch (op) {
    case SW_OP_WALK_UPDATE:
      return L ? walk_pp_bytes(*L) + walk_tc_ws_bytes(*L) : 0;
    case SW_OP_ATTN_PREFILL:
      if (!L || dtype != SW_F32) return 0;
      return cast_bytes(L->total_tokens, h_q, d) + 2 * cast_bytes(L->total_tokens, h_kv, d);
    case SW_OP_ATTN_DECODE:
      return L ? sw_decode_workspace_bytes(L->batch, h_q, h_kv, d, tau_max) : 0;
    default:
      return 0;
  }
}

SW_API size_t sw_decode_select_workspace_bytes(int32_t batch, int32_t max_blocks) {
  return (batch > 0 && max_blocks > 0) ? decode_select_ws_bytes(batch, max_blocks) : 0;
}

SW_API int32_t sw_decode_num_splits(int32_t batch, int32_t h_kv, int32_t d, int32_t tau_max) {
  check_arch();
  return decode_num_splits(batch, h_kv, tau_max, d);
}

SW_API size_t sw_decode_workspace_bytes(int32_t batch, int32_t h_q, int32_t h_kv, int32_t d, int32_t tau_max) {
  check_arch();
  return decode_ws_bytes(batch, h_q, d, decode_num_splits(batch, h_kv, tau_max, d));
}

SW_API int32_t sw_sparse_attn_prefill(const sw_layout* L, const sw_tensor* q, const sw_tensor* k, const sw_tensor* v,
                               const int32_t* idx, const int32_t* count, int32_t tau_max, float softmax_scale,
                               uint32_t flags, void* out, float* lse, void* ws, size_t ws_bytes,
                               sw_stream_t stream) {
  SW_TRY(validate_layout(L));
  SW_TRY(validate_tensor(q, "q"));
  SW_TRY(validate_tensor(k, "k"));
  SW_TRY(validate_tensor(v, "v"));
  SW_REQUIRE(idx && count && out, SW_ERR_INVALID_ARG, "idx / count / out is NULL");
  SW_REQUIRE(aligned16(out), SW_ERR_INVALID_ARG, "out is not 16-byte aligned");
  SW_REQUIRE(tau_max >= 1, SW_ERR_INVALID_ARG, "tau_max = %d", tau_max);
  SW_REQUIRE(q->dtype == k->dtype && k->dtype == v->dtype, SW_ERR_UNSUPPORTED, "q/k/v dtypes differ");
  SW_REQUIRE(q->d == k->d && k->d == v->d, SW_ERR_UNSUPPORTED, "q/k/v head_dim differ");
  SW_REQUIRE(k->heads == v->heads && q->heads % k->heads == 0, SW_ERR_INVALID_ARG,
             "h_q = %d must be a multiple of h_kv = %d", q->heads, k->heads);
  SW_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;

  AttnPrefillArgs a;
  a.L = L;
  a.h_q = q->heads; a.h_kv = k->heads; a.d = q->d;
  a.idx = idx; a.count = count; a.tau_max = tau_max;
  a.softmax_scale = softmax_scale; a.flags = flags;
  a.out = out; a.out_dtype = q->dtype; a.lse = lse;
  // kernel choice depends on shapes only: decide (and fail) before anything is launched
  const bool fits = attn_prefill_sm100_supported(a);
  const int32_t want = g_prefill_kernel.load();
  if (want == SW_PREFILL_TCGEN05 && !fits)
    return fail(SW_ERR_UNSUPPORTED, "sw_sparse_attn_prefill: SW_PREFILL_TCGEN05 needs d = 128 and h_q = 4 h_kv");
  if (q->dtype == SW_F32) {
    // P17: attention operands are rounded to bf16 by a cast pre-pass
    const size_t need = sw_workspace_bytes(SW_OP_ATTN_PREFILL, L, q->heads, k->heads, q->d, tau_max, SW_F32);
    SW_REQUIRE(ws != nullptr && ws_bytes >= need && aligned16(ws), SW_ERR_WORKSPACE,
               "sw_sparse_attn_prefill: fp32 inputs need %zu bytes of workspace, got %zu", need, ws_bytes);
    uint8_t* p = reinterpret_cast<uint8_t*>(ws);
    __nv_bfloat16* qb = reinterpret_cast<__nv_bfloat16*>(p);
    p += cast_bytes(L->total_tokens, q->heads, q->d);
    __nv_bfloat16* kb = reinterpret_cast<__nv_bfloat16*>(p);
    p += cast_bytes(L->total_tokens, k->heads, k->d);
    __nv_bfloat16* vb = reinterpret_cast<__nv_bfloat16*>(p);
    SW_TRY(launch_cast_f32_to_bf16((const float*)q->ptr, qb, L->total_tokens, q->heads, q->d, q->stride_tok, q->stride_head, st));
    SW_TRY(launch_cast_f32_to_bf16((const float*)k->ptr, kb, L->total_tokens, k->heads, k->d, k->stride_tok, k->stride_head, st));
    SW_TRY(launch_cast_f32_to_bf16((const float*)v->ptr, vb, L->total_tokens, v->heads, v->d, v->stride_tok, v->stride_head, st));
    a.q = qb; a.k = kb; a.v = vb;
    a.q_stride_head = q->d; a.q_stride_tok = (int64_t)q->heads * q->d;
    a.k_stride_head = k->d; a.k_stride_tok = (int64_t)k->heads * k->d;
    a.v_stride_head = v->d; a.v_stride_tok = (int64_t)v->heads * v->d;
  } else {
    a.q = (const __nv_bfloat16*)q->ptr; a.k = (const __nv_bfloat16*)k->ptr; a.v = (const __nv_bfloat16*)v->ptr;
    a.q_stride_tok = q->stride_tok; a.q_stride_head = q->stride_head;
    a.k_stride_tok = k->stride_tok; a.k_stride_head = k->stride_head;
    a.v_stride_tok = v->stride_tok; a.v_stride_head = v->stride_head;
  }
  if (fits && want != SW_PREFILL_GENERIC) {
    g_prefill_used = SW_PREFILL_TCGEN05;
    return launch_attn_prefill_sm100(a, st);
  }
  g_prefill_used = SW_PREFILL_GENERIC;
  return launch_attn_prefill_generic(a, st);
}

SW_API int32_t sw_set_prefill_kernel(int32_t which) {
  SW_REQUIRE(which >= SW_PREFILL_AUTO && which <= SW_PREFILL_TCGEN05, SW_ERR_INVALID_ARG,
             "sw_set_prefill_kernel: unknown value %d", which);
  return g_prefill_kernel.exchange(which);
}
SW_API int32_t sw_get_prefill_kernel_used(void) { return g_prefill_used; }

SW_API int32_t sw_set_walk_kernel(int32_t which) {
  SW_REQUIRE(which >= SW_WALK_AUTO && which <= SW_WALK_TCGEN05, SW_ERR_INVALID_ARG,
             "sw_set_walk_kernel: unknown value %d", which);
  return set_walk_kernel(which);
}
SW_API int32_t sw_get_walk_kernel_used(void) { return walk_kernel_used(); }

SW_API int32_t sw_sparse_attn_decode(int32_t batch, int32_t block, const sw_tensor* q, const sw_tensor* kcache,
                              const sw_tensor* vcache, int64_t stride_batch, const int32_t* seqlens,
                              const int32_t* idx, const int32_t* count, int32_t tau_max, float softmax_scale,
                              void* out, float* lse, void* ws, size_t ws_bytes, sw_stream_t stream) {
  SW_REQUIRE(batch >= 0, SW_ERR_INVALID_ARG, "batch = %d", batch);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  SW_TRY(validate_tensor(q, "q"));
  SW_TRY(validate_tensor(kcache, "kcache"));
  SW_TRY(validate_tensor(vcache, "vcache"));
  SW_REQUIRE(q->dtype == SW_BF16 && kcache->dtype == SW_BF16 && vcache->dtype == SW_BF16, SW_ERR_UNSUPPORTED,
             "decode attention takes bf16 q and caches");
  SW_REQUIRE(q->d == kcache->d && q->d == vcache->d, SW_ERR_UNSUPPORTED, "head_dim mismatch");
  SW_REQUIRE(kcache->heads == vcache->heads && q->heads % kcache->heads == 0 &&
                 q->heads / kcache->heads <= 16,
             SW_ERR_UNSUPPORTED, "GQA group h_q/h_kv = %d/%d must be an integer <= 16", q->heads, kcache->heads);
  SW_REQUIRE(seqlens && idx && count && out, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(tau_max >= 1 && stride_batch % 8 == 0, SW_ERR_INVALID_ARG, "tau_max / stride_batch");
  SW_TRY(check_arch());
  return launch_attn_decode(batch, block, *q, *kcache, *vcache, stride_batch, seqlens, idx, count, tau_max,
                            softmax_scale, out, lse, ws, ws_bytes, nullptr, 0, (cudaStream_t)stream);
}

SW_API int32_t sw_sparse_attn_decode_paged(int32_t batch, int32_t block, const sw_tensor* q, const sw_tensor* kpool,
                                    const sw_tensor* vpool, int64_t num_pages, const int32_t* block_table,
                                    int32_t table_stride, const int32_t* seqlens, const int32_t* idx,
                                    const int32_t* count, int32_t tau_max, float softmax_scale, void* out,
                                    float* lse, void* ws, size_t ws_bytes, sw_stream_t stream) {
  SW_REQUIRE(batch >= 0 && num_pages >= 0, SW_ERR_INVALID_ARG, "batch = %d / num_pages = %lld", batch, (long long)num_pages);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  SW_TRY(validate_tensor(q, "q"));
  SW_TRY(validate_tensor(kpool, "kpool"));
  SW_TRY(validate_tensor(vpool, "vpool"));
  SW_REQUIRE(q->dtype == SW_BF16 && kpool->dtype == SW_BF16 && vpool->dtype == SW_BF16, SW_ERR_UNSUPPORTED,
             "decode attention takes bf16 q and caches");
  SW_REQUIRE(q->d == kpool->d && q->d == vpool->d, SW_ERR_UNSUPPORTED, "head_dim mismatch");
  SW_REQUIRE(kpool->heads == vpool->heads && q->heads % kpool->heads == 0 && q->heads / kpool->heads <= 16,
             SW_ERR_UNSUPPORTED, "GQA group h_q/h_kv = %d/%d must be an integer <= 16", q->heads, kpool->heads);
  SW_REQUIRE(block_table && seqlens && idx && count && out, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(tau_max >= 1 && table_stride >= 1, SW_ERR_INVALID_ARG, "tau_max = %d / table_stride = %d", tau_max,
             table_stride);
  SW_TRY(check_arch());
  return launch_attn_decode(batch, block, *q, *kpool, *vpool, 0, seqlens, idx, count, tau_max, softmax_scale, out,
                            lse, ws, ws_bytes, block_table, table_stride, (cudaStream_t)stream);
}

}  // extern "C"
