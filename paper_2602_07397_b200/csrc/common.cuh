// Shared host/device helpers of libsw (sm_100a only).  No arithmetic of the method lives
// here: error plumbing, launch checks, small device utilities.
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/sw.h"

namespace sw {

// ---- thread-local error text ---------------------------------------------------------
void set_error(const char* fmt, ...);
int32_t fail(int32_t code, const char* fmt, ...);
int32_t check_arch();                      // SW_OK or SW_ERR_ARCH (cached per device)
int32_t check_launch(const char* what);    // cudaGetLastError -> SW_ERR_CUDA
int num_sms();
void count_launch(int n = 1);
uint64_t launches();           // kernels launched by this library (sw_launch_count)

#define SW_REQUIRE(cond, code, ...)            \
  do {                                         \
    if (!(cond)) return sw::fail((code), __VA_ARGS__); \
  } while (0)

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device property of a kernel.  It is set before every
// launch (a host-side table update, not a stream operation; legal during graph capture), so a process that
// drives several GPUs needs no per-device bookkeeping.
template <typename Kern>
static inline int32_t allow_dynamic_smem(Kern kern, size_t bytes, const char* what) {
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess)
    return check_launch(what);
  return SW_OK;
}

// Programmatic dependent launch (PDL): a kernel launched through launch_pdl may become resident while the kernel
// before it on the stream is still draining, once that kernel's CTAs have executed pdl_launch_dependents() (or
// exited); it must execute pdl_wait() before it touches anything its predecessors wrote.  Both device calls are
// no-ops when the kernel was launched the ordinary way, and a predecessor that never triggers simply gives the
// ordinary stream order.  Used along the decode layer (selection -> tail -> attention -> merge -> next selection),
// where every kernel is short and the launch gaps add up.
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                     Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline bool is_pow2(int x) { return x > 0 && (x & (x - 1)) == 0; }
static inline int cdiv(int a, int b) { return (a + b - 1) / b; }

int32_t validate_layout(const sw_layout* L);
int32_t validate_tensor(const sw_tensor* t, const char* name);

// ---- kernel launchers (one per translation unit) ---------------------------------------
int32_t launch_sketch(const sw_layout& L, const sw_tensor& x, const int8_t* signs, const int32_t* cols,
                      int r, float scale, float* sketch, float* mean, cudaStream_t st);
int32_t launch_sketch_qk(const sw_layout& L, const sw_tensor& q, const sw_tensor& k, const int8_t* signs,
                         const int32_t* cols, int r, float scale, float* qs, float* ks, float* qbar, float* kbar,
                         cudaStream_t st);
int32_t launch_copy_pool(const sw_layout& L, const sw_tensor& x, __nv_bfloat16* dst, float* sums, cudaStream_t st);
int32_t launch_sketch_from_pooled(const sw_layout& L, const float* sums, int heads, int d, const int8_t* signs,
                                  const int32_t* cols, int r, float scale, float* sketch, float* mean,
                                  cudaStream_t st);
int32_t launch_sketch_append(int batch, int block, int max_blocks, const sw_tensor& x,
                             const int32_t* seqlens, const int8_t* signs, const int32_t* cols, int r,
                             float scale, float* mean, float* sketch, float* tok_sketch, cudaStream_t st);
int32_t launch_block_scores(const sw_layout& L, const float* qs, const float* ks, int r, int s,
                            uint32_t flags, float* W, float* A, cudaStream_t st);
int32_t launch_block_scores_row(int batch, int block, int max_blocks, const float* q_tok, const float* ks,
                                const int32_t* seqlens, int r, int s, uint32_t flags, float* w_row,
                                cudaStream_t st);
int32_t launch_walk(const sw_layout& L, const float* R_prev, const float* W, int s, uint32_t flags,
                    float* R_out, void* ws, size_t ws_bytes, cudaStream_t st);
// workspace of sw_walk_update = [ping-pong matrix of the matrix-power reading | operand images of the tcgen05 GEMM]
static inline size_t walk_pp_bytes(const sw_layout& L) {
  return ((size_t)L.batch * L.max_blocks * L.max_blocks * sizeof(float) + 255) & ~(size_t)255;
}
bool walk_tc_supported(const sw_layout& L);
size_t walk_tc_ws_bytes(const sw_layout& L);
struct WalkImages {               // hi / lo TF32 operand images of the tensor-core walk GEMM (walk_images.cuh)
  float *r_hi, *r_lo, *w_hi, *w_lo;
  int pitch, rows;
};
WalkImages walk_images(const sw_layout& L, void* ws_images);
int32_t launch_split_tf32(const sw_layout& L, const float* R, const float* W, const WalkImages& im, int causal,
                          cudaStream_t st);
int32_t launch_walk_tc(const sw_layout& L, const WalkImages& im, float* dst, int causal, bool zero_upper,
                       cudaStream_t st);
int32_t launch_walk_simt(const sw_layout& L, const float* R_prev, const float* W, float* dst, int causal,
                         cudaStream_t st);
// fused selection chain (scores.cu / select.cu): scores + softmax + power (+ operand images) in one launch,
// row rescale + top-tau in one launch
int32_t launch_scores_fused(const sw_layout& L, const float* qs, const float* ks, int r, int s, uint32_t flags,
                            float* W, float* A, float* W2, const WalkImages* im, const float* R_prev,
                            cudaStream_t st);
bool scores_fused_supported(const sw_layout& L, int r);
int32_t launch_rescale_select(const sw_layout& L, float* R, const int32_t* tau, int tau_max, uint32_t flags,
                              int32_t* idx, int32_t* count, cudaStream_t st);
int32_t choose_walk_kernel(const sw_layout& L, size_t images_bytes);
void note_walk_kernel(int32_t which);
int32_t launch_copy_rows(const sw_layout& L, const float* src, float* dst, cudaStream_t st);
int32_t launch_row_rescale(const sw_layout& L, float* R, cudaStream_t st);
int32_t set_walk_kernel(int32_t which);
int32_t walk_kernel_used();
int32_t launch_walk_row(int batch, int block, int max_blocks, const float* r_prev, float* W_cache,
                        int64_t stride_seq, const float* w_row, const int32_t* seqlens, uint32_t flags,
                        float* r_out, cudaStream_t st);
int32_t launch_select(const sw_layout& L, const float* R, const int32_t* tau, int tau_max,
                      uint32_t flags, int32_t* idx, int32_t* count, cudaStream_t st);
int32_t launch_select_row(int batch, int block, int max_blocks, const float* r, const int32_t* seqlens,
                          const int32_t* tau, int tau_max, uint32_t flags, int32_t* idx, int32_t* count,
                          cudaStream_t st);

struct DecodeSelectArgs {
  int batch, block, max_blocks;
  sw_tensor q, k;                            // [batch, heads, d]; stride_tok = stride between sequences
  const int32_t* seqlens;
  const int8_t* signs;
  const int32_t* cols;
  int r;
  float scale;
  int s;
  uint32_t flags;
  float *kbar, *ks;
  float* W_cache;
  int64_t stride_seq;
  const float* r_prev;
  float* r_out;
  const int32_t* tau;
  int tau_max;
  int32_t *idx, *count;
  void* ws;
  size_t ws_bytes;
};
int32_t launch_decode_select(const DecodeSelectArgs& a, cudaStream_t st);
size_t decode_select_ws_bytes(int batch, int max_blocks);

struct AttnPrefillArgs {
  const sw_layout* L;
  const __nv_bfloat16 *q, *k, *v;           // bf16 operands (possibly the cast copies in ws)
  int64_t q_stride_tok, q_stride_head, k_stride_tok, k_stride_head, v_stride_tok, v_stride_head;
  int h_q, h_kv, d;
  const int32_t *idx, *count;
  int tau_max;
  float softmax_scale;
  uint32_t flags;
  void* out;                                // [total_tokens, h_q, d] contiguous
  int out_dtype;                            // SW_BF16 | SW_F32
  float* lse;
};
int32_t launch_attn_prefill_generic(const AttnPrefillArgs& a, cudaStream_t st);
bool attn_prefill_sm100_supported(const AttnPrefillArgs& a);
int32_t launch_attn_prefill_sm100(const AttnPrefillArgs& a, cudaStream_t st);
int32_t launch_cast_f32_to_bf16(const float* src, __nv_bfloat16* dst, int64_t tokens, int heads, int d,
                                int64_t stride_tok, int64_t stride_head, cudaStream_t st);

int decode_num_splits(int batch, int h_kv, int tau_max, int d);
size_t decode_ws_bytes(int batch, int h_q, int d, int nsplit);
int32_t launch_attn_decode(int batch, int block, const sw_tensor& q, const sw_tensor& kc,
                           const sw_tensor& vc, int64_t stride_batch, const int32_t* seqlens,
                           const int32_t* idx, const int32_t* count, int tau_max, float softmax_scale,
                           void* out, float* lse, void* ws, size_t ws_bytes, const int32_t* table,
                           int table_stride, cudaStream_t st);

}  // namespace sw

// ---- device utilities ------------------------------------------------------------------
#ifdef __CUDACC__
namespace swd {

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// pdl_wait(p, q, ...): wait, then pass the pointers through an empty asm.  Loads the compiler treats as invariant
// (__ldg, const __restrict__ parameters: ld.global.nc) are not ordered by a memory clobber -- measured: the loads of
// count[seq] and seqlens[seq] of the decode attention kernel were scheduled ABOVE griddepcontrol.wait and read what the
// selection kernel had not written yet (a wild block list, about one run in four).  A load through a pointer that
// comes out of an asm statement issued after the wait cannot move above it.  Every pointer to data an earlier
// kernel of the stream may have written goes through here before its first use.
template <typename T> __device__ __forceinline__ void pdl_launder(T*& p) { asm volatile("" : "+l"(p)); }
template <typename... P> __device__ __forceinline__ void pdl_wait(P*&... ptrs) {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  (pdl_launder(ptrs), ...);
}
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ int warp_sum_i(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// sequence that owns global block index gb: largest s with cu_blocks[s] <= gb
__device__ __forceinline__ int find_seq(const int32_t* __restrict__ cu, int batch, int gb) {
  int lo = 0, hi = batch - 1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (__ldg(cu + mid) <= gb) lo = mid; else hi = mid - 1;
  }
  return lo;
}

__device__ __forceinline__ uint4 ld_nc_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// x^s for an integer s >= 1 by repeated squaring; the small exponents in use (the configs' 1-3, the paper's 8) are
// straight-line code (s is uniform over a kernel: the switch does not diverge)
__device__ __forceinline__ float powi(float x, int s) {
  switch (s) {
    case 1: return x;
    case 2: return x * x;
    case 3: return x * x * x;
    case 4: { const float x2 = x * x; return x2 * x2; }
    case 8: { const float x2 = x * x, x4 = x2 * x2; return x4 * x4; }
    default: break;
  }
  float r = 1.f, b = x;
  while (s) { if (s & 1) r *= b; b *= b; s >>= 1; }
  return r;
}

}  // namespace swd
#endif
