// sw_sketch: Small-World Sketching, Alg. 1 Steps 1-4, sec 2.2.
// One fused pass: head mean + block mean (token-space sketch) -> sign flip D -> fast
// Walsh-Hadamard transform in registers / warp shuffles -> column sampling S -> scale.
// HBM-bound: every element of x is read exactly once with 128-bit loads; H_d is never
// materialised.
#include "common.cuh"
#include "sketch_common.cuh"

namespace {

using namespace swsk;

constexpr int kThreads = 256;
constexpr int kUnroll = 8;

template <typename T> struct Chunk;          // 8 consecutive elements of one row
template <> struct Chunk<__nv_bfloat16> {
  uint4 v;
  __device__ __forceinline__ void load(const __nv_bfloat16* p) { v = swd::ld_nc_v4(p); }
  // bf16 -> fp32 is a 16-bit shift; the two halves of a word are added with one packed FADD2
  __device__ __forceinline__ void add_to(float* acc) const {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    float2* a2 = reinterpret_cast<float2*>(acc);
#pragma unroll
    for (int i = 0; i < 4; ++i)
      a2[i] = __fadd2_rn(a2[i], make_float2(__uint_as_float(w[i] << 16), __uint_as_float(w[i] & 0xffff0000u)));
  }
  __device__ __forceinline__ void store_bf16(__nv_bfloat16* p) const { *reinterpret_cast<uint4*>(p) = v; }
};
template <> struct Chunk<float> {
  uint4 a, b;
  __device__ __forceinline__ void load(const float* p) {
    a = swd::ld_nc_v4(p);
    b = swd::ld_nc_v4(p + 4);
  }
  __device__ __forceinline__ void add_to(float* acc) const {
    const float* fa = reinterpret_cast<const float*>(&a);
    const float* fb = reinterpret_cast<const float*>(&b);
#pragma unroll
    for (int i = 0; i < 4; ++i) { acc[i] += fa[i]; acc[4 + i] += fb[i]; }
  }
  __device__ __forceinline__ void store_bf16(__nv_bfloat16* p) const {
    const float* fa = reinterpret_cast<const float*>(&a);
    const float* fb = reinterpret_cast<const float*>(&b);
    uint4 o;
    __nv_bfloat162 t;
    t = __floats2bfloat162_rn(fa[0], fa[1]); o.x = *reinterpret_cast<uint32_t*>(&t);
    t = __floats2bfloat162_rn(fa[2], fa[3]); o.y = *reinterpret_cast<uint32_t*>(&t);
    t = __floats2bfloat162_rn(fb[0], fb[1]); o.z = *reinterpret_cast<uint32_t*>(&t);
    t = __floats2bfloat162_rn(fb[2], fb[3]); o.w = *reinterpret_cast<uint32_t*>(&t);
    *reinterpret_cast<uint4*>(p) = o;
  }
};

// Sum of the rows (token, head) of tokens [tok0, tok0 + ntok) of x over this CTA's threads: thread t adds the
// 8 elements [8 (t % D8), +8) of rows t / D8, t / D8 + kThreads / D8, ... into acc[8].  kUnroll independent
// 128-bit loads in flight per thread.  dst != nullptr (copy_pool_kernel): the rows are also written, as bf16,
// to the packed [tokens, heads, D] tensor dst.
template <typename T, int D, bool kCopy>
__device__ __forceinline__ void accumulate_rows(const T* __restrict__ x, int64_t stride_tok, int64_t stride_head,
                                                int heads, int tok0, int ntok, float (&acc)[8],
                                                __nv_bfloat16* __restrict__ dst) {
  constexpr int D8 = D / 8;
  const int tid = threadIdx.x;
  const int chunk = tid % D8;                    // constant per thread: kThreads % D8 == 0
  const int rows_per_pass = kThreads / D8;       // (token, head) rows covered per pass
  const int total_rows = ntok * heads;
  int row = tid / D8;
  if (stride_head == D && stride_tok == (int64_t)heads * D) {
    // packed layout: the block is one contiguous run of ntok * heads rows of D elements (no index division)
    const T* xb = x + (int64_t)tok0 * stride_tok + chunk * 8;
    __nv_bfloat16* db = kCopy ? dst + (int64_t)tok0 * heads * D + chunk * 8 : nullptr;
    for (; row + (kUnroll - 1) * rows_per_pass < total_rows; row += kUnroll * rows_per_pass) {
      Chunk<T> c[kUnroll];
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) c[u].load(xb + (int64_t)(row + u * rows_per_pass) * D);
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        c[u].add_to(acc);
        if (kCopy) c[u].store_bf16(db + (int64_t)(row + u * rows_per_pass) * D);
      }
    }
    for (; row < total_rows; row += rows_per_pass) {
      Chunk<T> c;
      c.load(xb + (int64_t)row * D);
      c.add_to(acc);
      if (kCopy) c.store_bf16(db + (int64_t)row * D);
    }
    return;
  }
  for (; row + (kUnroll - 1) * rows_per_pass < total_rows; row += kUnroll * rows_per_pass) {
    Chunk<T> c[kUnroll];
    int tok[kUnroll], hd[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const int rr = row + u * rows_per_pass;
      tok[u] = rr / heads; hd[u] = rr - tok[u] * heads;
      c[u].load(x + (int64_t)(tok0 + tok[u]) * stride_tok + (int64_t)hd[u] * stride_head + chunk * 8);
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      c[u].add_to(acc);
      if (kCopy) c[u].store_bf16(dst + ((int64_t)(tok0 + tok[u]) * heads + hd[u]) * D + chunk * 8);
    }
  }
  for (; row < total_rows; row += rows_per_pass) {
    const int tok = row / heads, hd = row - tok * heads;
    Chunk<T> c;
    c.load(x + (int64_t)(tok0 + tok) * stride_tok + (int64_t)hd * stride_head + chunk * 8);
    c.add_to(acc);
    if (kCopy) c.store_bf16(dst + ((int64_t)(tok0 + tok) * heads + hd) * D + chunk * 8);
  }
}

// acc[8] of all threads -> s_vec[D] = column sums (s_part: [kThreads][9] scratch)
template <int D>
__device__ __forceinline__ void reduce_columns(const float (&acc)[8], float (*s_part)[9], float* s_vec) {
  constexpr int D8 = D / 8;
  const int tid = threadIdx.x;
#pragma unroll
  for (int i = 0; i < 8; ++i) s_part[tid][i] = acc[i];
  __syncthreads();
  if (tid < D) {
    const int ch = tid / 8, e = tid % 8;
    float s = 0.f;
    for (int k = 0; k < kThreads / D8; ++k) s += s_part[k * D8 + ch][e];
    s_vec[tid] = s;
  }
  __syncthreads();
}

__device__ __forceinline__ void block_tokens(const int32_t* cu_seqlens, const int32_t* cu_blocks, int batch, int B,
                                             int gb, int& tok0, int& ntok) {
  const int seq = swd::find_seq(cu_blocks, batch, gb);
  const int bi = gb - __ldg(cu_blocks + seq);
  tok0 = __ldg(cu_seqlens + seq) + bi * B;
  ntok = min(tok0 + B, __ldg(cu_seqlens + seq + 1)) - tok0;
}

template <typename T, int D>
__global__ void __launch_bounds__(kThreads)
sketch_kernel(const T* __restrict__ x, int64_t stride_tok, int64_t stride_head, int heads,
              const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ cu_blocks, int batch,
              int B, const int8_t* __restrict__ signs, const int32_t* __restrict__ cols, int r,
              float scale, float* __restrict__ sketch, float* __restrict__ mean) {
  __shared__ float s_part[kThreads][9];          // +1 pad
  __shared__ float s_vec[D];
  const int gb = blockIdx.x, tid = threadIdx.x;
  int tok0, ntok;
  block_tokens(cu_seqlens, cu_blocks, batch, B, gb, tok0, ntok);
  __align__(8) float acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.f;
  accumulate_rows<T, D, false>(x, stride_tok, stride_head, heads, tok0, ntok, acc, nullptr);
  reduce_columns<D>(acc, s_part, s_vec);
  if (tid < D) {
    const float m = s_vec[tid] / (float)(ntok * heads);   // P12: divide by the number of valid tokens
    s_vec[tid] = m;
    if (mean) mean[(int64_t)gb * D + tid] = m;
  }
  __syncthreads();
  sketch_tail<D>(s_vec, signs, cols, r, scale, sketch + (int64_t)gb * r);
}

// sw_sketch_qk: Q and K of one layer in ONE launch: CTA i < total_blocks sums query block i, the others key
// block i - total_blocks -- the body of sketch_kernel on either tensor.  HBM-bound and fair: every CTA gets the
// same share of the memory system, so the 512 KB query CTAs end together and the key CTAs fill in behind
// them; it does not matter which SM holds how many.  Measured on B200 (cfg 2, 336 MB per layer, kernels alone,
// back to back in a CUDA graph): this layout 54 us = 6.2 TB/s; equal 128 KB units (a quarter of a query block
// per CTA, the quarters added through distributed shared memory by 4-CTA clusters) 58 us; the same with the
// rows streamed through a cp.async.bulk ring of 3 x 32 KB per CTA 60 us -- and 71 / 80 us inside the
// power-capped step, where the register-load kernel keeps 57 us.
struct QkParams {
  const void *q, *k;
  int64_t q_stride_tok, q_stride_head, k_stride_tok, k_stride_head;
  int h_q, h_kv;
  const int32_t *cu_seqlens, *cu_blocks;
  int batch, B, total_blocks;
  const int8_t* signs;  const int32_t* cols;  int r;  float scale;
  float *qs, *ks, *qbar, *kbar;
};

template <typename T, int D>
__global__ void __launch_bounds__(kThreads)
sketch_qk_kernel(const QkParams p) {
  __shared__ float s_part[kThreads][9];
  __shared__ float s_vec[D];
  const int tid = threadIdx.x;
  const bool is_q = (int)blockIdx.x < p.total_blocks;
  const int gb = is_q ? blockIdx.x : blockIdx.x - p.total_blocks;
  int tok0, ntok;
  block_tokens(p.cu_seqlens, p.cu_blocks, p.batch, p.B, gb, tok0, ntok);
  __align__(8) float acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.f;
  if (is_q)
    accumulate_rows<T, D, false>(reinterpret_cast<const T*>(p.q), p.q_stride_tok, p.q_stride_head, p.h_q, tok0, ntok,
                                 acc, nullptr);
  else
    accumulate_rows<T, D, false>(reinterpret_cast<const T*>(p.k), p.k_stride_tok, p.k_stride_head, p.h_kv, tok0, ntok,
                                 acc, nullptr);
  reduce_columns<D>(acc, s_part, s_vec);
  const int heads = is_q ? p.h_q : p.h_kv;
  float* mean = is_q ? p.qbar : p.kbar;
  if (tid < D) {
    const float m = s_vec[tid] / (float)(ntok * heads);   // P12: divide by the number of valid tokens
    s_vec[tid] = m;
    if (mean) mean[(int64_t)gb * D + tid] = m;
  }
  __syncthreads();
  sketch_tail<D>(s_vec, p.signs, p.cols, p.r, p.scale, (is_q ? p.qs : p.ks) + (int64_t)gb * p.r);
}

// A producer that emits the pooled sums as a by-product ("custom CUDA kernels
// for block aggregation"): copies x (bf16 or fp32) into the packed bf16 tensor dst -- the cast pre-pass of P17,
// or a KV-cache append -- and writes sums[gb, :] = sum over the heads and valid tokens of block gb of x.
template <typename T, int D>
__global__ void __launch_bounds__(kThreads)
copy_pool_kernel(const T* __restrict__ x, int64_t stride_tok, int64_t stride_head, int heads,
                 const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ cu_blocks, int batch, int B,
                 __nv_bfloat16* __restrict__ dst, float* __restrict__ sums) {
  __shared__ float s_part[kThreads][9];
  __shared__ float s_vec[D];
  const int gb = blockIdx.x;
  int tok0, ntok;
  block_tokens(cu_seqlens, cu_blocks, batch, B, gb, tok0, ntok);
  __align__(8) float acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.f;
  accumulate_rows<T, D, true>(x, stride_tok, stride_head, heads, tok0, ntok, acc, dst);
  reduce_columns<D>(acc, s_part, s_vec);
  if (threadIdx.x < D) sums[(int64_t)gb * D + threadIdx.x] = s_vec[threadIdx.x];
}

// sw_sketch_from_pooled: Alg. 1 Steps 3-4 from per-block sums a producer left behind: divide
// by the number of pooled rows (P12), sign flip, FWHT, column pick, scale.  One warp per block.
template <int D>
__global__ void __launch_bounds__(128)
sketch_from_pooled_kernel(const float* __restrict__ sums, int heads, const int32_t* __restrict__ cu_seqlens,
                          const int32_t* __restrict__ cu_blocks, int batch, int B, int total_blocks,
                          const int8_t* __restrict__ signs, const int32_t* __restrict__ cols, int r, float scale,
                          float* __restrict__ sketch, float* __restrict__ mean) {
  __shared__ float s_vec[4][D];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int gb = blockIdx.x * 4 + warp;
  if (gb >= total_blocks) return;
  int tok0, ntok;
  block_tokens(cu_seqlens, cu_blocks, batch, B, gb, tok0, ntok);
  const float inv = 1.f / (float)(ntok * heads);
  for (int x = lane; x < D; x += 32) {
    const float m = sums[(int64_t)gb * D + x] * inv;
    s_vec[warp][x] = m;
    if (mean) mean[(int64_t)gb * D + x] = m;
  }
  __syncwarp();
  sketch_tail<D>(s_vec[warp], signs, cols, r, scale, sketch + (int64_t)gb * r, nullptr, warp);
}

// Decode (Alg. 2 Steps 2-3): one token per sequence; one CTA per sequence.
template <typename T, int D>
__global__ void __launch_bounds__(128)
sketch_append_kernel(const T* __restrict__ x, int64_t stride_seq, int64_t stride_head, int heads,
                     const int32_t* __restrict__ seqlens, int B, int max_blocks,
                     const int8_t* __restrict__ signs, const int32_t* __restrict__ cols, int r, float scale,
                     float* __restrict__ mean, float* __restrict__ sketch, float* __restrict__ tok_sketch) {
  __shared__ float s_vec[D];
  __shared__ float s_tok[D];
  const int seq = blockIdx.x;
  const int t = __ldg(seqlens + seq);
  const int bcur = (t - 1) / B;
  const int c = (t - 1) % B;                      // tokens already in block b_curr
  const int tid = threadIdx.x;
  if (tid < D) {
    float s = 0.f;
    for (int h = 0; h < heads; ++h)
      s += (float)x[(int64_t)seq * stride_seq + (int64_t)h * stride_head + tid];
    const float avg = s / (float)heads;           // PAPER.md:810 / 815
    s_tok[tid] = avg;
    if (mean) {
      float* mp = mean + ((int64_t)seq * max_blocks + bcur) * D + tid;
      const float m = (c == 0) ? avg : ((float)c * (*mp) + avg) / (float)(c + 1);
      *mp = m;
      s_vec[tid] = m;
    }
  }
  __syncthreads();
  if (mean && sketch)
    sketch_tail<D>(s_vec, signs, cols, r, scale, sketch + ((int64_t)seq * max_blocks + bcur) * r);
  if (tok_sketch) sketch_tail<D>(s_tok, signs, cols, r, scale, tok_sketch + (int64_t)seq * r);
}

}  // namespace

namespace sw {

int32_t launch_sketch(const sw_layout& L, const sw_tensor& x, const int8_t* signs, const int32_t* cols,
                      int r, float scale, float* sketch, float* mean, cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  dim3 grid(L.total_blocks), block(kThreads);
#define SW_LAUNCH(T, D)                                                                              \
  sketch_kernel<T, D><<<grid, block, 0, st>>>((const T*)x.ptr, x.stride_tok, x.stride_head, x.heads, \
                                              L.cu_seqlens, L.cu_blocks, L.batch, L.block, signs,    \
                                              cols, r, scale, sketch, mean)
  count_launch();
  if (x.dtype == SW_BF16 && x.d == 128) SW_LAUNCH(__nv_bfloat16, 128);
  else if (x.dtype == SW_BF16 && x.d == 64) SW_LAUNCH(__nv_bfloat16, 64);
  else if (x.dtype == SW_F32 && x.d == 128) SW_LAUNCH(float, 128);
  else if (x.dtype == SW_F32 && x.d == 64) SW_LAUNCH(float, 64);
  else return fail(SW_ERR_UNSUPPORTED, "sw_sketch: dtype %d / d %d", x.dtype, x.d);
#undef SW_LAUNCH
  return check_launch("sw_sketch");
}

int32_t launch_sketch_qk(const sw_layout& L, const sw_tensor& q, const sw_tensor& k, const int8_t* signs,
                         const int32_t* cols, int r, float scale, float* qs, float* ks, float* qbar, float* kbar,
                         cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  QkParams p;
  p.q = q.ptr; p.k = k.ptr; p.q_stride_tok = q.stride_tok; p.q_stride_head = q.stride_head;
  p.k_stride_tok = k.stride_tok; p.k_stride_head = k.stride_head; p.h_q = q.heads; p.h_kv = k.heads;
  p.cu_seqlens = L.cu_seqlens; p.cu_blocks = L.cu_blocks; p.batch = L.batch; p.B = L.block;
  p.total_blocks = L.total_blocks; p.signs = signs; p.cols = cols; p.r = r; p.scale = scale;
  p.qs = qs; p.ks = ks; p.qbar = qbar; p.kbar = kbar;
  void (*kern)(const QkParams) = nullptr;
  if (q.dtype == SW_BF16 && q.d == 128) kern = sketch_qk_kernel<__nv_bfloat16, 128>;
  else if (q.dtype == SW_BF16 && q.d == 64) kern = sketch_qk_kernel<__nv_bfloat16, 64>;
  else if (q.dtype == SW_F32 && q.d == 128) kern = sketch_qk_kernel<float, 128>;
  else if (q.dtype == SW_F32 && q.d == 64) kern = sketch_qk_kernel<float, 64>;
  else return fail(SW_ERR_UNSUPPORTED, "sw_sketch_qk: dtype %d / d %d", q.dtype, q.d);
  count_launch();
  kern<<<2 * L.total_blocks, kThreads, 0, st>>>(p);
  return check_launch("sw_sketch_qk");
}

int32_t launch_copy_pool(const sw_layout& L, const sw_tensor& x, __nv_bfloat16* dst, float* sums, cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  dim3 grid(L.total_blocks), block(kThreads);
#define SW_LAUNCH(T, D)                                                                                   \
  copy_pool_kernel<T, D><<<grid, block, 0, st>>>((const T*)x.ptr, x.stride_tok, x.stride_head, x.heads, \
                                                 L.cu_seqlens, L.cu_blocks, L.batch, L.block, dst, sums)
  count_launch();
  if (x.dtype == SW_BF16 && x.d == 128) SW_LAUNCH(__nv_bfloat16, 128);
  else if (x.dtype == SW_BF16 && x.d == 64) SW_LAUNCH(__nv_bfloat16, 64);
  else if (x.dtype == SW_F32 && x.d == 128) SW_LAUNCH(float, 128);
  else if (x.dtype == SW_F32 && x.d == 64) SW_LAUNCH(float, 64);
  else return fail(SW_ERR_UNSUPPORTED, "sw_copy_pool: dtype %d / d %d", x.dtype, x.d);
#undef SW_LAUNCH
  return check_launch("sw_copy_pool");
}

int32_t launch_sketch_from_pooled(const sw_layout& L, const float* sums, int heads, int d, const int8_t* signs,
                                  const int32_t* cols, int r, float scale, float* sketch, float* mean,
                                  cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  const int grid = cdiv(L.total_blocks, 4);
  count_launch();
  if (d == 128)
    sketch_from_pooled_kernel<128><<<grid, 128, 0, st>>>(sums, heads, L.cu_seqlens, L.cu_blocks, L.batch, L.block,
                                                         L.total_blocks, signs, cols, r, scale, sketch, mean);
  else if (d == 64)
    sketch_from_pooled_kernel<64><<<grid, 128, 0, st>>>(sums, heads, L.cu_seqlens, L.cu_blocks, L.batch, L.block,
                                                        L.total_blocks, signs, cols, r, scale, sketch, mean);
  else return fail(SW_ERR_UNSUPPORTED, "sw_sketch_from_pooled: d %d", d);
  return check_launch("sw_sketch_from_pooled");
}

int32_t launch_sketch_append(int batch, int block, int max_blocks, const sw_tensor& x,
                             const int32_t* seqlens, const int8_t* signs, const int32_t* cols, int r,
                             float scale, float* mean, float* sketch, float* tok_sketch, cudaStream_t st) {
  if (batch == 0) return SW_OK;
#define SW_LAUNCH(T, D)                                                                          \
  sketch_append_kernel<T, D><<<batch, 128, 0, st>>>((const T*)x.ptr, x.stride_tok, x.stride_head, \
                                                    x.heads, seqlens, block, max_blocks, signs,   \
                                                    cols, r, scale, mean, sketch, tok_sketch)
  count_launch();
  if (x.dtype == SW_BF16 && x.d == 128) SW_LAUNCH(__nv_bfloat16, 128);
  else if (x.dtype == SW_BF16 && x.d == 64) SW_LAUNCH(__nv_bfloat16, 64);
  else if (x.dtype == SW_F32 && x.d == 128) SW_LAUNCH(float, 128);
  else if (x.dtype == SW_F32 && x.d == 64) SW_LAUNCH(float, 64);
  else return fail(SW_ERR_UNSUPPORTED, "sw_sketch_append: dtype %d / d %d", x.dtype, x.d);
#undef SW_LAUNCH
  return check_launch("sw_sketch_append");
}

}  // namespace sw
