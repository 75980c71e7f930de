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
};

template <typename T, int D>
__global__ void __launch_bounds__(kThreads)
sketch_kernel(const T* __restrict__ x, int64_t stride_tok, int64_t stride_head, int heads,
              const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ cu_blocks, int batch,
              int B, const int8_t* __restrict__ signs, const int32_t* __restrict__ cols, int r,
              float scale, float* __restrict__ sketch, float* __restrict__ mean) {
  constexpr int D8 = D / 8;                      // 8-element chunks per head row
  __shared__ float s_part[kThreads][9];          // +1 pad
  __shared__ float s_vec[D];

  const int gb = blockIdx.x;
  const int seq = swd::find_seq(cu_blocks, batch, gb);
  const int bi = gb - __ldg(cu_blocks + seq);
  const int tok0 = __ldg(cu_seqlens + seq) + bi * B;
  const int tok_end = min(tok0 + B, __ldg(cu_seqlens + seq + 1));
  const int ntok = tok_end - tok0;

  const int tid = threadIdx.x;
  const int chunk = tid % D8;                    // constant per thread: kThreads % D8 == 0
  const int rows_per_pass = kThreads / D8;       // (token, head) rows covered per pass
  const int total_rows = ntok * heads;
  __align__(8) float acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.f;

  int row = tid / D8;
  if (stride_head == D && stride_tok == (int64_t)heads * D) {
    // packed layout: the block is one contiguous run of ntok * heads rows of D elements (no index division)
    const T* xb = x + (int64_t)tok0 * stride_tok + chunk * 8;
    for (; row + (kUnroll - 1) * rows_per_pass < total_rows; row += kUnroll * rows_per_pass) {
      Chunk<T> c[kUnroll];
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) c[u].load(xb + (int64_t)(row + u * rows_per_pass) * D);
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) c[u].add_to(acc);
    }
    for (; row < total_rows; row += rows_per_pass) {
      Chunk<T> c;
      c.load(xb + (int64_t)row * D);
      c.add_to(acc);
    }
  } else {
  // main loop: kUnroll independent 128-bit loads in flight per thread
  for (; row + (kUnroll - 1) * rows_per_pass < total_rows; row += kUnroll * rows_per_pass) {
    Chunk<T> c[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      int rr = row + u * rows_per_pass;
      int tok = rr / heads, hd = rr - tok * heads;
      c[u].load(x + (int64_t)(tok0 + tok) * stride_tok + (int64_t)hd * stride_head + chunk * 8);
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) c[u].add_to(acc);
  }
  for (; row < total_rows; row += rows_per_pass) {
    int tok = row / heads, hd = row - tok * heads;
    Chunk<T> c;
    c.load(x + (int64_t)(tok0 + tok) * stride_tok + (int64_t)hd * stride_head + chunk * 8);
    c.add_to(acc);
  }
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) s_part[tid][i] = acc[i];
  __syncthreads();
  if (tid < D) {
    const int ch = tid / 8, e = tid % 8;
    float s = 0.f;
    for (int k = 0; k < rows_per_pass; ++k) s += s_part[k * D8 + ch][e];
    const float m = s / (float)(ntok * heads);   // P12: divide by the number of valid tokens
    s_vec[tid] = m;
    if (mean) mean[(int64_t)gb * D + tid] = m;
  }
  __syncthreads();
  sketch_tail<D>(s_vec, signs, cols, r, scale, sketch + (int64_t)gb * r);
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
