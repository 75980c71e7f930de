// Layout of the hi / lo TF32 operand images of the tensor-core walk GEMM (walk_tc.cu) in the caller's
// workspace, shared by the kernels that write them (split_tf32_kernel, the fused score kernel) and the GEMM
// that reads them through TMA.  All sequences of a batch are stacked in ONE [rows, pitch] fp32 array per
// operand: pitch = max_blocks rounded up to 32 floats, sequence s owns the rows from
// row_base(s) = pad128(cu_blocks[s]) + 128 s (computable on the device from cu_blocks alone; leaves every
// sequence at least pad128(b_s) rows).  Everything a TMA box of the GEMM can touch is written: values inside
// [0, b_s) x [0, b_s), zeros in the padding rows and columns, so a box that hangs over the end of a sequence
// multiplies zeros, never stale workspace bits.  No arithmetic of the method lives here.
#pragma once

#include <stdint.h>

namespace swimg {

__host__ __device__ __forceinline__ int pitch_of(int max_blocks) { return (max_blocks + 31) & ~31; }
__host__ __device__ __forceinline__ int pad_rows(int b) { return (b + 127) & ~127; }
__host__ __device__ __forceinline__ int rows_bound(int total_blocks, int batch) { return pad_rows(total_blocks) + 128 * batch; }
#ifdef __CUDACC__
__device__ __forceinline__ int row_base(const int32_t* cu_blocks, int seq) {
  return pad_rows(__ldg(cu_blocks + seq)) + 128 * seq;
}
// columns [0, row_cols) of image row i are read by the GEMM: up to the end of the row's diagonal 128-tile when
// the operands are lower triangular, else the whole pitch
__device__ __forceinline__ int row_cols(int i, int pitch, int causal) {
  return causal ? min(pitch, (i / 128 + 1) * 128) : pitch;
}
__device__ __forceinline__ void split4(const float4& x, float4& h, float4& l) {
  h.x = __uint_as_float(__float_as_uint(x.x) & 0xffffe000u); l.x = x.x - h.x;
  h.y = __uint_as_float(__float_as_uint(x.y) & 0xffffe000u); l.y = x.y - h.y;
  h.z = __uint_as_float(__float_as_uint(x.z) & 0xffffe000u); l.z = x.z - h.z;
  h.w = __uint_as_float(__float_as_uint(x.w) & 0xffffe000u); l.w = x.w - h.w;
}
// One image row from one row of a packed b x b matrix (src_row = &M[i][0]; rows i >= b are padding).  The loads of
// kSplitUnroll float4s per thread are issued before the first one is used: with one load in flight a 2048-column
// row split by one warp was 16 dependent memory latencies.
constexpr int kSplitUnroll = 4;
__device__ __forceinline__ void split_row(const float* __restrict__ src_row, int i, int b, int pitch, int causal,
                                          float* __restrict__ hi, float* __restrict__ lo, int tid, int nthreads) {
  const int lim = row_cols(i, pitch, causal);
  const bool vec = i < b && (b & 3) == 0 && (reinterpret_cast<uintptr_t>(src_row) & 15u) == 0;
  for (int j0 = tid * 4; j0 < lim; j0 += kSplitUnroll * nthreads * 4) {
    float4 x[kSplitUnroll];
#pragma unroll
    for (int u = 0; u < kSplitUnroll; ++u) {
      const int j = j0 + u * nthreads * 4;
      x[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (i < b && j < lim) {
        if (vec) {
          if (j < b) x[u] = *reinterpret_cast<const float4*>(src_row + j);
        } else {
          if (j + 0 < b) x[u].x = src_row[j + 0];
          if (j + 1 < b) x[u].y = src_row[j + 1];
          if (j + 2 < b) x[u].z = src_row[j + 2];
          if (j + 3 < b) x[u].w = src_row[j + 3];
        }
      }
    }
#pragma unroll
    for (int u = 0; u < kSplitUnroll; ++u) {
      const int j = j0 + u * nthreads * 4;
      if (j < lim) {
        float4 h, l;
        split4(x[u], h, l);
        *reinterpret_cast<float4*>(hi + j) = h;
        *reinterpret_cast<float4*>(lo + j) = l;
      }
    }
  }
}
#endif

}  // namespace swimg
