// Feature-space sketch helpers shared by sketch.cu and decode_select.cu: in-warp fast Walsh-Hadamard
// transform and the sign-flip -> FWHT -> column-pick -> scale tail of Alg. 1 Step 4 (
// SRHT of Lemma A.6; readings P1, P2).
#pragma once

#include <stdint.h>

namespace swsk {

// In-warp FWHT of a d-vector held as EPL = d/32 consecutive elements per lane
// (element x = lane*EPL + e), natural (Sylvester) order: y[x] = sum_z v[z] (-1)^popcount(x&z).
template <int EPL>
__device__ __forceinline__ void fwht_warp(float (&v)[EPL], int lane) {
#pragma unroll
  for (int h = 1; h < EPL; h <<= 1) {
#pragma unroll
    for (int e = 0; e < EPL; ++e) {
      if ((e & h) == 0) {
        float a = v[e], b = v[e | h];
        v[e] = a + b;
        v[e | h] = a - b;
      }
    }
  }
#pragma unroll
  for (int m = 1; m < 32; m <<= 1) {
#pragma unroll
    for (int e = 0; e < EPL; ++e) {
      float other = __shfl_xor_sync(0xffffffffu, v[e], m);
      v[e] = (lane & m) ? (other - v[e]) : (v[e] + other);
    }
  }
}

// Shared tail: one warp (warp_id) turns the d-vector in s_vec into the r-vector of the sketch.
// signs / cols may live in global or shared memory (SG: int8_t or float elements; null = +1).
template <int D, typename SG>
__device__ __forceinline__ void sketch_tail(float* s_vec, const SG* signs, const int32_t* cols, int r, float scale,
                                            float* out_row, float* out_row2 = nullptr, int warp_id = 0) {
  constexpr int EPL = D / 32;
  const int lane = threadIdx.x & 31;
  if ((threadIdx.x >> 5) == warp_id) {
    float v[EPL];
#pragma unroll
    for (int e = 0; e < EPL; ++e) {
      int x = lane * EPL + e;
      float sg = signs ? (float)signs[x] : 1.f;
      v[e] = s_vec[x] * sg;
    }
    fwht_warp<EPL>(v, lane);
    __syncwarp();
#pragma unroll
    for (int e = 0; e < EPL; ++e) s_vec[lane * EPL + e] = v[e];
    __syncwarp();
    for (int c = lane; c < r; c += 32) {
      const float y = s_vec[cols[c]] * scale;
      out_row[c] = y;
      if (out_row2) out_row2[c] = y;
    }
  }
}

}  // namespace swsk
