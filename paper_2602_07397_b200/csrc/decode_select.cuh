// Bookkeeping shared by the two kernels of sw_decode_select (decode_select.cu: duties + W stream;
// decode_tail.cu: the per-sequence tail): tile sizes, the kernel parameter block, the chunk / duty arithmetic of
// one sequence and the chunk -> CTA map.  No arithmetic of the method lives here.
#pragma once

#include "common.cuh"

namespace swds {

constexpr int kThreads = 256;         // streaming kernel
constexpr int kTailThreads = 1024;    // tail kernel
constexpr int kTile = 64;            // columns per tile
constexpr int kRowGroups = 16;       // row lanes of the vector-matrix product
constexpr int kChunkRows = 64;
constexpr int kStages = 4;            // 4 x 16 KB ring + two r_prev rows + the prefix tables: two CTAs per SM
constexpr int kChunkBytes = kChunkRows * kTile * 4;
constexpr int kPieces = kChunkBytes / 16 / kThreads;     // 16-byte cp.async pieces per thread per chunk
constexpr int kMaxBatch = 512;       // sequence lengths and per-sequence work counts live in shared memory
constexpr int kMaxTiles = 255;       // column tiles per sequence (max_blocks <= 16320)
constexpr int kHeadRegs = 16;        // head values a thread holds while the loads of a duty are in flight
constexpr int kKU = 4;               // key-sketch float4s per thread and duty (64 columns x r <= 64)

struct Params {
  const void* q;  int64_t q_stride_seq, q_stride_head;  int h_q;
  const void* k;  int64_t k_stride_seq, k_stride_head;  int h_kv;
  const int32_t* seqlens;
  const int8_t* signs;  const int32_t* cols;  int r;  float scale;  float inv_sqrt_r;
  int s;  uint32_t flags;
  float* kbar;  float* ks;
  float* W;  int64_t w_stride_seq;
  const float* r_prev;  float* r_out;
  const int32_t* tau;  int tau_max;
  int32_t* idx;  int32_t* count;
  int batch, B, max_blocks;
  int use_async;                     // W streamed by cp.async (needs 16-byte aligned rows), else plain loads
  // workspace
  float* ws_scores;                  // [batch][mbp] raw scores of the new row
  float* ws_part;                    // [batch][tiles_max][slots][64] partial walk sums
  int mbp, tiles_max, slots;
  int g_stream;                      // grid of the streaming kernel (the tail derives the partial slots from it)
};

// Work bookkeeping of one sequence.  b_q = 64 a + e; column tile c < a has rows [64 c, b_q): a - c + (e > 0)
// chunks; tile a (the one that holds b_q) has (e > 0) chunks.  a + 1 duties.  No chunks without a walk
// (r_prev = NULL).
struct SeqInfo {
  int bq, a, eps;
  __device__ __forceinline__ int chunks(int tile, bool walk) const { return walk ? (tile < a ? a - tile + eps : eps) : 0; }
  __device__ __forceinline__ int chunks_before(int tile, bool walk) const {        // tile <= a
    return walk ? tile * a - tile * (tile - 1) / 2 + tile * eps : 0;
  }
  __device__ __forceinline__ int total_chunks(bool walk) const { return walk ? a * (a + 1) / 2 + a * eps + eps : 0; }
  __device__ __forceinline__ int duties() const { return a + 1; }
};
__device__ __forceinline__ SeqInfo seq_info(const int32_t* seqlens, int seq, int B) {
  SeqInfo s;
  const int t = seqlens[seq];                          // (a shared-memory copy after the first pass)
  s.bq = (t - 1) / B;                                  // block of the new token = b_curr
  s.a = s.bq / kTile;
  s.eps = (s.bq % kTile) != 0;
  return s;
}
// CTA that owns item g when T items are dealt to G CTAs as [i T / G, (i+1) T / G)
__device__ __forceinline__ int cta_of(long long g, int T, int G) {
  const long long num = (g + 1) * G - 1;
  return (num < (1ll << 31)) ? (int)((unsigned)num / (unsigned)T) : (int)(num / T);
}


}  // namespace swds

namespace sw {
int32_t launch_decode_tail(const swds::Params& p, cudaStream_t st);
}
