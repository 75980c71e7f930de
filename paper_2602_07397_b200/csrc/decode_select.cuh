// Bookkeeping shared by the three kernels of sw_decode_select (decode_duty.cu: Steps 2-4 per 64-column tile;
// decode_select.cu: the W stream of Step 5; decode_tail.cu: the per-sequence tail): tile sizes, the kernel
// parameter block, the chunk arithmetic of one sequence and the chunk -> CTA map.  No arithmetic of the method
// lives here.
#pragma once

#include "common.cuh"

namespace swds {

constexpr int kThreads = 256;         // streaming kernel
constexpr int kTailThreads = 1024;    // tail kernel
// duty kernel: tiles of 64 columns of the new score row
constexpr int kDutyThreads = 128;
constexpr int kDutyTile = 64;
constexpr int kDutyGroup = 1;         // tiles per CTA of the duty kernel
constexpr int kHeadRegs = 16;         // head values a thread holds while the loads of a tile are in flight
constexpr int kKU = 8;                // key-sketch float4s per thread and tile (64 columns x r <= 64)
// streaming kernel: chunk = kChunkRows rows x kTileW columns of the cached W = 16 KB; a row piece of a chunk is
// kTileW * 4 bytes of consecutive addresses (what a DRAM page likes), the pieces right of the diagonal are not read
#ifndef SW_DS_TILEW
#define SW_DS_TILEW 256
#endif
constexpr int kTileW = SW_DS_TILEW;
constexpr int kChunkBytes = 16384;
constexpr int kChunkRows = kChunkBytes / (kTileW * 4);
constexpr int kRho = kTileW / kChunkRows;              // row chunks per tile width
constexpr int kQuads = kTileW / 4;                     // float4 columns of a tile
constexpr int kRowGroups = kThreads / kQuads;          // threads that share a float4 column
constexpr int kRowsPerThread = kChunkRows / kRowGroups;
constexpr int kPieces = kChunkBytes / 16 / kThreads;   // 16-byte cp.async pieces per thread per chunk
#ifndef SW_DS_STAGES
#define SW_DS_STAGES 5
#endif
constexpr int kStages = SW_DS_STAGES; // ring of chunks: kStages x (16 KB + the chunk's r_prev values); two CTAs per SM
constexpr int kMaxBatch = 512;        // sequence lengths and per-sequence work counts live in shared memory
constexpr int kMaxTiles = 255;        // stream tiles per sequence the tail's slot table holds
static_assert(kChunkRows * kTileW * 4 == kChunkBytes && kChunkRows % kRowGroups == 0 && kTileW % kChunkRows == 0, "tile shape");

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
  int dtype, d;                      // of q / k_new
  int use_async;                     // W streamed by cp.async (needs 16-byte aligned rows), else plain loads
  int streamed;                      // the streaming kernel runs in front of the duty kernel (there is a walk state)
  // workspace
  float* ws_scores;                  // [batch][mbp] raw scores of the new row
  float* ws_part;                    // [g_stream + batch * tiles_max][kTileW] partial walk sums (see part_id)
  int mbp, tiles_max;                // mbp: max_blocks rounded up to kTileW; tiles_max = mbp / kTileW
  int g_stream;                      // grid of the streaming kernel (the tail derives the partial slots from it)
};

// Stream bookkeeping of one sequence.  Rows [0, b_q) of the cached W take part in Step 5 (row b_q is the new row,
// added by the tail).  Column tile c holds columns [c kTileW, (c + 1) kTileW); its rows above c kTileW are zero
// (lower-triangular), so it is streamed as rows [c kTileW, b_q) in chunks of kChunkRows: nr - c kRho chunks with
// nr = ceil(b_q / kChunkRows).  nt = ceil(b_q / kTileW) tiles have chunks.  No chunks without a walk (r_prev = NULL).
struct SeqInfo {
  int bq, nr, nt;
  __device__ __forceinline__ int chunks(int tile) const { return tile < nt ? nr - tile * kRho : 0; }
  __device__ __forceinline__ int chunks_before(int tile) const { return tile * nr - kRho * (tile * (tile - 1) / 2); }   // tile <= nt
  __device__ __forceinline__ int total_chunks() const { return chunks_before(nt); }
};
// A length outside [1, max_blocks B] marks an idle slot of the batch (sw.h: sw_decode_select): no chunks, no key
// update, no score row; the tail writes an empty selection for it.
__device__ __forceinline__ bool seq_live(int t, int B, int max_blocks) { return t >= 1 && (t - 1) / B < max_blocks; }
__device__ __forceinline__ SeqInfo seq_info(const int32_t* seqlens, int seq, int B, int max_blocks, bool walk) {
  SeqInfo s;
  const int t = seqlens[seq];                          // (a shared-memory copy in the streaming kernel)
  const bool live = seq_live(t, B, max_blocks);
  s.bq = live ? (t - 1) / B : 0;                       // block of the new token = b_curr
  s.nr = walk ? (s.bq + kChunkRows - 1) / kChunkRows : 0;
  s.nt = walk ? (s.bq + kTileW - 1) / kTileW : 0;
  return s;
}
// CTA that owns item g when T items are dealt to G CTAs as [i T / G, (i+1) T / G)
__device__ __forceinline__ int cta_of(long long g, int T, int G) {
  const long long num = (g + 1) * G - 1;
  return (num < (1ll << 31)) ? (int)((unsigned)num / (unsigned)T) : (int)(num / T);
}
// One partial (kTileW floats) per (tile, CTA that holds chunks of it).  Both the CTA index and the running tile
// index (tiles with chunks, counted over the batch) grow along the chunk order, so cta + tile_index is unique:
// the partials of a tile are the consecutive ids [first_cta + ti, last_cta + ti].
__device__ __forceinline__ int part_id(int cta, int tile_index) { return cta + tile_index; }

}  // namespace swds

namespace sw {
int32_t launch_decode_duty(const swds::Params& p, cudaStream_t st);
int32_t launch_decode_tail(const swds::Params& p, cudaStream_t st);
}
