// sw_decode_select: Alg. 2 Steps 2-6 for one new token per sequence: running key-block
// mean + sketches (Steps 2-3), the new row of W (Steps 3-4), the row-vector walk r^k = r^{k-1} W'^k (Step 5,
// SURVEY 8(a) row a6), the max-abs rescale (P9) and the top-tau selection (Step 6).  HBM-bound on the cached W
// (4 b^2/2 bytes per sequence).  Three kernels, chained as programmatic dependents:
//   this file         Step 5's stream: sum_{m < b_q} r_prev[m] W[m][j] over the whole grid, whatever the batch;
//   decode_duty.cu    Steps 2-4 per (sequence, 256 columns): sketches, running key mean, raw scores of the new row;
//   decode_tail.cu    per sequence: softmax, W_new = A^s (stored as row b_q of the cache), r, rescale, top-tau.
//
// The stream: the block-causal part of the cached W is cut into chunks of kChunkRows rows x kTileW columns (16 KB;
// column tile c = rows [c kTileW, b_q), the rows above are zero), numbered over all sequences tile by tile; CTA i
// takes the contiguous range [i T / G, (i+1) T / G) of the T chunks, streams it through a cp.async ring (the pieces
// right of the diagonal are not requested: zero fill), accumulates r_prev[m] W[m][j] over the chunks of one tile in
// registers and leaves one kTileW-float partial per (tile, CTA) in the workspace (fixed slots, fixed summation
// order: deterministic).  The r_prev values of a chunk's rows ride in the chunk's own cp.async group.
// A row piece of a chunk is kTileW * 4 = 1 KB of consecutive addresses: with 256-byte pieces (64-column tiles) the
// stream reached 70 % of the HBM bandwidth, DRAM pages being opened for a quarter of their content.
// The duty kernel is this kernel's programmatic dependent, released after griddepcontrol.wait here: its CTAs (two
// fit beside the two streaming CTAs of an SM) run beside the stream, which they neither read nor feed.
// DESIGN.md sec. 6.2 has the measurements behind these choices.
#include <algorithm>

#include "common.cuh"
#include "decode_select.cuh"
#include "sm100.cuh"

namespace {

using namespace swds;

__device__ __forceinline__ void cp_async16_zfill(uint32_t dst, const void* src, int bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }

__global__ void __launch_bounds__(kThreads, 2)
decode_stream_kernel(const Params p_in) {
  Params p = p_in;                                    // (the pointers to earlier kernels' data pass through pdl_wait)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = (int)gridDim.x, me = (int)blockIdx.x;
  const bool async = p.use_async;
  const int mb = p.max_blocks;

  extern __shared__ __align__(128) uint8_t smem_raw[];
  uint8_t* s_ring = smem_raw;                                          // [kStages][16 KB]
  float* s_rp = reinterpret_cast<float*>(s_ring + (size_t)kStages * kChunkBytes);   // [kStages][kChunkRows] r_prev of the chunk's rows
  float* s_part = s_rp + kStages * kChunkRows;                         // [kRowGroups][kTileW]
  __shared__ int s_pref[kMaxBatch + 1];                                // exclusive prefix of chunks per sequence
  __shared__ int s_tpref[kMaxBatch + 1];                               // exclusive prefix of tiles with chunks
  __shared__ int s_len[kMaxBatch];                                     // sequence lengths (read once from HBM)
  __shared__ int s_scan[2][kThreads / 32];

  // Launched as a programmatic dependent: nothing an earlier kernel of the stream may have written (the sequence
  // lengths included) is read before this wait, and the duty kernel is released behind this one's CTAs only after it.
  swd::pdl_wait(p.W, p.r_prev, p.seqlens);
  swd::pdl_launch_dependents();
  // ---- chunk and tile counts of all sequences: exclusive prefixes in shared memory ----------------------
  {
    constexpr int kPer = kMaxBatch / kThreads;
    static_assert(kMaxBatch % kThreads == 0, "the prefix pass gives every thread kMaxBatch / kThreads sequences");
    int vc[kPer], vt[kPer], sc = 0, st = 0;
#pragma unroll
    for (int e = 0; e < kPer; ++e) {
      const int sq = tid * kPer + e;
      vc[e] = 0; vt[e] = 0;
      if (sq < p.batch) {
        s_len[sq] = __ldcg(p.seqlens + sq);
        const SeqInfo si = seq_info(s_len, sq, p.B, mb, true);
        vc[e] = si.total_chunks(); vt[e] = si.nt;
      }
      sc += vc[e]; st += vt[e];
    }
    int ic = sc, it = st;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int uc = __shfl_up_sync(0xffffffffu, ic, o), ut = __shfl_up_sync(0xffffffffu, it, o);
      if (lane >= o) { ic += uc; it += ut; }
    }
    if (lane == 31) { s_scan[0][warp] = ic; s_scan[1][warp] = it; }
    __syncthreads();
    int bc = 0, bt = 0;
    for (int w = 0; w < warp; ++w) { bc += s_scan[0][w]; bt += s_scan[1][w]; }
    int rc = bc + ic - sc, rt = bt + it - st;
#pragma unroll
    for (int e = 0; e < kPer; ++e) {
      const int sq = tid * kPer + e;
      if (sq <= p.batch) { s_pref[sq] = rc; s_tpref[sq] = rt; }
      rc += vc[e]; rt += vt[e];
    }
    // the pass above covers sq <= kMaxBatch - 1: with a full batch (batch = kMaxBatch) the totals are the last
    // thread's running sums (sequences past the batch count zero)
    if (tid == kThreads - 1) { s_pref[kMaxBatch] = rc; s_tpref[kMaxBatch] = rt; }
    __syncthreads();
  }
  const int T = s_pref[p.batch];
  // chunks are dealt to the first Gc = min(G, T) CTAs, so that every one of them has at least one
  const int Gc = max(1, min(G, T));
  const int g_begin = me < Gc ? (int)((long long)me * T / Gc) : T, g_end = me < Gc ? (int)((long long)(me + 1) * T / Gc) : T;
  const int n_my = g_end - g_begin;
  if (n_my == 0) return;

  // ---- cursors over this CTA's chunks (thread-uniform).  The chunk loop is sensitive to its instruction count (a
  // few dozen extra integer instructions per chunk cost 3 us, measured), so a cursor carries what a step needs --
  // first row, chunks left in the tile, the tile's base pointers -- and recomputes only when it leaves a tile.
  struct Cursor {
    int seq, tile, chunk, n_tile, m0, bq;            // n_tile: chunks of the tile; m0: first row of the chunk
    const float* wt;                                 // &W[seq][0][tile kTileW]
    const float* rp;                                 // r_prev of the sequence
  };
  auto enter_tile = [&](Cursor& c, const SeqInfo& si) {
    c.n_tile = si.chunks(c.tile);
    c.bq = si.bq;
    c.m0 = c.tile * kTileW + c.chunk * kChunkRows;
    c.wt = p.W + (int64_t)c.seq * p.w_stride_seq + c.tile * kTileW;
    c.rp = p.r_prev + (int64_t)c.seq * mb;
  };
  auto locate = [&](int g) {
    Cursor c;
    int lo = 0, hi = p.batch - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (s_pref[mid] <= g) lo = mid; else hi = mid - 1; }
    c.seq = lo;
    const SeqInfo si = seq_info(s_len, c.seq, p.B, mb, true);
    const int local = g - s_pref[c.seq];
    int tl = 0, th = max(si.nt - 1, 0);
    while (tl < th) { const int mid = (tl + th + 1) >> 1; if (si.chunks_before(mid) <= local) tl = mid; else th = mid - 1; }
    c.tile = tl;
    c.chunk = local - si.chunks_before(tl);
    enter_tile(c, si);
    return c;
  };
  auto advance = [&](Cursor& c) {
    ++c.chunk;
    c.m0 += kChunkRows;
    if (c.chunk < c.n_tile) return;
    SeqInfo si = seq_info(s_len, c.seq, p.B, mb, true);
    c.chunk = 0;
    ++c.tile;
    while (c.seq < p.batch && c.tile >= si.nt) {     // next sequence that has chunks
      c.tile = 0;
      if (++c.seq < p.batch) si = seq_info(s_len, c.seq, p.B, mb, true);
    }
    if (c.seq < p.batch) enter_tile(c, si);
  };
  Cursor cc = locate(g_begin), pc = cc;

  // ---- W stream: chunk = rows [m0, m0 + kChunkRows) x columns [tile kTileW, +kTileW) --------------------------
  // piece u of a thread: row rr_u = (u kThreads + tid) / kQuads of the chunk, float4 column tid % kQuads
  const int q4 = (tid % kQuads) * 4, rr0 = tid / kQuads;
  int p_left = n_my, issued = 0;
  auto issue_next = [&]() {                           // all threads: request the next chunk (or an empty group)
    if (p_left > 0) {
      const int st = issued % kStages;
      const uint32_t dst = sm100::smem_u32(s_ring + (size_t)st * kChunkBytes) + tid * 16;
      const float* src = pc.wt + (int64_t)pc.m0 * mb + q4;
      const int c4 = pc.tile * kTileW + q4;
#pragma unroll
      for (int u = 0; u < kPieces; ++u) {
        const int rr = rr0 + u * (kThreads / kQuads), m = pc.m0 + rr;
        // rows >= b_q are not part of the product; W[m][j] = 0 for j > m (block-causal): not requested
        const bool ok = m < pc.bq && c4 <= m && c4 < mb;
        cp_async16_zfill(dst + u * (kThreads * 16), ok ? src + rr * mb : pc.wt, ok ? 16 : 0);
      }
      if (tid < kChunkRows / 4) {
        const int m = pc.m0 + tid * 4;
        const bool ok = m < mb;
        cp_async16_zfill(sm100::smem_u32(s_rp + st * kChunkRows + tid * 4), ok ? pc.rp + m : pc.rp, ok ? 16 : 0);
      }
      ++issued; advance(pc); --p_left;
    }
    cp_async_commit();
  };
  if (async)
    for (int i = 0; i < kStages - 1; ++i) issue_next();

  // ---- Step 5, r_prev[m] W[m][j] over this CTA's range ---------------------------------------------------------
  int consumed = 0;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  const int cq = tid % kQuads, rg = tid / kQuads;
  for (int it = 0; it < n_my; ++it) {
    const int seq = cc.seq, tile = cc.tile, m0 = cc.m0;
    const int rows = min(kChunkRows, cc.bq - m0);     // rows >= b_q are not part of the product
    if (async) {
      asm volatile("cp.async.wait_group %0;" ::"n"(kStages - 2) : "memory");   // chunk `consumed` landed
      __syncthreads();                                // ... for every thread; the previous chunk is fully consumed
      issue_next();                                   // refill the stage the previous chunk occupied
      const int st = consumed % kStages;
      const float* box = reinterpret_cast<const float*>(s_ring + (size_t)st * kChunkBytes);
      const float* rp = s_rp + st * kChunkRows;
#pragma unroll
      for (int u = 0; u < kRowsPerThread; ++u) {
        const int rr = rg + u * kRowGroups;
        if (rr < rows) {
          const float4 v = *reinterpret_cast<const float4*>(box + rr * kTileW + cq * 4);
          const float a = rp[rr];
          acc.x = fmaf(a, v.x, acc.x);
          acc.y = fmaf(a, v.y, acc.y);
          acc.z = fmaf(a, v.z, acc.z);
          acc.w = fmaf(a, v.w, acc.w);
        }
      }
      ++consumed;
    } else {
      const float* Wm = p.W + (int64_t)seq * p.w_stride_seq;
      const int c4 = tile * kTileW + cq * 4;
      for (int rr = rg; rr < rows; rr += kRowGroups) {
        const int m = m0 + rr;
        const float a = __ldcg(cc.rp + m);
        const float* wr = Wm + (int64_t)m * mb;
        if (c4 + 0 <= m) acc.x = fmaf(a, __ldcg(wr + c4 + 0), acc.x);
        if (c4 + 1 <= m) acc.y = fmaf(a, __ldcg(wr + c4 + 1), acc.y);
        if (c4 + 2 <= m) acc.z = fmaf(a, __ldcg(wr + c4 + 2), acc.z);
        if (c4 + 3 <= m) acc.w = fmaf(a, __ldcg(wr + c4 + 3), acc.w);
      }
    }
    if (it == n_my - 1 || cc.chunk + 1 >= cc.n_tile) {
      // one partial per (tile, CTA)
      *reinterpret_cast<float4*>(s_part + rg * kTileW + cq * 4) = acc;
      __syncthreads();
      if (tid < kTileW) {
        float v = 0.f;
#pragma unroll
        for (int g = 0; g < kRowGroups; ++g) v += s_part[g * kTileW + tid];      // fixed order
        p.ws_part[(int64_t)part_id(me, s_tpref[seq] + tile) * kTileW + tid] = v;
      }
      __syncthreads();
      acc = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    advance(cc);
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// upper bound of the chunks of one sequence (b_q = max_blocks - 1)
static int max_chunks_per_seq(int max_blocks) {
  const int bq = std::max(max_blocks - 1, 0);
  const int nr = sw::cdiv(bq, kChunkRows), nt = sw::cdiv(bq, kTileW);
  return nt * nr - kRho * (nt * (nt - 1) / 2);
}
constexpr int kMaxStreamGrid = 512;

}  // namespace

namespace sw {

size_t decode_select_ws_bytes(int batch, int max_blocks) {
  const size_t tiles = (size_t)cdiv(max_blocks, kTileW), mbp = tiles * kTileW;
  return 256 + sizeof(float) * (size_t)batch * mbp + sizeof(float) * ((size_t)kMaxStreamGrid + (size_t)batch * tiles) * kTileW;
}

int32_t launch_decode_select(const DecodeSelectArgs& a, cudaStream_t st) {
  if (a.batch == 0) return SW_OK;
  if (a.batch > kMaxBatch) return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: batch %d > %d", a.batch, kMaxBatch);
  if (cdiv(a.max_blocks, kTileW) > kMaxTiles)
    return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: max_blocks %d too large", a.max_blocks);
  const size_t need = decode_select_ws_bytes(a.batch, a.max_blocks);
  if (a.ws == nullptr || a.ws_bytes < need)
    return fail(SW_ERR_WORKSPACE, "sw_decode_select: workspace %zu < %zu bytes", a.ws_bytes, need);
  Params p;
  p.q = a.q.ptr; p.q_stride_seq = a.q.stride_tok; p.q_stride_head = a.q.stride_head; p.h_q = a.q.heads;
  p.k = a.k.ptr; p.k_stride_seq = a.k.stride_tok; p.k_stride_head = a.k.stride_head; p.h_kv = a.k.heads;
  p.dtype = a.q.dtype; p.d = a.q.d;
  p.seqlens = a.seqlens; p.signs = a.signs; p.cols = a.cols; p.r = a.r; p.scale = a.scale;
  p.inv_sqrt_r = 1.0f / sqrtf((float)a.r);
  p.s = a.s; p.flags = a.flags; p.kbar = a.kbar; p.ks = a.ks; p.W = a.W_cache; p.w_stride_seq = a.stride_seq;
  p.r_prev = a.r_prev; p.r_out = a.r_out; p.tau = a.tau; p.tau_max = a.tau_max; p.idx = a.idx; p.count = a.count;
  p.batch = a.batch; p.B = a.block; p.max_blocks = a.max_blocks;
  p.tiles_max = cdiv(a.max_blocks, kTileW); p.mbp = p.tiles_max * kTileW;
  uint8_t* w = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(a.ws) + 255) & ~(uintptr_t)255);
  p.ws_scores = reinterpret_cast<float*>(w);
  w += sizeof(float) * (size_t)a.batch * p.mbp;
  p.ws_part = reinterpret_cast<float*>(w);
  const long long work = (long long)a.batch * max_chunks_per_seq(a.max_blocks);
  p.g_stream = (int)std::max<long long>(1, std::min<long long>(work, std::min(2 * num_sms(), kMaxStreamGrid)));
  // cp.async stream of the cached W (and of r_prev) needs 16-byte aligned row pieces; otherwise plain loads
  p.use_async = a.r_prev != nullptr && aligned16(a.W_cache) && aligned16(a.r_prev) && (a.max_blocks & 3) == 0 &&
                (a.stride_seq & 3) == 0;

  // launch 1: the W stream of Step 5 (nothing to stream without a walk state)
  p.streamed = (a.r_prev != nullptr && a.max_blocks > 1) ? 1 : 0;
  if (p.streamed) {
    const size_t smem = (size_t)kStages * kChunkBytes + sizeof(float) * ((size_t)kStages * kChunkRows + (size_t)kRowGroups * kTileW);
    if (int32_t rc = allow_dynamic_smem(decode_stream_kernel, smem, "sw_decode_select(stream) smem attribute")) return rc;
    count_launch();
    launch_pdl(decode_stream_kernel, dim3(p.g_stream), dim3(kThreads), smem, st, p);
    if (int32_t rc = check_launch("sw_decode_select(stream)")) return rc;
  }
  // launch 2: Steps 2-4 (sketches, running key mean, raw score row), beside the stream
  if (int32_t rc = launch_decode_duty(p, st)) return rc;
  // launch 3: per-sequence tail
  return launch_decode_tail(p, st);
}

}  // namespace sw
