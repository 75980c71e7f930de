// sw_decode_select: Alg. 2 Steps 2-6 for one new token per sequence: running key-block
// mean + sketches (Steps 2-3), the new row of W (Steps 3-4), the row-vector walk r^k = r^{k-1} W'^k (Step 5,
// SURVEY 8(a) row a6), the max-abs rescale (P9) and the top-tau selection (Step 6).  HBM-bound on the cached W
// (4 b^2/2 bytes per sequence).  Two kernels; this file holds the first: everything that touches HBM-sized data.
//
// The whole grid (two CTAs per SM) works on the batch, whatever its size.  Two kinds of work are dealt out:
//  * chunks: 64 rows x 64 columns of the block-causal part of the cached W (rows [64 c, b_q) of column tile
//    c), numbered over all sequences; CTA i streams the contiguous range [i T / G, (i+1) T / G) of the T
//    chunks through a cp.async ring, accumulates r_prev[m] W[m][j] over the chunks of one column tile in
//    registers and leaves one 64-float partial per (tile, CTA) in the workspace (fixed slots, fixed
//    summation order: deterministic);
//  * duties: one per (sequence, column tile), dealt the same way: q~_t (and, on the tile that holds b_q, the
//    running key-block mean and its sketch) and the raw scores of the tile's 64 columns.
// A CTA runs its duties first.  Every load they need (head values, key-sketch rows, the old mean) and the
// r_prev rows of the stream are requested BEFORE the first chunks of the W stream: on an SM that keeps
// ~160 KB of the stream in flight a load issued behind it waits ~3 us (queue depth / per-SM bandwidth).
// The second kernel (decode_tail.cu, one CTA of 1024 threads per sequence, launched as a programmatic dependent
// so that it becomes resident while the last CTAs of this one drain) turns the raw score row and the partial
// sums into W_new = A^s, r, the rescaled r_out and the block list.  An earlier version ran that tail on the last
// CTA to finish a sequence (one launch, a completion counter in the workspace): 256 threads made the radix
// select and the row passes a 12 us serial chain (two warps per scheduler: every pass is bound by the dependent
// issue latency), a quarter of a decode layer; 1024 threads do it in a fraction of that.
// DESIGN.md sec. 6.2 has the measurements behind these choices.
#include <algorithm>

#include "common.cuh"
#include "decode_select.cuh"
#include "sketch_common.cuh"
#include "sm100.cuh"

namespace {

using namespace swds;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }

template <typename TIn, int D>
__global__ void __launch_bounds__(kThreads, 2)
decode_select_kernel(const Params p) {
  // the tail kernel is launched as a programmatic dependent: let it become resident as SMs drain
  swd::pdl_launch_dependents();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = (int)gridDim.x, me = (int)blockIdx.x;
  const bool walk = p.r_prev != nullptr;
  const bool async = walk && p.use_async;
  const int mb = p.max_blocks;
  const int rstride = p.mbp + kChunkRows;

  extern __shared__ __align__(128) uint8_t smem_raw[];
  float* s_rprev = reinterpret_cast<float*>(smem_raw);                 // [2][mbp + 64] r_prev of two sequences
  float* s_part = s_rprev + 2 * rstride;                               // [kRowGroups][64]
  uint8_t* s_ring = reinterpret_cast<uint8_t*>(
      (reinterpret_cast<uintptr_t>(s_part + kRowGroups * kTile) + 127) & ~(uintptr_t)127);   // [kStages][16 KB]
  __shared__ __align__(16) float s_vec[D], s_qt[128], s_kt[128], s_sign[D];
  __shared__ float s_hx[kThreads / D][D];
  __shared__ int32_t s_cols[128];
  __shared__ int s_pref[kMaxBatch + 1];                                // exclusive prefix of chunks per sequence
  __shared__ int s_dpref[kMaxBatch + 1];                               // exclusive prefix of duties per sequence
  __shared__ int s_len[kMaxBatch];                                     // sequence lengths (read once from HBM)
  __shared__ int s_scan[2][kThreads / 32];

  // ---- chunk and duty counts of all sequences: exclusive prefixes in shared memory -------------------
  {
    constexpr int kPer = kMaxBatch / kThreads;
    int vc[kPer], vd[kPer], sc = 0, sd = 0;
#pragma unroll
    for (int e = 0; e < kPer; ++e) {
      const int sq = tid * kPer + e;
      vc[e] = 0; vd[e] = 0;
      if (sq < p.batch) {
        s_len[sq] = __ldg(p.seqlens + sq);
        const SeqInfo si = seq_info(s_len, sq, p.B);
        vc[e] = si.total_chunks(walk); vd[e] = si.duties();
      }
      sc += vc[e]; sd += vd[e];
    }
    int ic = sc, id = sd;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int uc = __shfl_up_sync(0xffffffffu, ic, o), ud = __shfl_up_sync(0xffffffffu, id, o);
      if (lane >= o) { ic += uc; id += ud; }
    }
    if (lane == 31) { s_scan[0][warp] = ic; s_scan[1][warp] = id; }
    if (tid < D) s_sign[tid] = p.signs ? (float)p.signs[tid] : 1.f;
    if (tid < p.r && tid < 128) s_cols[tid] = p.cols[tid];
    __syncthreads();
    int bc = 0, bd = 0;
    for (int w = 0; w < warp; ++w) { bc += s_scan[0][w]; bd += s_scan[1][w]; }
    int rc = bc + ic - sc, rd = bd + id - sd;
#pragma unroll
    for (int e = 0; e < kPer; ++e) {
      const int sq = tid * kPer + e;
      if (sq <= p.batch) { s_pref[sq] = rc; s_dpref[sq] = rd; }
      rc += vc[e]; rd += vd[e];
    }
    __syncthreads();
  }
  const int T = s_pref[p.batch], ND = s_dpref[p.batch];
  // chunks are dealt to the first Gc = min(G, T) CTAs, so that every one of them has at least one: the partial
  // slots of a tile (one per CTA that shares it) are then contiguous
  const int Gc = max(1, min(G, T));
  const int g_begin = me < Gc ? (int)((long long)me * T / Gc) : T, g_end = me < Gc ? (int)((long long)(me + 1) * T / Gc) : T;
  const int d_begin = (int)((long long)me * ND / G), d_end = (int)((long long)(me + 1) * ND / G);
  const int n_my = g_end - g_begin;
  if (n_my == 0 && d_begin == d_end) return;

  auto find_seq = [&](const int* pref, int g) {
    int lo = 0, hi = p.batch - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (pref[mid] <= g) lo = mid; else hi = mid - 1; }
    return lo;
  };

  // ---- cursors over this CTA's chunks (thread-uniform) ------------------------------------------------
  struct Cursor { int seq, tile, chunk; SeqInfo si; };
  auto locate = [&](int g) {
    Cursor c;
    c.seq = find_seq(s_pref, g);
    c.si = seq_info(s_len, c.seq, p.B);
    const int local = g - s_pref[c.seq];
    int tl = 0, th = c.si.a;
    while (tl < th) { const int mid = (tl + th + 1) >> 1; if (c.si.chunks_before(mid, walk) <= local) tl = mid; else th = mid - 1; }
    c.tile = tl;
    c.chunk = local - c.si.chunks_before(tl, walk);
    return c;
  };
  auto advance = [&](Cursor& c) {
    ++c.chunk;
    while (c.seq < p.batch && c.chunk >= c.si.chunks(c.tile, walk)) {
      c.chunk = 0;
      if (++c.tile > c.si.a) {
        c.tile = 0;
        if (++c.seq < p.batch) c.si = seq_info(s_len, c.seq, p.B);
      }
    }
  };
  Cursor cc, pc;
  cc.seq = cc.tile = cc.chunk = 0; cc.si.bq = cc.si.a = cc.si.eps = 0;
  int seq_first = 0;
  if (n_my > 0) { cc = locate(g_begin); seq_first = cc.seq; }
  pc = cc;

  // Launched as a programmatic dependent itself: what is above (work prefixes, cursors; sequence lengths only)
  // overlaps the tail of the kernel before this one; everything below reads what earlier kernels produced.
  swd::pdl_wait();

  // ---- W stream: chunk = rows [64 tile + 64 chunk, +64) x columns [64 tile, +64) of the sequence's cached W
  int p_left = n_my, issued = 0;
  auto issue_next = [&]() {                           // all threads: request the next chunk (or an empty group)
    if (p_left > 0) {
      const float* Wseq = p.W + (int64_t)pc.seq * p.w_stride_seq;
      const int m0 = (pc.tile + pc.chunk) * kTile;
      const uint32_t dst = sm100::smem_u32(s_ring + (size_t)(issued % kStages) * kChunkBytes);
#pragma unroll
      for (int u = 0; u < kPieces; ++u) {
        const int pcs = u * kThreads + tid, rr = pcs >> 4, c4 = pc.tile * kTile + (pcs & 15) * 4;
        if (m0 + rr < pc.si.bq && c4 < mb)            // rows >= b_q / columns >= max_blocks are never read
          cp_async16(dst + pcs * 16, Wseq + (int64_t)(m0 + rr) * mb + c4);
      }
      ++issued; advance(pc); --p_left;
    }
    cp_async_commit();
  };
  // r_prev of the first two sequences of this CTA's chunk range (group 0 of the cp.async stream), then the
  // first kStages - 1 chunks.  Called once, after the loads of the last duty have been issued.
  auto start_stream = [&]() {
    if (n_my == 0) return;                            // (no chunks without a walk)
    for (int q2 = 0; q2 < 2; ++q2) {
      const int sq = seq_first + q2;
      if (sq < p.batch && (q2 == 0 || s_pref[sq] < g_end)) {
        const float* rp = p.r_prev + (int64_t)sq * mb;
        if (async)
          for (int i = tid * 4; i < mb; i += kThreads * 4) cp_async16(sm100::smem_u32(s_rprev + q2 * rstride + i), rp + i);
        else
          for (int i = tid; i < mb; i += kThreads) s_rprev[q2 * rstride + i] = __ldg(rp + i);
      }
    }
    if (async) {
      cp_async_commit();
      for (int i = 0; i < kStages - 1; ++i) issue_next();
    }
  };

  // ================= duties: Steps 2-4 for one column tile each ==========================================
  constexpr int kGroups = kThreads / D;
  const int q4 = p.r >> 2;                            // float4s per sketch row
  const bool vec_ok = (p.r & 3) == 0 && q4 >= 1 && q4 <= 32 && (q4 & (q4 - 1)) == 0 && kTile * q4 <= kKU * kThreads &&
                      (reinterpret_cast<uintptr_t>(p.ks) & 15u) == 0;
  const int hx = tid % D, hg = tid / D;
  int qt_seq = -1;
  bool stream_started = false;
  for (int dty = d_begin; dty < d_end; ++dty) {
    const int seq = find_seq(s_dpref, dty), tile = dty - s_dpref[seq];
    const SeqInfo si = seq_info(s_len, seq, p.B);
    const int bq = si.bq, hi = bq + 1, col0 = tile * kTile;
    const bool need_q = qt_seq != seq, need_k = tile == si.a;   // tile a owns the key-side update of Step 2
    const float* ksb = p.ks + (int64_t)seq * mb * p.r;
    const int part = vec_ok ? (tid & (q4 - 1)) : 0, per_pass = vec_ok ? kThreads / q4 : 1;
    const int colq = vec_ok ? tid / q4 : 0;
    // ---- all loads of the duty, before anything waits on memory: unconditional loads from clamped (always
    // valid) addresses, raw values kept in registers -- a predicated load followed by its convert made every
    // group of loads wait for the previous one (5 us instead of one memory latency)
    TIn qraw[kHeadRegs], kraw[kHeadRegs];
    float4 kv[kKU];
    const TIn* qp = reinterpret_cast<const TIn*>(p.q) + (int64_t)seq * p.q_stride_seq + hx;
    const TIn* kp = reinterpret_cast<const TIn*>(p.k) + (int64_t)seq * p.k_stride_seq + hx;
#pragma unroll
    for (int u = 0; u < kHeadRegs; ++u) {
      const int h = hg + u * kGroups;
      qraw[u] = qp[(int64_t)min(h, p.h_q - 1) * p.q_stride_head];
      kraw[u] = kp[(int64_t)min(h, p.h_kv - 1) * p.k_stride_head];
    }
    const int cnt = (s_len[seq] - 1) % p.B;                        // tokens already in block b_curr
    float* kb = p.kbar + ((int64_t)seq * mb + bq) * D;
    const float kbar_old = kb[tid & (D - 1)];
#pragma unroll
    for (int u = 0; u < kKU; ++u) {
      const int cj = u * per_pass + colq;
      const int j = min(col0 + min(cj, kTile - 1), bq);                        // clamped: always a valid row
      kv[u] = vec_ok ? *reinterpret_cast<const float4*>(ksb + (int64_t)j * p.r + part * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (dty == d_end - 1) { start_stream(); stream_started = true; }
    // ---- head means, running key-block mean, sketches ----------------------------------------------------
    if (need_q || need_k) {
      float sq = 0.f, sk = 0.f;
#pragma unroll
      for (int u = 0; u < kHeadRegs; ++u) {
        const int h = hg + u * kGroups;
        if (h < p.h_q) sq += (float)qraw[u];
        if (h < p.h_kv) sk += (float)kraw[u];
      }
      if (need_q) for (int h = hg + kHeadRegs * kGroups; h < p.h_q; h += kGroups) sq += (float)qp[(int64_t)h * p.q_stride_head];
      if (need_k) for (int h = hg + kHeadRegs * kGroups; h < p.h_kv; h += kGroups) sk += (float)kp[(int64_t)h * p.k_stride_head];
      if (need_q) {
        s_hx[hg][hx] = sq;
        __syncthreads();
        if (tid < D) {
          float a = 0.f;
#pragma unroll
          for (int g = 0; g < kGroups; ++g) a += s_hx[g][tid];
          s_vec[tid] = a / (float)p.h_q;
        }
        __syncthreads();
        swsk::sketch_tail<D>(s_vec, s_sign, s_cols, p.r, p.scale, s_qt);         // q~_t
        qt_seq = seq;
        __syncthreads();
      }
      if (need_k) {
        s_hx[hg][hx] = sk;
        __syncthreads();
        if (tid < D) {
          float a = 0.f;
#pragma unroll
          for (int g = 0; g < kGroups; ++g) a += s_hx[g][tid];
          const float avg = a / (float)p.h_kv;
          const float mn = (cnt == 0) ? avg : ((float)cnt * kbar_old + avg) / (float)(cnt + 1);
          kb[tid] = mn;
          s_vec[tid] = mn;
        }
        __syncthreads();
        swsk::sketch_tail<D>(s_vec, s_sign, s_cols, p.r, p.scale, s_kt, p.ks + ((int64_t)seq * mb + bq) * p.r);
        __syncthreads();
      }
    }
    // ---- raw scores of the tile's columns (Steps 3-4; column b_q from the fresh sketch) --------------------
    float* sc = p.ws_scores + (int64_t)seq * p.mbp;
    if (vec_ok) {
      // q4 adjacent lanes share one column; partial dots meet in a fixed xor butterfly
      const float4 qv = *reinterpret_cast<const float4*>(s_qt + part * 4);
#pragma unroll
      for (int u = 0; u < kKU; ++u) {
        if (u * per_pass >= kTile) break;                                        // warp-uniform
        const int cj = u * per_pass + colq, j = col0 + cj;
        if (j == bq) kv[u] = *reinterpret_cast<const float4*>(s_kt + part * 4);
        float a = fmaf(qv.w, kv[u].w, fmaf(qv.z, kv[u].z, fmaf(qv.y, kv[u].y, qv.x * kv[u].x)));
        for (int o = q4 >> 1; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if (part == 0 && cj < kTile && j < hi) sc[j] = a * p.inv_sqrt_r;
      }
    } else {
      for (int cj = warp; cj < kTile; cj += kThreads / 32) {
        const int j = col0 + cj;
        if (j < hi) {
          const float* kr = (j == bq) ? s_kt : ksb + (int64_t)j * p.r;
          float a = 0.f;
          for (int c = lane; c < p.r; c += 32) a = fmaf(s_qt[c], kr[c], a);
          a = swd::warp_sum(a);
          if (lane == 0) sc[j] = a * p.inv_sqrt_r;
        }
      }
    }
  }
  if (!stream_started) start_stream();

  // ================= chunks: Step 5, r_prev[m] W[m][j] over this CTA's range ===============================
  int cur_seq = -1, consumed = 0;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  const int cq = tid & 15, rg = tid >> 4;
  const float* rprev_cur = s_rprev;
  for (int it = 0; it < n_my; ++it) {
    const SeqInfo& si = cc.si;
    const int seq = cc.seq, tile = cc.tile, bq = si.bq;
    if (seq != cur_seq) {
      cur_seq = seq;
      const int slot2 = seq - seq_first;
      if (slot2 < 2) {
        rprev_cur = s_rprev + slot2 * rstride;        // requested up front
      } else {                                        // a range over more than two (tiny) sequences: reload
        __syncthreads();
        const float* rp = p.r_prev + (int64_t)seq * mb;
        for (int i = tid; i < mb; i += kThreads) s_rprev[i] = __ldg(rp + i);
        rprev_cur = s_rprev;
        __syncthreads();
      }
    }
    const int m0 = (tile + cc.chunk) * kTile;
    const int rows = min(kChunkRows, bq - m0);        // rows >= b_q are not part of the product
    if (async) {
      asm volatile("cp.async.wait_group %0;" ::"n"(kStages - 2) : "memory");   // chunk `consumed` (and r_prev) landed
      __syncthreads();                                // ... for every thread; the previous chunk is fully consumed
      issue_next();                                   // refill the stage the previous chunk occupied
      const float* box = reinterpret_cast<const float*>(s_ring + (size_t)(consumed % kStages) * kChunkBytes);
#pragma unroll
      for (int u = 0; u < kChunkRows / kRowGroups; ++u) {
        const int rr = rg + u * kRowGroups;
        if (rr < rows) {
          const float4 v = *reinterpret_cast<const float4*>(box + rr * kTile + cq * 4);
          const float a = rprev_cur[m0 + rr];
          acc.x = fmaf(a, v.x, acc.x);
          acc.y = fmaf(a, v.y, acc.y);
          acc.z = fmaf(a, v.z, acc.z);
          acc.w = fmaf(a, v.w, acc.w);
        }
      }
      ++consumed;
    } else {
      if (it == 0) __syncthreads();                   // s_rprev is complete
      const float* Wm = p.W + (int64_t)seq * p.w_stride_seq;
      const int c4 = tile * kTile + cq * 4;
      for (int rr = rg; rr < rows; rr += kRowGroups) {
        const float a = rprev_cur[m0 + rr];
        const float* wr = Wm + (int64_t)(m0 + rr) * mb;
        if (c4 + 0 < mb) acc.x = fmaf(a, __ldg(wr + c4 + 0), acc.x);
        if (c4 + 1 < mb) acc.y = fmaf(a, __ldg(wr + c4 + 1), acc.y);
        if (c4 + 2 < mb) acc.z = fmaf(a, __ldg(wr + c4 + 2), acc.z);
        if (c4 + 3 < mb) acc.w = fmaf(a, __ldg(wr + c4 + 3), acc.w);
      }
    }
    if (it == n_my - 1 || cc.chunk + 1 >= si.chunks(tile, walk)) {
      // one partial per (tile, CTA): slot = rank of this CTA among the CTAs that share the tile
      *reinterpret_cast<float4*>(s_part + rg * kTile + cq * 4) = acc;
      __syncthreads();
      if (tid < kTile) {
        float v = 0.f;
#pragma unroll
        for (int g = 0; g < kRowGroups; ++g) v += s_part[g * kTile + tid];      // fixed order
        const long long f0 = s_pref[seq] + si.chunks_before(tile, walk);
        const int slot = me - cta_of(f0, T, Gc);
        p.ws_part[(((int64_t)seq * p.tiles_max + tile) * p.slots + slot) * kTile + tid] = v;
      }
      __syncthreads();
      acc = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    advance(cc);
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

}  // namespace

namespace sw {

static int ds_grid(int batch, int max_blocks) {
  const int a = (max_blocks - 1) / kTile;
  const long long work = (long long)batch * ((long long)a * (a + 1) / 2 + a + 1);   // >= chunks, >= duties
  return (int)std::min<long long>(work, 2LL * num_sms());
}

size_t decode_select_ws_bytes(int batch, int max_blocks) {
  const size_t tiles = (size_t)cdiv(max_blocks, kTile), mbp = tiles * kTile;
  return 256 + sizeof(float) * (size_t)batch * mbp + sizeof(float) * (size_t)batch * tiles * tiles * kTile;
}

int32_t launch_decode_select(const DecodeSelectArgs& a, cudaStream_t st) {
  if (a.batch == 0) return SW_OK;
  if (a.batch > kMaxBatch) return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: batch %d > %d", a.batch, kMaxBatch);
  if (cdiv(a.max_blocks, kTile) > kMaxTiles)
    return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: max_blocks %d too large", a.max_blocks);
  const size_t need = decode_select_ws_bytes(a.batch, a.max_blocks);
  if (a.ws == nullptr || a.ws_bytes < need)
    return fail(SW_ERR_WORKSPACE, "sw_decode_select: workspace %zu < %zu bytes", a.ws_bytes, need);
  Params p;
  p.q = a.q.ptr; p.q_stride_seq = a.q.stride_tok; p.q_stride_head = a.q.stride_head; p.h_q = a.q.heads;
  p.k = a.k.ptr; p.k_stride_seq = a.k.stride_tok; p.k_stride_head = a.k.stride_head; p.h_kv = a.k.heads;
  p.seqlens = a.seqlens; p.signs = a.signs; p.cols = a.cols; p.r = a.r; p.scale = a.scale;
  p.inv_sqrt_r = 1.0f / sqrtf((float)a.r);
  p.s = a.s; p.flags = a.flags; p.kbar = a.kbar; p.ks = a.ks; p.W = a.W_cache; p.w_stride_seq = a.stride_seq;
  p.r_prev = a.r_prev; p.r_out = a.r_out; p.tau = a.tau; p.tau_max = a.tau_max; p.idx = a.idx; p.count = a.count;
  p.batch = a.batch; p.B = a.block; p.max_blocks = a.max_blocks;
  p.tiles_max = cdiv(a.max_blocks, kTile); p.mbp = p.tiles_max * kTile; p.slots = p.tiles_max;
  uint8_t* w = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(a.ws) + 255) & ~(uintptr_t)255);
  p.ws_scores = reinterpret_cast<float*>(w);
  w += sizeof(float) * (size_t)a.batch * p.mbp;
  p.ws_part = reinterpret_cast<float*>(w);
  p.g_stream = ds_grid(a.batch, a.max_blocks);

  void (*kern)(const Params) = nullptr;
  const int d = a.q.d;
  if (a.q.dtype == SW_BF16 && d == 128) kern = decode_select_kernel<__nv_bfloat16, 128>;
  else if (a.q.dtype == SW_BF16 && d == 64) kern = decode_select_kernel<__nv_bfloat16, 64>;
  else if (a.q.dtype == SW_F32 && d == 128) kern = decode_select_kernel<float, 128>;
  else if (a.q.dtype == SW_F32 && d == 64) kern = decode_select_kernel<float, 64>;
  else return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: dtype %d / d %d", a.q.dtype, d);

  // cp.async stream of the cached W (and of r_prev) needs 16-byte aligned row pieces; otherwise plain loads
  p.use_async = a.r_prev != nullptr && aligned16(a.W_cache) && aligned16(a.r_prev) && (a.max_blocks & 3) == 0 &&
                (a.stride_seq & 3) == 0;

  const size_t smem = sizeof(float) * (2 * ((size_t)p.mbp + kChunkRows) + kRowGroups * kTile) + 128 +
                      (size_t)kStages * kChunkBytes;
  if (smem > 200 * 1024 || sizeof(float) * (size_t)p.mbp > 160 * 1024)
    return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: max_blocks %d too large", a.max_blocks);
  if (int32_t rc = allow_dynamic_smem(kern, smem, "sw_decode_select smem attribute")) return rc;
  count_launch();
  launch_pdl(kern, dim3(p.g_stream), dim3(kThreads), smem, st, p);
  if (int32_t rc = check_launch("sw_decode_select")) return rc;
  return launch_decode_tail(p, st);
}

}  // namespace sw
