// sw_decode_select: Alg. 2 Steps 2-6 for one new token per sequence, fused into
// ONE kernel: running key-block mean + sketches (Steps 2-3), the new row of W (Steps 3-4), the
// row-vector walk r^k = r^{k-1} W'^k (Step 5), the max-abs rescale (P9) and the
// top-tau selection (Step 6).  HBM-bound on the cached W (4 b^2/2 bytes per sequence).
//
// The whole grid (two CTAs per SM) streams the cached W, whatever the batch: the work of the batch is
// cut into items -- one 64-row x 64-column chunk of the block-causal part of W each (rows [64 c, b_q) of
// column tile c), at least one item per column tile -- numbered over all sequences, and CTA i takes the
// contiguous range [i T / G, (i+1) T / G) of the T items.  A CTA accumulates r_prev[m] W[m][j] over its
// chunks of one column tile in registers and leaves one 64-float partial per (tile, CTA) in the workspace
// (fixed slots, fixed summation order: deterministic).  The first item of every column tile also carries the
// "score duty": q~_t (and, on the tile that holds b_q, the running key-block mean and its sketch) and the
// raw scores of its 64 columns.  Nothing waits on another CTA: every CTA counts the items it has finished
// per sequence with one atomic, and the CTA that completes a sequence runs that sequence's tail -- softmax
// statistics of the score row, W_new = A^s, r = sum of partials + r_prev[b_q] W_new, rescale, radix select
// (select.cuh) -- on a row of at most max_blocks floats in shared memory.  The counters live in the
// caller's workspace and are left at zero by every completed call.
// The cached W streams through a cp.async ring (5 x 16 KB per CTA), requested before the score duty runs;
// the new row of W is stored as row b_q of the cache (Alg. 2 Step 4).  DESIGN.md sec. 6.2 has the
// measurements behind these choices.
#include <algorithm>

#include "common.cuh"
#include "select.cuh"
#include "sketch_common.cuh"
#include "sm100.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kTile = 64;            // columns per tile
constexpr int kRowGroups = 16;       // row lanes of the vector-matrix product
constexpr int kChunkRows = 64;
constexpr int kStages = 5;
constexpr int kChunkBytes = kChunkRows * kTile * 4;
constexpr int kPieces = kChunkBytes / 16 / kThreads;     // 16-byte cp.async pieces per thread per chunk
constexpr int kMaxBatch = 1024;      // per-sequence item counts are scanned in shared memory

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
  unsigned int* ws_cnt;              // [batch] items finished per sequence (zero between calls)
  float* ws_scores;                  // [batch][mbp] raw scores of the new row
  float* ws_part;                    // [batch][tiles_max][slots][64] partial walk sums
  int mbp, tiles_max, slots;
};

// Item bookkeeping of one sequence.  b_q = 64 a + e; column tile c < a has rows [64 c, b_q): a - c + (e > 0)
// chunks; tile a (the one that holds b_q) has (e > 0) chunks and always one item.  Without a walk
// (r_prev = NULL) every tile is a single score-only item.
struct SeqInfo {
  int bq, a, eps;
  __device__ __forceinline__ int chunks(int tile, bool walk) const { return walk ? (tile < a ? a - tile + eps : eps) : 0; }
  __device__ __forceinline__ int items(int tile, bool walk) const { return max(1, chunks(tile, walk)); }
  __device__ __forceinline__ int items_before(int tile, bool walk) const {        // tile <= a
    return walk ? tile * a - tile * (tile - 1) / 2 + tile * eps : tile;
  }
  __device__ __forceinline__ int total(bool walk) const { return walk ? a * (a + 1) / 2 + a * eps + 1 : a + 1; }
};
__device__ __forceinline__ SeqInfo seq_info(const int32_t* seqlens, int seq, int B) {
  SeqInfo s;
  const int t = __ldg(seqlens + seq);
  s.bq = (t - 1) / B;                                  // block of the new token = b_curr
  s.a = s.bq / kTile;
  s.eps = (s.bq % kTile) != 0;
  return s;
}
// CTA that owns global item g when T items are dealt to G CTAs as [i T / G, (i+1) T / G)
__device__ __forceinline__ int cta_of(long long g, int T, int G) { return (int)(((g + 1) * G - 1) / T); }

__device__ __forceinline__ float block_max(float v, float* s_red) {
  v = swd::warp_max(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float m = s_red[0];
#pragma unroll
  for (int w = 1; w < kThreads / 32; ++w) m = fmaxf(m, s_red[w]);
  return m;
}
__device__ __forceinline__ float block_sum(float v, float* s_red) {
  v = swd::warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float m = 0.f;
#pragma unroll
  for (int w = 0; w < kThreads / 32; ++w) m += s_red[w];
  return m;
}

template <typename TIn, int D>
__global__ void __launch_bounds__(kThreads, 2)
decode_select_kernel(const Params p) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = (int)gridDim.x;
  const bool walk = p.r_prev != nullptr;
  const bool async = walk && p.use_async;
  const bool soft = p.flags & SW_SCORE_SOFTMAX;
  const int mb = p.max_blocks;

  extern __shared__ __align__(128) uint8_t smem_raw[];
  float* s_rprev = reinterpret_cast<float*>(smem_raw);                 // [mbp + 64] r_prev of the current sequence
  float* s_part = s_rprev + p.mbp + kChunkRows;                        // [kRowGroups][64]
  uint8_t* s_ring = reinterpret_cast<uint8_t*>(
      (reinterpret_cast<uintptr_t>(s_part + kRowGroups * kTile) + 127) & ~(uintptr_t)127);   // [kStages][16 KB]
  float* s_row = reinterpret_cast<float*>(s_ring);                     // [mbp] tail only (the ring is idle then)
  __shared__ __align__(16) float s_vec[D], s_qt[128], s_kt[128], s_sign[D];
  __shared__ float s_hx[kThreads / D][D];
  __shared__ int32_t s_cols[128];
  __shared__ float s_red[kThreads / 32];
  __shared__ int s_pref[kMaxBatch + 1];                                // exclusive prefix of items per sequence
  __shared__ int s_scan[kThreads / 32];
  __shared__ int s_last;                                               // this CTA has at least one tail to run
  __shared__ unsigned s_tailmask[kMaxBatch / 32];                      // sequences whose tail this CTA runs
  __shared__ swsel::Scratch scratch;

  // ---- item counts of all sequences: exclusive prefix in shared memory ------------------------------
  {
    constexpr int kPer = kMaxBatch / kThreads;
    int v[kPer], sum = 0;
#pragma unroll
    for (int e = 0; e < kPer; ++e) {
      const int sq = tid * kPer + e;
      v[e] = (sq < p.batch) ? seq_info(p.seqlens, sq, p.B).total(walk) : 0;
      sum += v[e];
    }
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += u;
    }
    if (lane == 31) s_scan[warp] = incl;
    if (tid < D) s_sign[tid] = p.signs ? (float)p.signs[tid] : 1.f;
    if (tid < kMaxBatch / 32) s_tailmask[tid] = 0u;
    if (tid == 0) s_last = 0;
    if (tid < p.r && tid < 128) s_cols[tid] = p.cols[tid];
    __syncthreads();
    int base = 0;
    for (int w = 0; w < warp; ++w) base += s_scan[w];
    int run = base + incl - sum;
#pragma unroll
    for (int e = 0; e < kPer; ++e) {
      const int sq = tid * kPer + e;
      if (sq <= p.batch) s_pref[sq] = run;
      run += v[e];
    }
    __syncthreads();
  }
  const int T = s_pref[p.batch];
  const int g_begin = (int)((long long)blockIdx.x * T / G), g_end = (int)((long long)(blockIdx.x + 1) * T / G);
  const int n_my = g_end - g_begin;
  if (n_my == 0) return;

  // ---- cursors over this CTA's items (thread-uniform) -------------------------------------------------
  struct Cursor { int seq, tile, chunk; SeqInfo si; };
  auto locate = [&](int g) {
    Cursor c;
    int lo = 0, hi = p.batch - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (s_pref[mid] <= g) lo = mid; else hi = mid - 1; }
    c.seq = lo;
    c.si = seq_info(p.seqlens, lo, p.B);
    const int local = g - s_pref[lo];
    int tl = 0, th = c.si.a;
    while (tl < th) { const int mid = (tl + th + 1) >> 1; if (c.si.items_before(mid, walk) <= local) tl = mid; else th = mid - 1; }
    c.tile = tl;
    c.chunk = local - c.si.items_before(tl, walk);
    return c;
  };
  auto advance = [&](Cursor& c) {
    if (++c.chunk >= c.si.items(c.tile, walk)) {
      c.chunk = 0;
      if (++c.tile > c.si.a) {
        c.tile = 0;
        if (++c.seq < p.batch) c.si = seq_info(p.seqlens, c.seq, p.B);
      }
    }
  };
  Cursor cc = locate(g_begin), pc = cc;

  // ---- W stream: chunk = rows [64 tile + 64 chunk, +64) x columns [64 tile, +64) of the sequence's cached W
  int p_left = n_my, issued = 0;
  auto issue_next = [&]() {                           // all threads: request the next chunk (or an empty group)
    while (p_left > 0 && pc.si.chunks(pc.tile, walk) == 0) { advance(pc); --p_left; }
    if (p_left > 0) {
      const float* Wseq = p.W + (int64_t)pc.seq * p.w_stride_seq;
      const int m0 = (pc.tile + pc.chunk) * kTile;
      const uint32_t dst = sm100::smem_u32(s_ring + (size_t)(issued % kStages) * kChunkBytes);
#pragma unroll
      for (int u = 0; u < kPieces; ++u) {
        const int pcs = u * kThreads + tid, rr = pcs >> 4, c4 = pc.tile * kTile + (pcs & 15) * 4;
        if (m0 + rr < pc.si.bq && c4 < mb)            // rows >= b_q / columns >= max_blocks are never read
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + pcs * 16),
                       "l"(Wseq + (int64_t)(m0 + rr) * mb + c4) : "memory");
      }
      ++issued; advance(pc); --p_left;
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  if (async)
    for (int i = 0; i < kStages - 1; ++i) issue_next();

  // head mean of x[seq] (all heads) -> s_vec (fp32), by all threads
  constexpr int kGroups = kThreads / D;
  auto head_mean = [&](const void* base, int64_t stride_seq, int64_t stride_head, int heads, int seq) {
    const int hx = tid % D, hg = tid / D;
    const TIn* xp = reinterpret_cast<const TIn*>(base) + (int64_t)seq * stride_seq + hx;
    constexpr int kRegs = 16;
    float v[kRegs];
#pragma unroll
    for (int u = 0; u < kRegs; ++u) {
      const int h = hg + u * kGroups;
      v[u] = (h < heads) ? (float)xp[(int64_t)h * stride_head] : 0.f;
    }
    float sm = 0.f;
#pragma unroll
    for (int u = 0; u < kRegs; ++u) sm += v[u];
    for (int h = hg + kRegs * kGroups; h < heads; h += kGroups) sm += (float)xp[(int64_t)h * stride_head];
    s_hx[hg][hx] = sm;
    __syncthreads();
    if (tid < D) {
      float a = 0.f;
#pragma unroll
      for (int g = 0; g < kGroups; ++g) a += s_hx[g][tid];
      s_vec[tid] = a / (float)heads;
    }
    __syncthreads();
  };

  const int q4 = p.r >> 2;                            // float4s per sketch row
  int cur_seq = -1, qt_seq = -1, done_in_seq = 0, consumed = 0;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  bool acc_live = false;
  const int cq = tid & 15, rg = tid >> 4;

  // tail of one sequence (this CTA finished its last item): Steps 4-6 on the whole row
  auto run_tail = [&](int seq) {
    const SeqInfo si = seq_info(p.seqlens, seq, p.B);
    const int bq = si.bq, hi = bq + 1;
    __threadfence();
    const float* sc = p.ws_scores + (int64_t)seq * p.mbp;
    float lmax = -INFINITY;
    for (int j = tid; j < hi; j += kThreads) { const float v = __ldcg(sc + j); s_row[j] = v; lmax = fmaxf(lmax, v); }
    float m = 0.f, inv_l = 1.f;
    if (soft) {
      m = block_max(lmax, s_red);
      float e = 0.f;
      for (int j = tid; j < hi; j += kThreads) e += expf(s_row[j] - m);
      inv_l = 1.f / block_sum(e, s_red);
    }
    // W_new = A^s; Alg. 2 Step 4 cache update: the new row becomes row b_q of the cached W,
    // zeros right of the diagonal.  Row b_q is never read while b_q is the current block.
    float* wrow = p.W + (int64_t)seq * p.w_stride_seq + (int64_t)bq * mb;
    const float rq = walk ? __ldg(p.r_prev + (int64_t)seq * mb + bq) : 1.f;
    const int base_g = s_pref[seq];
    float lamax = 0.f;
    for (int j = tid; j < mb; j += kThreads) {
      float w = 0.f, v = 0.f;
      if (j < hi) {
        const float sj = s_row[j];
        w = swd::powi(soft ? expf(sj - m) * inv_l : sj, p.s);
        // Step 5: r_out[j] = sum_{m < b_q} r_prev[m] W[m][j] + r_prev[b_q] w[j]; the partial sums in slot order
        const int tile = j / kTile, nch = si.chunks(tile, walk);
        if (nch > 0) {
          const long long f0 = base_g + si.items_before(tile, walk);
          const int i0 = cta_of(f0, T, G), i1 = cta_of(f0 + nch - 1, T, G);
          const float* pp = p.ws_part + (((int64_t)seq * p.tiles_max + tile) * p.slots) * kTile + (j & (kTile - 1));
          for (int sl = 0; sl <= i1 - i0; ++sl) v += __ldcg(pp + sl * kTile);
        }
        v = fmaf(rq, w, v);
        s_row[j] = v;
        lamax = fmaxf(lamax, fabsf(v));
      }
      wrow[j] = w;
    }
    const float amax = block_max(lamax, s_red);           // (its barriers also publish s_row)
    const bool rescale = (p.flags & SW_ROWNORM) && amax > 0.f;
    float* ro = p.r_out + (int64_t)seq * mb;
    for (int j = tid; j < mb; j += kThreads) {
      float v = 0.f;
      if (j < hi) { v = rescale ? s_row[j] / amax : s_row[j]; s_row[j] = v; }
      ro[j] = v;
    }
    __syncthreads();
    // Step 6: S = TopK(r[0..b_q), tau - |forced|) U {b_q} (U {0})
    const int tt = max(0, min(__ldg(p.tau + seq), p.tau_max));
    swsel::RowJob J = swsel::make_job(hi, bq, true, p.flags & SW_FORCE_FIRST, tt);
    const float* row = s_row;
    swsel::select_row([row](int j) { return row[j]; }, J, p.idx + (int64_t)seq * p.tau_max, p.tau_max,
                      p.count + seq, scratch);
    if (tid == 0) p.ws_cnt[seq] = 0;                      // leave the counter ready for the next call
    __syncthreads();
  };

  // this CTA has finished `done_in_seq` items of sequence `seq`: publish, and take the tail if it was the last
  auto finish_seq = [&](int seq) {
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      const unsigned total = (unsigned)(s_pref[seq + 1] - s_pref[seq]);
      const unsigned old = atomicAdd(p.ws_cnt + seq, (unsigned)done_in_seq);
      // the tail runs after this CTA's streaming work (its row buffer aliases the ring)
      if (old + (unsigned)done_in_seq == total) { s_tailmask[seq >> 5] |= 1u << (seq & 31); s_last = 1; }
    }
    done_in_seq = 0;
  };

  for (int it = 0; it < n_my; ++it) {
    const SeqInfo& si = cc.si;
    const int seq = cc.seq, tile = cc.tile, bq = si.bq;
    if (seq != cur_seq) {
      if (cur_seq >= 0) finish_seq(cur_seq);
      cur_seq = seq;
      __syncthreads();
      if (walk) {
        const float* rp = p.r_prev + (int64_t)seq * mb;
        for (int i = tid; i < p.mbp + kChunkRows; i += kThreads) s_rprev[i] = (i <= bq) ? __ldg(rp + i) : 0.f;
      }
    }
    if (cc.chunk == 0) {
      // ---- score duty of (seq, tile): Steps 2-4 for columns [64 tile, 64 tile + 64) ------------------------
      if (qt_seq != seq) {
        head_mean(p.q, p.q_stride_seq, p.q_stride_head, p.h_q, seq);
        swsk::sketch_tail<D>(s_vec, s_sign, s_cols, p.r, p.scale, s_qt);       // q~_t
        qt_seq = seq;
        __syncthreads();
      }
      if (tile == si.a) {
        // the tile that holds column b_q owns the key-side update of Step 2
        const int cnt = (__ldg(p.seqlens + seq) - 1) % p.B;                    // tokens already in block b_curr
        float kbar_old = 0.f;
        float* kb = p.kbar + ((int64_t)seq * mb + bq) * D;
        if (cnt != 0 && tid < D) kbar_old = kb[tid];
        head_mean(p.k, p.k_stride_seq, p.k_stride_head, p.h_kv, seq);
        if (tid < D) {
          const float avg = s_vec[tid];
          const float mn = (cnt == 0) ? avg : ((float)cnt * kbar_old + avg) / (float)(cnt + 1);
          kb[tid] = mn;
          s_vec[tid] = mn;
        }
        __syncthreads();
        swsk::sketch_tail<D>(s_vec, s_sign, s_cols, p.r, p.scale, s_kt, p.ks + ((int64_t)seq * mb + bq) * p.r);
        __syncthreads();
      }
      const float* ksb = p.ks + (int64_t)seq * mb * p.r;
      float* sc = p.ws_scores + (int64_t)seq * p.mbp;
      const int hi = bq + 1, col0 = tile * kTile;
      const bool vec_scores = (p.r & 3) == 0 && q4 <= 32 && (reinterpret_cast<uintptr_t>(ksb) & 15u) == 0;
      if (vec_scores) {
        // q4 adjacent lanes share one column; all loads of the tile are issued before the first use
        const int part = tid & (q4 - 1), per_pass = kThreads / q4;
        const float4 qv = *reinterpret_cast<const float4*>(s_qt + part * 4);
        constexpr int kU = 8;
        for (int c0 = 0; c0 < kTile; c0 += kU * per_pass) {
          float4 kv[kU];
#pragma unroll
          for (int u = 0; u < kU; ++u) {
            const int cj = c0 + u * per_pass + tid / q4, j = col0 + cj;
            kv[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (cj < kTile && j < hi) {
              const float* kp2 = (j == bq) ? s_kt : ksb + (int64_t)j * p.r;
              kv[u] = *reinterpret_cast<const float4*>(kp2 + part * 4);
            }
          }
#pragma unroll
          for (int u = 0; u < kU; ++u) {
            if (c0 + u * per_pass >= kTile) break;                              // warp-uniform
            const int cj = c0 + u * per_pass + tid / q4, j = col0 + cj;
            float a = fmaf(qv.w, kv[u].w, fmaf(qv.z, kv[u].z, fmaf(qv.y, kv[u].y, qv.x * kv[u].x)));
            for (int o = q4 >> 1; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
            if (part == 0 && cj < kTile && j < hi) sc[j] = a * p.inv_sqrt_r;
          }
        }
      } else {
        for (int cj = warp; cj < kTile; cj += kThreads / 32) {
          const int j = col0 + cj;
          if (j < hi) {
            const float* kp = (j == bq) ? s_kt : ksb + (int64_t)j * p.r;
            float a = 0.f;
            for (int c = lane; c < p.r; c += 32) a = fmaf(s_qt[c], kp[c], a);
            a = swd::warp_sum(a);
            if (lane == 0) sc[j] = a * p.inv_sqrt_r;
          }
        }
      }
    }
    const int nch = si.chunks(tile, walk);
    if (nch > 0) {
      // ---- Step 5, one chunk: acc[j] += sum_m r_prev[m] W[m][j] over rows [m0, m0 + 64) ---------------------
      const int m0 = (tile + cc.chunk) * kTile;
      const int rows = min(kChunkRows, bq - m0);
      if (async) {
        asm volatile("cp.async.wait_group %0;" ::"n"(kStages - 2) : "memory");   // chunk `consumed` has landed
        __syncthreads();                              // ... for every thread; the previous chunk is fully consumed
        issue_next();                                 // refill the stage the previous chunk occupied
        const float* box = reinterpret_cast<const float*>(s_ring + (size_t)(consumed % kStages) * kChunkBytes);
#pragma unroll
        for (int u = 0; u < kChunkRows / kRowGroups; ++u) {
          const int rr = rg + u * kRowGroups;
          if (rr < rows) {
            const float4 v = *reinterpret_cast<const float4*>(box + rr * kTile + cq * 4);
            const float a = s_rprev[m0 + rr];
            acc.x = fmaf(a, v.x, acc.x);
            acc.y = fmaf(a, v.y, acc.y);
            acc.z = fmaf(a, v.z, acc.z);
            acc.w = fmaf(a, v.w, acc.w);
          }
        }
        ++consumed;
      } else {
        __syncthreads();                              // s_rprev is complete
        const float* Wm = p.W + (int64_t)seq * p.w_stride_seq;
        const int c4 = tile * kTile + cq * 4;
        for (int rr = rg; rr < rows; rr += kRowGroups) {
          const float a = s_rprev[m0 + rr];
          const float* wr = Wm + (int64_t)(m0 + rr) * mb;
          if (c4 + 0 < mb) acc.x = fmaf(a, __ldg(wr + c4 + 0), acc.x);
          if (c4 + 1 < mb) acc.y = fmaf(a, __ldg(wr + c4 + 1), acc.y);
          if (c4 + 2 < mb) acc.z = fmaf(a, __ldg(wr + c4 + 2), acc.z);
          if (c4 + 3 < mb) acc.w = fmaf(a, __ldg(wr + c4 + 3), acc.w);
        }
      }
      acc_live = true;
    }
    ++done_in_seq;
    const bool tile_ends = (it == n_my - 1) || (cc.chunk + 1 >= si.items(tile, walk));
    if (tile_ends && acc_live) {
      // one partial per (tile, CTA): slot = rank of this CTA among the CTAs that share the tile
      *reinterpret_cast<float4*>(s_part + rg * kTile + cq * 4) = acc;
      __syncthreads();
      if (tid < kTile) {
        float v = 0.f;
#pragma unroll
        for (int g = 0; g < kRowGroups; ++g) v += s_part[g * kTile + tid];      // fixed order
        const long long f0 = s_pref[seq] + si.items_before(tile, walk);
        const int slot = (int)blockIdx.x - cta_of(f0, T, G);
        p.ws_part[(((int64_t)seq * p.tiles_max + tile) * p.slots + slot) * kTile + tid] = v;
      }
      __syncthreads();
      acc = make_float4(0.f, 0.f, 0.f, 0.f);
      acc_live = false;
    }
    advance(cc);
  }
  const int seq_first = locate(g_begin).seq;
  finish_seq(cur_seq);
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  if (s_last)
    for (int sq = seq_first; sq <= cur_seq; ++sq)
      if ((s_tailmask[sq >> 5] >> (sq & 31)) & 1u) run_tail(sq);
}

}  // namespace

namespace sw {

static int ds_grid(int batch, int max_blocks) {
  const int a = (max_blocks - 1) / kTile;
  const long long items = (long long)batch * ((long long)a * (a + 1) / 2 + a + 1);
  return (int)std::min<long long>(items, 2LL * num_sms());
}

size_t decode_select_ws_bytes(int batch, int max_blocks) {
  const size_t tiles = (size_t)cdiv(max_blocks, kTile), mbp = tiles * kTile;
  return 256 + (((size_t)batch * 4 + 255) & ~(size_t)255) + sizeof(float) * (size_t)batch * mbp +
         sizeof(float) * (size_t)batch * tiles * tiles * kTile;
}

int32_t launch_decode_select(const DecodeSelectArgs& a, cudaStream_t st) {
  if (a.batch == 0) return SW_OK;
  if (a.batch > kMaxBatch) return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: batch %d > %d", a.batch, kMaxBatch);
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
  p.ws_cnt = reinterpret_cast<unsigned int*>(w);
  w += ((size_t)a.batch * 4 + 255) & ~(size_t)255;
  p.ws_scores = reinterpret_cast<float*>(w);
  w += sizeof(float) * (size_t)a.batch * p.mbp;
  p.ws_part = reinterpret_cast<float*>(w);

  void (*kern)(const Params) = nullptr;
  const int d = a.q.d;
  if (a.q.dtype == SW_BF16 && d == 128) kern = decode_select_kernel<__nv_bfloat16, 128>;
  else if (a.q.dtype == SW_BF16 && d == 64) kern = decode_select_kernel<__nv_bfloat16, 64>;
  else if (a.q.dtype == SW_F32 && d == 128) kern = decode_select_kernel<float, 128>;
  else if (a.q.dtype == SW_F32 && d == 64) kern = decode_select_kernel<float, 64>;
  else return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: dtype %d / d %d", a.q.dtype, d);

  // cp.async stream of the cached W needs 16-byte aligned row pieces; otherwise the plain-load path runs
  p.use_async = a.r_prev != nullptr && aligned16(a.W_cache) && (a.max_blocks & 3) == 0 && (a.stride_seq & 3) == 0;

  const size_t ring = std::max((size_t)kStages * kChunkBytes, sizeof(float) * (size_t)p.mbp);
  const size_t smem = sizeof(float) * ((size_t)p.mbp + kChunkRows + kRowGroups * kTile) + 128 + ring;
  if (smem > 200 * 1024) return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: max_blocks %d too large", a.max_blocks);
  if (int32_t rc = allow_dynamic_smem(kern, smem, "sw_decode_select smem attribute")) return rc;
  count_launch();
  kern<<<ds_grid(a.batch, a.max_blocks), kThreads, smem, st>>>(p);
  return check_launch("sw_decode_select");
}

}  // namespace sw
