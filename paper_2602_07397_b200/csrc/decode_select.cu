// sw_decode_select: Alg. 2 Steps 2-6 for one new token per sequence, fused into
// ONE kernel: running key-block mean + sketches (Steps 2-3), the new row of W (Steps 3-4), the
// row-vector walk r^k = r^{k-1} W'^k (Step 5), the max-abs rescale (P9) and the
// top-tau selection (Step 6).  HBM-bound on the cached W (4 b^2/2 bytes per sequence).
//
// One thread-block cluster per sequence.  The key-block columns are cut into 64-column tiles dealt
// to the CTAs of the cluster boustrophedon-wise (tile p*C + rank on even passes, p*C + C-1-rank on
// odd ones) so that the triangular W traffic is balanced; a CTA computes the scores, the walk and
// the rescaled r for its own columns only.  Row-global quantities cross the cluster through
// distributed shared memory: (max, sum-exp) of the score row, the max-abs of r, and finally the r
// values themselves, which every CTA pushes into rank 0's shared memory where the radix select
// (select.cuh) runs.  Three cluster barriers in total.
// The cached W streams through a cp.async ring (5 x 16 KB per CTA, two CTAs per SM), its first chunks
// and the key-sketch rows of the score row are requested before anything else; the new row of W is
// stored as row b_q of the cache (Alg. 2 Step 4).  DESIGN.md sec. 6.2 has the measurements behind
// these choices.
#include <cooperative_groups.h>

#include <algorithm>

#include "common.cuh"

// Phase stamps for tuning (compiled in only with -DSW_PHASE_PROF; the product build has none).
#ifdef SW_PHASE_PROF
__device__ unsigned long long g_sw_prof[4096 * 16];
extern "C" __attribute__((visibility("default"))) void* sw_debug_prof_ptr() {
  void* p = nullptr;
  cudaGetSymbolAddress(&p, g_sw_prof);
  return p;
}
#define SW_STAMP(k)                                                                 \
  do {                                                                              \
    if (threadIdx.x == 0) {                                                         \
      unsigned long long t_;                                                        \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                        \
      g_sw_prof[(blockIdx.x & 4095) * 16 + (k)] = t_;                               \
    }                                                                               \
  } while (0)
#else
#define SW_STAMP(k) do { } while (0)
#endif

#include "select.cuh"
#include "sketch_common.cuh"
#include "sm100.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int kThreads = 256;
constexpr int kTile = 64;            // columns per tile
constexpr int kRowGroups = 16;       // row lanes of the vector-matrix product
constexpr int kUnroll = 8;           // independent 16-byte loads in flight per thread
constexpr int kMaxCluster = 16;
// W stream: cp.async ring of kStages chunks of 64 rows x 64 columns fp32 (16 KB).  Measured on B200
// (one CTA per SM streaming HBM): cp.async 16 KB x 8 stages 6.8 TB/s, 8 KB x 8 5.5 TB/s; a TMA ring
// (cp.async.bulk[.tensor] + mbarrier) pays ~0.27 us per box whatever its size, so it needs >= 32 KB
// boxes, and the 128-bit register loads used before held only 32 KB per SM in flight (1.7 TB/s).
// 5 stages keep the CTA under ~105 KB of shared memory so that two CTAs fit on an SM: one GPC of the
// B200 has fewer than 16 free SMs, and with one CTA per SM only 7 clusters of 16 were co-resident.
constexpr int kChunkRows = 64;
constexpr int kStages = 5;
constexpr int kChunkBytes = kChunkRows * kTile * 4;
constexpr int kPieces = kChunkBytes / 16 / kThreads;     // 16-byte cp.async pieces per thread per chunk

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
  int B, max_blocks, slots;
  int use_async;                     // W streamed by cp.async (needs 16-byte aligned rows), else plain loads
};

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

template <typename T, int D>
__global__ void __launch_bounds__(kThreads)
decode_select_kernel(const Params p) {
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks();
  const int rk = (int)cluster.block_rank();
  const int seq = blockIdx.x / C;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  extern __shared__ __align__(128) uint8_t smem_raw[];
  const int mbp = ((p.max_blocks + kTile - 1) / kTile) * kTile + kChunkRows;   // zero-padded r_prev
  float* s_rprev = reinterpret_cast<float*>(smem_raw);                 // [mbp]
  float* s_w = s_rprev + mbp;                                          // [slots][64]: S -> w -> r
  float* s_part = s_w + p.slots * kTile;                               // [kRowGroups][64]
  uint8_t* s_ring = reinterpret_cast<uint8_t*>(
      (reinterpret_cast<uintptr_t>(s_part + kRowGroups * kTile) + 127) & ~(uintptr_t)127);   // [kStages][16 KB]
  float* s_rfull = reinterpret_cast<float*>(s_ring);                   // [max_blocks] on rank 0, after the walk
  __shared__ __align__(16) float s_vec[D], s_veck[D], s_qt[128], s_kt[128], s_sign[D];
  __shared__ float s_hq[kThreads / D][D], s_hk[kThreads / D][D];
  __shared__ int32_t s_cols[128];
  __shared__ float s_red[kThreads / 32];
  __shared__ float s_stat[2], s_amax[1];
  __shared__ swsel::Scratch scratch;

  const int t = __ldg(p.seqlens + seq);
  const int bq = (t - 1) / p.B;                      // block of the new token = b_curr
  const int nb = (t + p.B - 1) / p.B;
  const int cnt_in_block = (t - 1) % p.B;            // tokens already in block b_curr
  const bool causal = p.flags & SW_CAUSAL, soft = p.flags & SW_SCORE_SOFTMAX;
  const int hi = causal ? bq + 1 : nb;               // columns that can be unmasked
  const int n_tiles = (hi + kTile - 1) / kTile;
  const int mb = p.max_blocks;
  auto tile_of = [&](int pass) { return pass * C + ((pass & 1) ? C - 1 - rk : rk); };
  // the CTA that owns column b_q also owns the key-side update of Step 2
  const int bq_tile = bq / kTile, bq_pass = bq_tile / C;
  const bool owns_bq = tile_of(bq_pass) == bq_tile;

  // ---- operand loads of Steps 2-3, issued before anything waits: head values of q and k (heads dealt
  // to kGroups thread groups), the old running mean, the SRHT signs and columns
  constexpr int kGroups = kThreads / D, kHeadRegs = 16;
  const int hx = tid % D, hx_g = tid / D;
  const T* qp = reinterpret_cast<const T*>(p.q) + (int64_t)seq * p.q_stride_seq + hx;
  const T* kp = reinterpret_cast<const T*>(p.k) + (int64_t)seq * p.k_stride_seq + hx;
  float qreg[kHeadRegs], kreg[kHeadRegs];
#pragma unroll
  for (int u = 0; u < kHeadRegs; ++u) {
    const int h = hx_g + u * kGroups;
    qreg[u] = (h < p.h_q) ? (float)qp[(int64_t)h * p.q_stride_head] : 0.f;
    kreg[u] = (owns_bq && h < p.h_kv) ? (float)kp[(int64_t)h * p.k_stride_head] : 0.f;
  }
  float kbar_old = 0.f;
  if (owns_bq && cnt_in_block != 0 && tid >= 128 && tid < 128 + D)
    kbar_old = p.kbar[((int64_t)seq * mb + bq) * D + (tid - 128)];
  if (tid < D) s_sign[tid] = p.signs ? (float)p.signs[tid] : 1.f;
  if (tid < p.r && tid < 128) s_cols[tid] = p.cols[tid];

  // first batch of key-sketch rows of Steps 3-4 (up to 8 x 16 bytes per thread): requested here, ahead of
  // the W stream in the memory queues; column b_q is patched from shared memory at use
  const float* ksb = p.ks + (int64_t)seq * mb * p.r;
  const int q4 = p.r >> 2;                            // float4s per sketch row
  const bool vec_scores = (p.r & 3) == 0 && q4 <= 32 && (reinterpret_cast<uintptr_t>(ksb) & 15u) == 0;
  constexpr int kU = 8;
  float4 kv0[kU];
  if (vec_scores) {
    const int per_pass = kTile * q4, total = p.slots * per_pass;
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const int i = u * kThreads + tid;
      const int pass = i / per_pass, tile = tile_of(pass);
      const int j = tile * kTile + (i - pass * per_pass) / q4;
      kv0[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (i < total && tile < n_tiles && j < hi && j != bq)
        kv0[u] = *reinterpret_cast<const float4*>(ksb + (int64_t)j * p.r + (tid & (q4 - 1)) * 4);
    }
  }

  // ---- W stream (Step 5 operand): rows [m_lo, b_q) of this CTA's column tiles, 64-row TMA boxes.
  // Nothing in it depends on this step's q/k, so the first kStages - 1 chunks are requested up front
  // and land while Steps 2-4 run.
  const bool walk = p.r_prev != nullptr;
  const bool async = walk && p.use_async;
  auto chunks_of = [&](int pass) {
    const int tile = tile_of(pass);
    const int m_lo = causal ? tile * kTile : 0;
    return (tile < n_tiles && bq > m_lo) ? (bq - m_lo + kChunkRows - 1) / kChunkRows : 0;
  };
  const float* Wseq = p.W + (int64_t)seq * p.w_stride_seq;
  int pr_pass = 0, pr_chunk = 0, pr_issued = 0;       // producer cursor (same in every thread)
  auto issue_next = [&]() {                           // all threads: request the next chunk (or an empty group)
    while (pr_pass < p.slots && pr_chunk >= chunks_of(pr_pass)) { ++pr_pass; pr_chunk = 0; }
    if (pr_pass < p.slots) {
      const int tile = tile_of(pr_pass);
      const int m0 = (causal ? tile * kTile : 0) + pr_chunk * kChunkRows;
      const uint32_t dst = sm100::smem_u32(s_ring + (size_t)(pr_issued % kStages) * kChunkBytes);
#pragma unroll
      for (int u = 0; u < kPieces; ++u) {
        const int pc = u * kThreads + tid, rr = pc >> 4, c4 = tile * kTile + (pc & 15) * 4;
        if (m0 + rr < bq && c4 < mb)                  // rows >= b_q / columns >= max_blocks are never read
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + pc * 16),
                       "l"(Wseq + (int64_t)(m0 + rr) * mb + c4) : "memory");
      }
      ++pr_issued; ++pr_chunk;
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  if (async)
    for (int i = 0; i < kStages - 1; ++i) issue_next();

  SW_STAMP(0);
  // ---- Steps 2-3: head means, running key-block mean, sketches ----------------------------------
  // (the q / k / signs / cols loads were issued before the W prologue: one memory latency for all)
  {
    float sq = 0.f, sk = 0.f;
#pragma unroll
    for (int u = 0; u < kHeadRegs; ++u) { sq += qreg[u]; sk += kreg[u]; }
    for (int h = hx_g + kHeadRegs * kGroups; h < p.h_q; h += kGroups) sq += (float)qp[(int64_t)h * p.q_stride_head];
    if (owns_bq)
      for (int h = hx_g + kHeadRegs * kGroups; h < p.h_kv; h += kGroups) sk += (float)kp[(int64_t)h * p.k_stride_head];
    s_hq[hx_g][hx] = sq;
    s_hk[hx_g][hx] = sk;
  }
  __syncthreads();
  if (tid < D) {
    float sq = 0.f;
#pragma unroll
    for (int g = 0; g < kGroups; ++g) sq += s_hq[g][tid];
    s_vec[tid] = sq / (float)p.h_q;
  } else if (owns_bq && tid >= 128 && tid < 128 + D) {
    const int x = tid - 128;
    float sk = 0.f;
#pragma unroll
    for (int g = 0; g < kGroups; ++g) sk += s_hk[g][x];
    const float avg = sk / (float)p.h_kv;
    const float m = (cnt_in_block == 0) ? avg : ((float)cnt_in_block * kbar_old + avg) / (float)(cnt_in_block + 1);
    p.kbar[((int64_t)seq * mb + bq) * D + x] = m;
    s_veck[x] = m;
  }
  __syncthreads();
  swsk::sketch_tail<D>(s_vec, s_sign, s_cols, p.r, p.scale, s_qt);      // q~_t
  if (owns_bq)
    swsk::sketch_tail<D>(s_veck, s_sign, s_cols, p.r, p.scale, s_kt, p.ks + ((int64_t)seq * mb + bq) * p.r, 4);
  __syncthreads();

  SW_STAMP(1);
  // ---- Steps 3-4: the new row of scores for this CTA's columns ------------------------------------
  float lmax = -INFINITY;
  if (vec_scores) {
    // q4 adjacent lanes share one column: all of a tile's sketch rows are requested before the first
    // use (one memory latency per pass), partial dots meet in a fixed xor butterfly
    const int per_pass = kTile * q4, total = p.slots * per_pass;
    const int part = tid & (q4 - 1);
    const float4 qv = *reinterpret_cast<const float4*>(s_qt + part * 4);
    for (int i0 = 0; i0 < total; i0 += kU * kThreads) {
      float4 kv[kU];
      bool ok[kU];
#pragma unroll
      for (int u = 0; u < kU; ++u) {
        const int i = i0 + u * kThreads + tid;
        const int pass = i / per_pass, tile = tile_of(pass);
        const int j = tile * kTile + (i - pass * per_pass) / q4;
        ok[u] = i < total && tile < n_tiles && j < hi;
        kv[u] = (i0 == 0) ? kv0[u] : make_float4(0.f, 0.f, 0.f, 0.f);
        if (ok[u] && (i0 != 0 || j == bq)) {
          const float* kp2 = (j == bq) ? s_kt : ksb + (int64_t)j * p.r;
          kv[u] = *reinterpret_cast<const float4*>(kp2 + part * 4);
        }
      }
#pragma unroll
      for (int u = 0; u < kU; ++u) {
        const int i = i0 + u * kThreads + tid;
        if (i0 + u * kThreads >= total) break;                          // warp-uniform
        float acc = fmaf(qv.w, kv[u].w, fmaf(qv.z, kv[u].z, fmaf(qv.y, kv[u].y, qv.x * kv[u].x)));
        for (int o = q4 >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        const float sc = ok[u] ? acc * p.inv_sqrt_r : -INFINITY;
        if (part == 0 && i < total) s_w[i / q4] = sc;                   // = s_w[pass * kTile + column]
        lmax = fmaxf(lmax, sc);
      }
    }
  } else {
    for (int pass = 0; pass < p.slots; ++pass) {
      const int tile = tile_of(pass);
      for (int cj = warp; cj < kTile; cj += kThreads / 32) {
        const int j = tile * kTile + cj;
        float sc = -INFINITY;
        if (tile < n_tiles && j < hi) {
          const float* kp = (j == bq) ? s_kt : ksb + (int64_t)j * p.r;
          float acc = 0.f;
          for (int c = lane; c < p.r; c += 32) acc = fmaf(s_qt[c], kp[c], acc);
          sc = swd::warp_sum(acc) * p.inv_sqrt_r;
        }
        if (lane == 0) s_w[pass * kTile + cj] = sc;
        lmax = fmaxf(lmax, sc);
      }
    }
  }
  __syncthreads();
  SW_STAMP(2);
  if (soft) {
    const float m_i = block_max(lmax, s_red);
    float e = 0.f;
    for (int i = tid; i < p.slots * kTile; i += kThreads) {
      const float sc = s_w[i];
      if (sc > -INFINITY) e += expf(sc - m_i);
    }
    const float l_i = block_sum(e, s_red);
    if (tid == 0) { s_stat[0] = m_i; s_stat[1] = l_i; }
    cluster.sync();
    float m_r = -INFINITY, l_r = 0.f;
    if (tid < C) {
      const float* rs = cluster.map_shared_rank(s_stat, tid);
      m_r = rs[0]; l_r = rs[1];
    }
    const float m = block_max(m_r, s_red);
    const float l = block_sum((m_r > -INFINITY) ? l_r * expf(m_r - m) : 0.f, s_red);
    const float inv_l = 1.f / l;
    for (int i = tid; i < p.slots * kTile; i += kThreads) {
      const float sc = s_w[i];
      s_w[i] = (sc > -INFINITY) ? swd::powi(expf(sc - m) * inv_l, p.s) : 0.f;
    }
  } else {
    cluster.sync();                                   // keep the barrier count uniform
    for (int i = tid; i < p.slots * kTile; i += kThreads) {
      const float sc = s_w[i];
      s_w[i] = (sc > -INFINITY) ? swd::powi(sc, p.s) : 0.f;
    }
  }
  __syncthreads();
  // Alg. 2 Step 4 cache update: the new row becomes row b_q of the cached W, zeros right
  // of the diagonal.  Row b_q is never read while b_q is the current block (the walk reads rows < b_q).
  {
    float* wrow = p.W + (int64_t)seq * p.w_stride_seq + (int64_t)bq * mb;
    for (int i = tid; i < p.slots * kTile; i += kThreads) {
      const int pass = i / kTile;
      const int j = tile_of(pass) * kTile + (i - pass * kTile);
      if (j < mb) wrow[j] = s_w[i];                    // masked columns hold 0 already
    }
  }

  SW_STAMP(3);
  // ---- Step 5: r_out[j] = sum_{m < b_q} r_prev[m] W[m][j] + r_prev[b_q] w[j] --------------------------
  float lamax = 0.f;
  if (p.r_prev != nullptr) {
    const float* rp = p.r_prev + (int64_t)seq * mb;
    for (int i = tid; i < mbp; i += kThreads) s_rprev[i] = (i <= bq) ? __ldg(rp + i) : 0.f;
    __syncthreads();
    const float* Wm = p.W + (int64_t)seq * p.w_stride_seq;
    const int cq = tid & 15, rg = tid >> 4;
    const bool vec_ok = (mb & 3) == 0 && ((reinterpret_cast<uintptr_t>(Wm) & 15u) == 0);
    int cons = 0;                                     // chunks consumed so far (cp.async path)
    for (int pass = 0; pass < p.slots; ++pass) {
      const int tile = tile_of(pass);
      const int col0 = tile * kTile;
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      if (async) {
        const int m_lo = causal ? col0 : 0;
        const int nch = chunks_of(pass);
        for (int ch = 0; ch < nch; ++ch, ++cons) {
          asm volatile("cp.async.wait_group %0;" ::"n"(kStages - 2) : "memory");   // chunk `cons` has landed
          __syncthreads();                            // ... for every thread; chunk cons-1 is fully consumed
          issue_next();                               // refill the stage chunk cons-1 occupied
          const int m0 = m_lo + ch * kChunkRows;
          const int rows = min(kChunkRows, bq - m0);  // rows >= b_q are not part of the product
          const float* box = reinterpret_cast<const float*>(s_ring + (size_t)(cons % kStages) * kChunkBytes);
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
        }
      } else
      if (tile < n_tiles) {
        const int m_lo = causal ? col0 : 0;           // W[m][j] = 0 for m < j
        const int c4 = col0 + cq * 4;
        if (vec_ok && col0 + kTile <= mb) {
          int m = m_lo + rg;
          for (; m + (kUnroll - 1) * kRowGroups < bq; m += kUnroll * kRowGroups) {
            uint4 v[kUnroll];
#pragma unroll
            for (int u = 0; u < kUnroll; ++u)
              v[u] = swd::ld_nc_v4(Wm + (int64_t)(m + u * kRowGroups) * mb + c4);
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
              const float a = s_rprev[m + u * kRowGroups];
              acc.x = fmaf(a, __uint_as_float(v[u].x), acc.x);
              acc.y = fmaf(a, __uint_as_float(v[u].y), acc.y);
              acc.z = fmaf(a, __uint_as_float(v[u].z), acc.z);
              acc.w = fmaf(a, __uint_as_float(v[u].w), acc.w);
            }
          }
          for (; m < bq; m += kRowGroups) {
            const uint4 v = swd::ld_nc_v4(Wm + (int64_t)m * mb + c4);
            const float a = s_rprev[m];
            acc.x = fmaf(a, __uint_as_float(v.x), acc.x);
            acc.y = fmaf(a, __uint_as_float(v.y), acc.y);
            acc.z = fmaf(a, __uint_as_float(v.z), acc.z);
            acc.w = fmaf(a, __uint_as_float(v.w), acc.w);
          }
        } else {
          for (int m = m_lo + rg; m < bq; m += kRowGroups) {
            const float a = s_rprev[m];
            const float* wr = Wm + (int64_t)m * mb;
            if (c4 + 0 < mb) acc.x = fmaf(a, __ldg(wr + c4 + 0), acc.x);
            if (c4 + 1 < mb) acc.y = fmaf(a, __ldg(wr + c4 + 1), acc.y);
            if (c4 + 2 < mb) acc.z = fmaf(a, __ldg(wr + c4 + 2), acc.z);
            if (c4 + 3 < mb) acc.w = fmaf(a, __ldg(wr + c4 + 3), acc.w);
          }
        }
      }
      *reinterpret_cast<float4*>(s_part + rg * kTile + cq * 4) = acc;
      __syncthreads();
      if (tid < kTile) {
        float v = 0.f;
#pragma unroll
        for (int g = 0; g < kRowGroups; ++g) v += s_part[g * kTile + tid];      // fixed order
        const int j = col0 + tid;
        v = (tile < n_tiles && j < hi) ? fmaf(s_rprev[bq], s_w[pass * kTile + tid], v) : 0.f;
        s_w[pass * kTile + tid] = v;
        lamax = fmaxf(lamax, fabsf(v));
      }
      __syncthreads();
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
  } else {
    // r^{-1} = e_{b_q}: the product is row b_q of W', i.e. the new row itself
    for (int i = tid; i < p.slots * kTile; i += kThreads) lamax = fmaxf(lamax, fabsf(s_w[i]));
  }

  SW_STAMP(4);
  // ---- P9 rescale, write r_out, gather the row on rank 0 ---------------------------------------------
  const float amax_i = block_max(lamax, s_red);
  if (tid == 0) s_amax[0] = amax_i;
  cluster.sync();
  float a_r = 0.f;
  if (tid < C) a_r = *cluster.map_shared_rank(s_amax, tid);
  const float amax = block_max(a_r, s_red);
  const bool rescale = (p.flags & SW_ROWNORM) && amax > 0.f;
  float* ro = p.r_out + (int64_t)seq * mb;
  float* rfull0 = cluster.map_shared_rank(s_rfull, 0);
  for (int i = tid; i < p.slots * kTile; i += kThreads) {
    const int pass = i / kTile;
    const int tile = tile_of(pass);
    const int j = tile * kTile + (i - pass * kTile);
    if (tile < n_tiles && j < mb) {
      const float v = rescale ? s_w[i] / amax : s_w[i];
      ro[j] = v;
      if (j < hi) rfull0[j] = v;
    }
  }
  for (int j = n_tiles * kTile + rk * kThreads + tid; j < mb; j += C * kThreads) ro[j] = 0.f;
  cluster.sync();
  SW_STAMP(5);

  // ---- Step 6 on rank 0: S = TopK(r[0..b_q), tau - |forced|) U {b_q} (U {0}) ----------------------------
  if (rk == 0) {
    const int tt = max(0, min(__ldg(p.tau + seq), p.tau_max));
    swsel::RowJob J = swsel::make_job(hi, bq, true, p.flags & SW_FORCE_FIRST, tt);
    const float* row = s_rfull;
    swsel::select_row([row](int j) { return row[j]; }, J, p.idx + (int64_t)seq * p.tau_max, p.tau_max,
                      p.count + seq, scratch);
  }
  SW_STAMP(6);
}

}  // namespace

namespace sw {

static int pick_cluster(int batch, int max_blocks) {
  const int tiles = cdiv(max_blocks, kTile);
  int c = kMaxCluster;
  while (c > 1 && (c > tiles || (int64_t)batch * c > 2 * num_sms())) c >>= 1;
  return c;
}

int32_t launch_decode_select(const DecodeSelectArgs& a, cudaStream_t st) {
  if (a.batch == 0) return SW_OK;
  Params p;
  p.q = a.q.ptr; p.q_stride_seq = a.q.stride_tok; p.q_stride_head = a.q.stride_head; p.h_q = a.q.heads;
  p.k = a.k.ptr; p.k_stride_seq = a.k.stride_tok; p.k_stride_head = a.k.stride_head; p.h_kv = a.k.heads;
  p.seqlens = a.seqlens; p.signs = a.signs; p.cols = a.cols; p.r = a.r; p.scale = a.scale;
  p.inv_sqrt_r = 1.0f / sqrtf((float)a.r);
  p.s = a.s; p.flags = a.flags; p.kbar = a.kbar; p.ks = a.ks; p.W = a.W_cache; p.w_stride_seq = a.stride_seq;
  p.r_prev = a.r_prev; p.r_out = a.r_out; p.tau = a.tau; p.tau_max = a.tau_max; p.idx = a.idx; p.count = a.count;
  p.B = a.block; p.max_blocks = a.max_blocks;

  void (*kern)(const Params) = nullptr;
  const int d = a.q.d;
  if (a.q.dtype == SW_BF16 && d == 128) kern = decode_select_kernel<__nv_bfloat16, 128>;
  else if (a.q.dtype == SW_BF16 && d == 64) kern = decode_select_kernel<__nv_bfloat16, 64>;
  else if (a.q.dtype == SW_F32 && d == 128) kern = decode_select_kernel<float, 128>;
  else if (a.q.dtype == SW_F32 && d == 64) kern = decode_select_kernel<float, 64>;
  else return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: dtype %d / d %d", a.q.dtype, d);

  // cp.async stream of the cached W needs 16-byte aligned row pieces; otherwise the plain-load path runs
  p.use_async = a.r_prev != nullptr && a.W_cache != nullptr && aligned16(a.W_cache) && (a.max_blocks & 3) == 0 &&
                (a.stride_seq & 3) == 0;

  int C = pick_cluster(a.batch, a.max_blocks);
  for (;; C >>= 1) {
    p.slots = cdiv(cdiv(a.max_blocks, kTile), C);
    const size_t mbp = (size_t)cdiv(a.max_blocks, kTile) * kTile + kChunkRows;
    const size_t ring = std::max(p.use_async ? (size_t)kStages * kChunkBytes : 0, sizeof(float) * (size_t)((a.max_blocks + 3) & ~3));
    const size_t smem = sizeof(float) * (mbp + (size_t)p.slots * kTile + kRowGroups * kTile) + 128 + ring;
    if (smem > 220 * 1024) return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: max_blocks %d too large", a.max_blocks);
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (C > 8) cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(a.batch * C);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, p);
    if (e == cudaSuccess) { count_launch(); break; }
    cudaGetLastError();
    if (C == 1) return fail(SW_ERR_CUDA, "sw_decode_select: %s", cudaGetErrorString(e));
  }
  return check_launch("sw_decode_select");
}

}  // namespace sw
