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
#include <cooperative_groups.h>

#include "common.cuh"
#include "select.cuh"
#include "sketch_common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int kThreads = 256;
constexpr int kTile = 64;            // columns per tile
constexpr int kRowGroups = 16;       // row lanes of the vector-matrix product
constexpr int kUnroll = 8;           // independent 16-byte loads in flight per thread
constexpr int kMaxCluster = 16;

struct Params {
  const void* q;  int64_t q_stride_seq, q_stride_head;  int h_q;
  const void* k;  int64_t k_stride_seq, k_stride_head;  int h_kv;
  const int32_t* seqlens;
  const int8_t* signs;  const int32_t* cols;  int r;  float scale;  float inv_sqrt_r;
  int s;  uint32_t flags;
  float* kbar;  float* ks;
  const float* W;  int64_t w_stride_seq;
  const float* r_prev;  float* r_out;
  const int32_t* tau;  int tau_max;
  int32_t* idx;  int32_t* count;
  int B, max_blocks, slots;
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

  extern __shared__ __align__(16) uint8_t smem_raw[];
  const int mb4 = (p.max_blocks + 3) & ~3;                             // keeps the float4 rows aligned
  float* s_rprev = reinterpret_cast<float*>(smem_raw);                 // [max_blocks]
  float* s_rfull = s_rprev + mb4;                                      // [max_blocks] (used on rank 0)
  float* s_w = s_rfull + mb4;                                          // [slots][64]: S -> w -> r
  float* s_part = s_w + p.slots * kTile;                               // [kRowGroups][64]
  __shared__ float s_vec[D], s_qt[128], s_kt[128];
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

  // ---- Steps 2-3: head means, running key-block mean, sketches ----------------------------------
  if (tid < D) {
    const T* qp = reinterpret_cast<const T*>(p.q) + (int64_t)seq * p.q_stride_seq + tid;
    float sq = 0.f;
    for (int h = 0; h < p.h_q; ++h) sq += (float)qp[(int64_t)h * p.q_stride_head];
    s_vec[tid] = sq / (float)p.h_q;
  }
  __syncthreads();
  swsk::sketch_tail<D>(s_vec, p.signs, p.cols, p.r, p.scale, s_qt);     // q~_t
  __syncthreads();
  if (owns_bq) {
    if (tid < D) {
      const T* kp = reinterpret_cast<const T*>(p.k) + (int64_t)seq * p.k_stride_seq + tid;
      float sk = 0.f;
      for (int h = 0; h < p.h_kv; ++h) sk += (float)kp[(int64_t)h * p.k_stride_head];
      const float avg = sk / (float)p.h_kv;
      float* mp = p.kbar + ((int64_t)seq * mb + bq) * D + tid;
      const float m = (cnt_in_block == 0) ? avg : ((float)cnt_in_block * (*mp) + avg) / (float)(cnt_in_block + 1);
      *mp = m;
      s_vec[tid] = m;
    }
    __syncthreads();
    swsk::sketch_tail<D>(s_vec, p.signs, p.cols, p.r, p.scale, s_kt, p.ks + ((int64_t)seq * mb + bq) * p.r);
  }
  __syncthreads();

  // ---- Steps 3-4: the new row of scores for this CTA's columns ------------------------------------
  const float* ksb = p.ks + (int64_t)seq * mb * p.r;
  float lmax = -INFINITY;
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
  __syncthreads();
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

  // ---- Step 5: r_out[j] = sum_{m < b_q} r_prev[m] W[m][j] + r_prev[b_q] w[j] --------------------------
  float lamax = 0.f;
  if (p.r_prev != nullptr) {
    const float* rp = p.r_prev + (int64_t)seq * mb;
    for (int i = tid; i <= bq; i += kThreads) s_rprev[i] = __ldg(rp + i);
    __syncthreads();
    const float* Wm = p.W + (int64_t)seq * p.w_stride_seq;
    const int cq = tid & 15, rg = tid >> 4;
    const bool vec_ok = (mb & 3) == 0 && ((reinterpret_cast<uintptr_t>(Wm) & 15u) == 0);
    for (int pass = 0; pass < p.slots; ++pass) {
      const int tile = tile_of(pass);
      const int col0 = tile * kTile;
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
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
  } else {
    // r^{-1} = e_{b_q}: the product is row b_q of W', i.e. the new row itself
    for (int i = tid; i < p.slots * kTile; i += kThreads) lamax = fmaxf(lamax, fabsf(s_w[i]));
  }

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

  // ---- Step 6 on rank 0: S = TopK(r[0..b_q), tau - |forced|) U {b_q} (U {0}) ----------------------------
  if (rk == 0) {
    const int tt = max(0, min(__ldg(p.tau + seq), p.tau_max));
    swsel::RowJob J = swsel::make_job(hi, bq, true, p.flags & SW_FORCE_FIRST, tt);
    const float* row = s_rfull;
    swsel::select_row([row](int j) { return row[j]; }, J, p.idx + (int64_t)seq * p.tau_max, p.tau_max,
                      p.count + seq, scratch);
  }
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

  int C = pick_cluster(a.batch, a.max_blocks);
  for (;; C >>= 1) {
    p.slots = cdiv(cdiv(a.max_blocks, kTile), C);
    const size_t smem = sizeof(float) * ((size_t)2 * ((a.max_blocks + 3) & ~3) + (size_t)p.slots * kTile + kRowGroups * kTile);
    if (smem > 200 * 1024) return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: max_blocks %d too large", a.max_blocks);
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
    if (e == cudaSuccess) break;
    cudaGetLastError();
    if (C == 1) return fail(SW_ERR_CUDA, "sw_decode_select: %s", cudaGetErrorString(e));
  }
  return check_launch("sw_decode_select");
}

}  // namespace sw
