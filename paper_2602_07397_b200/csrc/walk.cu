// sw_walk_update: Sketch-Determined Walk, R^k = R^{k-1} W^k (Lemma A.11 PAPER.md:571-576,
// Alg. 1 Step 6 PAPER.md:783-787), followed by the per-row max-abs rescale (P9).
// fp32 SIMT GEMM (true fp32 FMA: selection parity needs ~1e-5 relative accuracy) that exploits
// the block-causal structure: R_prev and W are lower triangular, so output tile (ti, tj) is zero
// for tj > ti and its reduction runs over k-tiles tj..ti only (about 1/3 of the dense 2 b^3).
#include <atomic>

#include "common.cuh"

namespace {

constexpr int TM = 64, TN = 64, TK = 16, PAD = 4;
constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads)
walk_gemm_kernel(const float* __restrict__ Rp, const float* __restrict__ Wp, float* __restrict__ Op,
                 const int32_t* __restrict__ cu_blocks, const int64_t* __restrict__ cu_sq, int causal) {
  __shared__ __align__(16) float As[2][TK][TM + PAD];   // As[k][m]  (transposed on store)
  __shared__ __align__(16) float Bs[2][TK][TN + PAD];   // Bs[k][n]
  const int seq = blockIdx.z;
  const int b = __ldg(cu_blocks + seq + 1) - __ldg(cu_blocks + seq);
  const int ti = blockIdx.y, tj = blockIdx.x;
  const int row0 = ti * TM, col0 = tj * TN;
  if (row0 >= b || col0 >= b) return;
  const int64_t off = __ldg(cu_sq + seq);
  const float* A = Rp + off;
  const float* Bm = Wp + off;
  float* C = Op + off;
  const int tid = threadIdx.x, ty = tid / 16, tx = tid % 16;

  if (causal && tj > ti) {                    // strictly upper tile: zeros
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      int r = row0 + ty * 4 + e;
      if (r < b)
#pragma unroll
        for (int f = 0; f < 4; ++f) {
          int c = col0 + tx * 4 + f;
          if (c < b) C[(int64_t)r * b + c] = 0.f;
        }
    }
    return;
  }
  const int k_begin = causal ? col0 : 0;                    // W[m][j] = 0 for m < j
  const int k_end = causal ? min(b, row0 + TM) : b;         // R[i][m] = 0 for m > i
  const int nk = (k_end - k_begin + TK - 1) / TK;

  // global -> register staging: A tile 64x16 (4 consecutive k per thread), B tile 16x64
  const int a_row = tid / 4, a_k = (tid % 4) * 4;
  const int b_k = tid / 16, b_c = (tid % 16) * 4;
  float ra[4], rb[4];
  auto load_tiles = [&](int kt) {
    const int k0 = k_begin + kt * TK;
    const int gr = row0 + a_row;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      int gk = k0 + a_k + e;
      ra[e] = (gr < b && gk < k_end) ? __ldg(A + (int64_t)gr * b + gk) : 0.f;
    }
    const int gk = k0 + b_k;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      int gc = col0 + b_c + e;
      rb[e] = (gk < k_end && gc < b) ? __ldg(Bm + (int64_t)gk * b + gc) : 0.f;
    }
  };
  auto store_tiles = [&](int buf) {
#pragma unroll
    for (int e = 0; e < 4; ++e) As[buf][a_k + e][a_row] = ra[e];
    *reinterpret_cast<float4*>(&Bs[buf][b_k][b_c]) = make_float4(rb[0], rb[1], rb[2], rb[3]);
  };

  float acc[4][4];
#pragma unroll
  for (int e = 0; e < 4; ++e)
#pragma unroll
    for (int f = 0; f < 4; ++f) acc[e][f] = 0.f;

  load_tiles(0);
  store_tiles(0);
  __syncthreads();
  for (int kt = 0; kt < nk; ++kt) {
    const int buf = kt & 1;
    if (kt + 1 < nk) load_tiles(kt + 1);
#pragma unroll
    for (int k = 0; k < TK; ++k) {
      const float4 a = *reinterpret_cast<const float4*>(&As[buf][k][ty * 4]);
      const float4 bv = *reinterpret_cast<const float4*>(&Bs[buf][k][tx * 4]);
      const float av[4] = {a.x, a.y, a.z, a.w}, bw[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
      for (int e = 0; e < 4; ++e)
#pragma unroll
        for (int f = 0; f < 4; ++f) acc[e][f] = fmaf(av[e], bw[f], acc[e][f]);
    }
    if (kt + 1 < nk) store_tiles(buf ^ 1);
    __syncthreads();
  }
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    int r = row0 + ty * 4 + e;
    if (r < b)
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        int c = col0 + tx * 4 + f;
        if (c < b) C[(int64_t)r * b + c] = (causal && c > r) ? 0.f : acc[e][f];
      }
  }
}

// dst[i,:] = src[i,:] / max_j |src[i,j]|  (rownorm != 0), or a plain copy.  One CTA per row.
__global__ void __launch_bounds__(128)
row_rescale_kernel(const float* __restrict__ src, float* __restrict__ dst,
                   const int32_t* __restrict__ cu_blocks, const int64_t* __restrict__ cu_sq, int batch,
                   int rownorm) {
  __shared__ float s_red[4];
  const int gb = blockIdx.x;
  const int seq = swd::find_seq(cu_blocks, batch, gb);
  const int blk0 = __ldg(cu_blocks + seq);
  const int b = __ldg(cu_blocks + seq + 1) - blk0;
  const int i = gb - blk0;
  const int64_t off = __ldg(cu_sq + seq) + (int64_t)i * b;
  const float* s = src + off;
  float* d = dst + off;
  const int tid = threadIdx.x;
  float m = 0.f;
  if (rownorm) {
    for (int j = tid; j < b; j += 128) m = fmaxf(m, fabsf(s[j]));
    m = swd::warp_max(m);
    if ((tid & 31) == 0) s_red[tid >> 5] = m;
    __syncthreads();
    m = fmaxf(fmaxf(s_red[0], s_red[1]), fmaxf(s_red[2], s_red[3]));
    if (!(m > 0.f) && src == dst) return;      // all-zero row: untouched (P9)
  }
  if (rownorm && m > 0.f) {
    for (int j = tid; j < b; j += 128) d[j] = s[j] / m;
  } else if (src != dst) {
    for (int j = tid; j < b; j += 128) d[j] = s[j];
  }
}

// Decode: r_out = r_prev * W'  with W' = W_cache except row b_q = w_row (see sw.h).
// CTA = 32 columns x 8 row lanes; deterministic reduction order.
__global__ void __launch_bounds__(256)
walk_row_kernel(const float* __restrict__ r_prev, float* Wc, int64_t stride_seq,
                const float* __restrict__ w_row, const int32_t* __restrict__ seqlens, int B,
                int max_blocks, int causal, float* __restrict__ r_out) {
  __shared__ float s_part[8][33];
  const int seq = blockIdx.y;
  const int t = __ldg(seqlens + seq);
  const int bq = (t - 1) / B;
  const int nb = (t + B - 1) / B;
  const int lane = threadIdx.x & 31, rl = threadIdx.x >> 5;
  const int j = blockIdx.x * 32 + lane;
  const int j_hi = causal ? bq + 1 : nb;
  float* W = Wc + (int64_t)seq * stride_seq;
  const float* wr = w_row + (int64_t)seq * max_blocks;
  float* out = r_out + (int64_t)seq * max_blocks;
  if (blockIdx.x * 32 >= max_blocks) return;
  float acc = 0.f;
  if (j < j_hi) {
    if (r_prev == nullptr) {                               // r^{-1} = e_{b_q}
      if (rl == 0) acc = wr[j];
    } else {
      const float* rp = r_prev + (int64_t)seq * max_blocks;
      const int m_lo = causal ? (blockIdx.x * 32) : 0;     // W[m][j] = 0 for m < j
      for (int m = m_lo + rl; m < bq; m += 8) acc = fmaf(__ldg(rp + m), __ldg(W + (int64_t)m * max_blocks + j), acc);
      if (rl == 0) acc = fmaf(__ldg(rp + bq), wr[j], acc);
    }
  }
  s_part[rl][lane] = acc;
  __syncthreads();
  if (rl == 0 && j < max_blocks) {
    float v = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) v += s_part[k][lane];
    out[j] = (j < j_hi) ? v : 0.f;
    // Alg. 2 Step 4 cache update: the new row becomes row b_q of the cached W (rows < b_q were the only
    // ones read above, by any CTA)
    W[(int64_t)bq * max_blocks + j] = (j < j_hi) ? wr[j] : 0.f;
  }
}

__global__ void __launch_bounds__(256)
vec_rescale_kernel(float* __restrict__ r, int max_blocks) {
  __shared__ float s_red[8];
  float* v = r + (int64_t)blockIdx.x * max_blocks;
  float m = 0.f;
  for (int j = threadIdx.x; j < max_blocks; j += 256) m = fmaxf(m, fabsf(v[j]));
  m = swd::warp_max(m);
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = m;
  __syncthreads();
  m = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) m = fmaxf(m, s_red[k]);
  if (m > 0.f)
    for (int j = threadIdx.x; j < max_blocks; j += 256) v[j] = v[j] / m;
}

}  // namespace

namespace sw {

static std::atomic<int32_t> g_walk_kernel{SW_WALK_AUTO};      // process-wide test / benchmark switch
static thread_local int32_t g_walk_used = 0;
constexpr int kWalkTcMinBlocks = 512;      // SW_WALK_AUTO: tensor-core path from this max_blocks on

int32_t set_walk_kernel(int32_t which) { return g_walk_kernel.exchange(which); }
int32_t walk_kernel_used() { return g_walk_used; }
void note_walk_kernel(int32_t which) { g_walk_used = which; }

// SW_WALK_SIMT / SW_WALK_TCGEN05 for this problem and workspace (images_bytes = bytes available for the operand
// images), or a negative status when SW_WALK_TCGEN05 was forced and does not fit.
int32_t choose_walk_kernel(const sw_layout& L, size_t images_bytes) {
  const int32_t want = g_walk_kernel.load();
  const size_t tc_bytes = walk_tc_ws_bytes(L);
  const bool fits = tc_bytes > 0 && images_bytes >= tc_bytes;
  if (want == SW_WALK_TCGEN05 && !fits)
    return fail(tc_bytes == 0 ? SW_ERR_UNSUPPORTED : SW_ERR_WORKSPACE,
                "sw_walk_update: SW_WALK_TCGEN05 needs max_blocks >= 256 and %zu bytes of workspace for the operand images",
                tc_bytes);
  if (want == SW_WALK_SIMT || !fits) return SW_WALK_SIMT;
  return (want == SW_WALK_TCGEN05 || L.max_blocks >= kWalkTcMinBlocks) ? SW_WALK_TCGEN05 : SW_WALK_SIMT;
}

int32_t launch_walk_simt(const sw_layout& L, const float* R_prev, const float* W, float* dst, int causal,
                         cudaStream_t st) {
  dim3 grid(cdiv(L.max_blocks, TN), cdiv(L.max_blocks, TM), L.batch);
  count_launch();
  walk_gemm_kernel<<<grid, kThreads, 0, st>>>(R_prev, W, dst, L.cu_blocks, L.cu_sq, causal);
  return check_launch("sw_walk_update");
}

int32_t launch_copy_rows(const sw_layout& L, const float* src, float* dst, cudaStream_t st) {
  count_launch();
  row_rescale_kernel<<<L.total_blocks, 128, 0, st>>>(src, dst, L.cu_blocks, L.cu_sq, L.batch, 0);
  return check_launch("sw_walk_update");
}

int32_t launch_row_rescale(const sw_layout& L, float* R, cudaStream_t st) {
  count_launch();
  row_rescale_kernel<<<L.total_blocks, 128, 0, st>>>(R, R, L.cu_blocks, L.cu_sq, L.batch, 1);
  return check_launch("sw_walk_update");
}

int32_t launch_walk(const sw_layout& L, const float* R_prev, const float* W, int s, uint32_t flags,
                    float* R_out, void* ws, size_t ws_bytes, cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  const int causal = (flags & SW_CAUSAL) ? 1 : 0;
  const int nprod = (flags & SW_POW_MATRIX) ? s : 1;
  // workspace = [ping-pong matrix (batch * max_blocks^2 floats) | hi/lo images of the tcgen05 path]
  const size_t pp_bytes = walk_pp_bytes(L);
  const bool have_ws = ws != nullptr && (reinterpret_cast<uintptr_t>(ws) & 127u) == 0 && ws_bytes > pp_bytes;
  const int32_t which = choose_walk_kernel(L, have_ws ? ws_bytes - pp_bytes : 0);
  if (which < 0) return which;
  const bool use_tc = which == SW_WALK_TCGEN05;
  WalkImages im = {};
  if (use_tc) im = walk_images(L, reinterpret_cast<uint8_t*>(ws) + pp_bytes);
  g_walk_used = which;
  const float* cur = R_prev;
  bool w_split = false;
  for (int k = 1; k <= nprod; ++k) {
    // the last product must land in R_out; alternate with the workspace before that
    float* dst = ((nprod - k) % 2 == 0) ? R_out : reinterpret_cast<float*>(ws);
    int32_t rc;
    if (cur == nullptr) {                   // identity * W = W
      rc = launch_copy_rows(L, W, dst, st);
    } else if (use_tc) {
      rc = launch_split_tf32(L, cur, w_split ? nullptr : W, im, causal, st);
      if (rc == SW_OK) rc = launch_walk_tc(L, im, dst, causal, /*zero_upper=*/true, st);
      w_split = true;
    } else {
      rc = launch_walk_simt(L, cur, W, dst, causal, st);
    }
    if (rc != SW_OK) return rc;
    cur = dst;
  }
  if (flags & SW_ROWNORM) return launch_row_rescale(L, R_out, st);
  return SW_OK;
}

int32_t launch_walk_row(int batch, int block, int max_blocks, const float* r_prev, float* W_cache,
                        int64_t stride_seq, const float* w_row, const int32_t* seqlens, uint32_t flags,
                        float* r_out, cudaStream_t st) {
  if (batch == 0) return SW_OK;
  dim3 grid(cdiv(max_blocks, 32), batch);
  count_launch((flags & SW_ROWNORM) ? 2 : 1);
  walk_row_kernel<<<grid, 256, 0, st>>>(r_prev, W_cache, stride_seq, w_row, seqlens, block, max_blocks,
                                        (flags & SW_CAUSAL) ? 1 : 0, r_out);
  if (flags & SW_ROWNORM) vec_rescale_kernel<<<batch, 256, 0, st>>>(r_out, max_blocks);
  return check_launch("sw_walk_update_row");
}

}  // namespace sw
