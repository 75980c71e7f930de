// sw_block_scores: Alg. 1 Steps 5-6a, eq. PAPER.md:69.
//   S = Q~ K~^T / sqrt(r); block-causal mask (P6); row softmax (P5); W = A^(.s) (P4).
// True fp32 (no TF32): the selection is sensitive to ~1e-5 relative score differences.
// A CTA owns kRows query rows of one sequence and sweeps the key blocks in tiles of kCols
// staged through shared memory; pass 1 writes raw S and keeps a running (max, sum) per row,
// pass 2 re-reads its own rows (L2-resident) and writes A and W.
#include "common.cuh"

namespace {

constexpr int kRows = 16;
constexpr int kCols = 64;
constexpr int kThreads = 256;
constexpr int kRMax = 128;           // r <= d <= 128

__global__ void __launch_bounds__(kThreads)
block_scores_kernel(const float* __restrict__ qs, const float* __restrict__ ks, int r, int s,
                    uint32_t flags, const int32_t* __restrict__ cu_blocks,
                    const int64_t* __restrict__ cu_sq, float* __restrict__ W, float* __restrict__ A,
                    float inv_sqrt_r) {
  extern __shared__ float smem[];
  float* s_q = smem;                              // [kRows][r]
  float* s_k = s_q + kRows * kRMax;               // [kCols][r+1]
  float* s_t = s_k + kCols * (kRMax + 1);         // [kRows][kCols+1]
  __shared__ float s_m[kRows], s_l[kRows];

  const int seq = blockIdx.y;                     // grid = (row tiles of the longest sequence, batch)
  const int row0 = blockIdx.x * kRows;
  const int blk0 = __ldg(cu_blocks + seq);
  const int b = __ldg(cu_blocks + seq + 1) - blk0;
  if (row0 >= b) return;
  float* Wm = W + __ldg(cu_sq + seq);
  float* Am = A ? A + __ldg(cu_sq + seq) : nullptr;
  const bool causal = flags & SW_CAUSAL;
  const bool soft = flags & SW_SCORE_SOFTMAX;
  const bool matpow = flags & SW_POW_MATRIX;
  const int nrows = min(kRows, b - row0);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int rp = r + 1;

  for (int i = tid; i < kRows * r; i += kThreads) {
    int rr = i / r, c = i - rr * r;
    s_q[rr * kRMax + c] = (rr < nrows) ? qs[(int64_t)(blk0 + row0 + rr) * r + c] : 0.f;
  }
  if (tid < kRows) { s_m[tid] = -INFINITY; s_l[tid] = 0.f; }
  __syncthreads();

  const int last_row = row0 + nrows - 1;
  const int col_end = causal ? min(b, last_row + 1) : b;     // columns that can be unmasked
  const int col = tid % kCols;                     // key column inside the tile
  const int rg = tid / kCols;                      // rows rg*4 .. rg*4+3

  for (int c0 = 0; c0 < col_end; c0 += kCols) {
    for (int i = tid; i < kCols * r; i += kThreads) {
      int kk = i / r, c = i - kk * r;
      s_k[kk * rp + c] = (c0 + kk < b) ? ks[(int64_t)(blk0 + c0 + kk) * r + c] : 0.f;
    }
    __syncthreads();
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    const float* kp = s_k + col * rp;
    const float* qp = s_q + (rg * 4) * kRMax;
    for (int c = 0; c < r; ++c) {
      float kv = kp[c];
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[e] = fmaf(qp[e * kRMax + c], kv, acc[e]);
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) s_t[(rg * 4 + e) * (kCols + 1) + col] = acc[e] * inv_sqrt_r;
    __syncthreads();
    // per-row running softmax statistics + coalesced store of the raw scores (2 rows per warp)
#pragma unroll
    for (int rr2 = 0; rr2 < 2; ++rr2) {
      const int rr = warp * 2 + rr2;
      const int gi = row0 + rr;
      if (rr < nrows) {
        float v0 = s_t[rr * (kCols + 1) + lane], v1 = s_t[rr * (kCols + 1) + lane + 32];
        const int j0 = c0 + lane, j1 = c0 + lane + 32;
        const bool ok0 = j0 < b && (!causal || j0 <= gi), ok1 = j1 < b && (!causal || j1 <= gi);
        if (j0 < b) Wm[(int64_t)gi * b + j0] = ok0 ? v0 : 0.f;
        if (j1 < b) Wm[(int64_t)gi * b + j1] = ok1 ? v1 : 0.f;
        if (soft) {
          float mx = swd::warp_max(fmaxf(ok0 ? v0 : -INFINITY, ok1 ? v1 : -INFINITY));
          float m_old = s_m[rr];
          float m_new = fmaxf(m_old, mx);
          float e = 0.f;
          if (ok0) e += expf(v0 - m_new);
          if (ok1) e += expf(v1 - m_new);
          e = swd::warp_sum(e);
          __syncwarp();
          if (lane == 0 && m_new > -INFINITY) {
            s_l[rr] = s_l[rr] * ((m_old == -INFINITY) ? 0.f : expf(m_old - m_new)) + e;
            s_m[rr] = m_new;
          }
          __syncwarp();
        }
      }
    }
    __syncthreads();
  }

  // pass 2: A = exp(S - m) / l (or raw S), W = A^s; masked / upper-triangular entries are 0
  for (int rr = warp; rr < nrows; rr += kThreads / 32) {
    const int gi = row0 + rr;
    const float m = s_m[rr], inv_l = soft ? 1.f / s_l[rr] : 1.f;
    float* wrow = Wm + (int64_t)gi * b;
    float* arow = Am ? Am + (int64_t)gi * b : nullptr;
    for (int j = lane; j < b; j += 32) {
      const bool ok = !causal || j <= gi;
      float a = 0.f;
      if (ok) {
        float v = wrow[j];
        a = soft ? expf(v - m) * inv_l : v;
      }
      if (arow) arow[j] = a;
      wrow[j] = ok ? (matpow ? a : swd::powi(a, s)) : 0.f;
    }
  }
}

// Decode row (Alg. 2 Steps 3-4): one CTA per sequence.
__global__ void __launch_bounds__(256)
block_scores_row_kernel(const float* __restrict__ q_tok, const float* __restrict__ ks,
                        const int32_t* __restrict__ seqlens, int B, int max_blocks, int r, int s,
                        uint32_t flags, float* __restrict__ w_row, float inv_sqrt_r) {
  __shared__ float s_q[kRMax];
  __shared__ float s_red[8];
  __shared__ float s_stat[2];
  const int seq = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int t = __ldg(seqlens + seq);
  const int bq = (t - 1) / B;
  const int nb = (t + B - 1) / B;                              // blocks in the cache
  const bool causal = flags & SW_CAUSAL, soft = flags & SW_SCORE_SOFTMAX;
  const int hi = causal ? bq + 1 : nb;
  for (int c = tid; c < r; c += 256) s_q[c] = q_tok[(int64_t)seq * r + c];
  __syncthreads();
  float* out = w_row + (int64_t)seq * max_blocks;
  const float* kb = ks + (int64_t)seq * max_blocks * r;
  float mx = -INFINITY;
  for (int j = tid; j < hi; j += 256) {
    const float* kp = kb + (int64_t)j * r;
    float acc = 0.f;
    for (int c = 0; c < r; ++c) acc = fmaf(s_q[c], kp[c], acc);
    acc *= inv_sqrt_r;
    out[j] = acc;
    mx = fmaxf(mx, acc);
  }
  float m = 0.f, inv_l = 1.f;
  if (soft) {
    mx = swd::warp_max(mx);
    if (lane == 0) s_red[warp] = mx;
    __syncthreads();
    if (tid == 0) { float v = s_red[0]; for (int w = 1; w < 8; ++w) v = fmaxf(v, s_red[w]); s_stat[0] = v; }
    __syncthreads();
    m = s_stat[0];
    float e = 0.f;
    for (int j = tid; j < hi; j += 256) e += expf(out[j] - m);
    e = swd::warp_sum(e);
    if (lane == 0) s_red[warp] = e;
    __syncthreads();
    if (tid == 0) { float v = 0.f; for (int w = 0; w < 8; ++w) v += s_red[w]; s_stat[1] = v; }
    __syncthreads();
    inv_l = 1.f / s_stat[1];
  }
  for (int j = tid; j < max_blocks; j += 256) {
    float w = 0.f;
    if (j < hi) {
      float a = soft ? expf(out[j] - m) * inv_l : out[j];
      w = swd::powi(a, s);
    }
    out[j] = w;
  }
}

}  // namespace

namespace sw {

static size_t scores_smem_bytes() {
  return sizeof(float) * (kRows * kRMax + kCols * (kRMax + 1) + kRows * (kCols + 1));
}

int32_t launch_block_scores(const sw_layout& L, const float* qs, const float* ks, int r, int s,
                            uint32_t flags, float* W, float* A, cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  static bool attr_set = false;
  const size_t smem = scores_smem_bytes();
  if (!attr_set) {
    cudaFuncSetAttribute(block_scores_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr_set = true;
  }
  dim3 grid(cdiv(L.max_blocks, kRows), L.batch);
  block_scores_kernel<<<grid, kThreads, smem, st>>>(qs, ks, r, s, flags, L.cu_blocks, L.cu_sq, W, A,
                                                    1.0f / sqrtf((float)r));
  return check_launch("sw_block_scores");
}

int32_t launch_block_scores_row(int batch, int block, int max_blocks, const float* q_tok, const float* ks,
                                const int32_t* seqlens, int r, int s, uint32_t flags, float* w_row,
                                cudaStream_t st) {
  if (batch == 0) return SW_OK;
  block_scores_row_kernel<<<batch, 256, 0, st>>>(q_tok, ks, seqlens, block, max_blocks, r, s, flags,
                                                 w_row, 1.0f / sqrtf((float)r));
  return check_launch("sw_block_scores_row");
}

}  // namespace sw
