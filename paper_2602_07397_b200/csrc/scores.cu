// sw_block_scores: Alg. 1 Steps 5-6a, eq. PAPER.md:69.
//   S = Q~ K~^T / sqrt(r); block-causal mask (P6); row softmax (P5); W = A^(.s) (P4).
// True fp32 (no TF32): the selection is sensitive to ~1e-5 relative score differences.
// Two launches: (1) score_tile_kernel - one CTA per (16 query rows x 64 key columns) tile on or below
// the block diagonal writes the raw masked scores S into W (b = 512: 144 CTAs instead of the 32
// row-sweeping CTAs of the first version, 56 -> ~8 us); (2) score_rows_kernel - one warp per row reads
// its row twice from L2 (max / sum-exp, then normalise) and writes A and W = A^s in place.
#include "common.cuh"

namespace {

constexpr int kRows = 16;
constexpr int kCols = 64;
constexpr int kThreads = 256;
constexpr int kRMax = 128;           // r <= d <= 128

__global__ void __launch_bounds__(kThreads)
score_tile_kernel(const float* __restrict__ qs, const float* __restrict__ ks, int r, uint32_t flags,
                  const int32_t* __restrict__ cu_blocks, const int64_t* __restrict__ cu_sq,
                  float* __restrict__ W, float inv_sqrt_r) {
  extern __shared__ float smem[];
  float* s_q = smem;                              // [kRows][r]
  float* s_k = s_q + kRows * kRMax;               // [kCols][r+1]
  float* s_t = s_k + kCols * (kRMax + 1);         // [kRows][kCols+1]

  const int seq = blockIdx.z;                     // grid = (column tiles, row tiles, batch)
  const int row0 = blockIdx.y * kRows, c0 = blockIdx.x * kCols;
  const int blk0 = __ldg(cu_blocks + seq);
  const int b = __ldg(cu_blocks + seq + 1) - blk0;
  const bool causal = flags & SW_CAUSAL;
  if (row0 >= b || c0 >= b) return;
  const int nrows = min(kRows, b - row0);
  if (causal && c0 > row0 + nrows - 1) return;    // tile entirely above the diagonal: score_rows zero-fills
  float* Wm = W + __ldg(cu_sq + seq);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int rp = r + 1;

  if ((r & 3) == 0) {                             // 128-bit loads of the sketch rows
    const int r4 = r >> 2;
    for (int i = tid; i < kRows * r4; i += kThreads) {
      const int rr = i / r4, c = (i - rr * r4) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (rr < nrows) v = *reinterpret_cast<const float4*>(qs + (int64_t)(blk0 + row0 + rr) * r + c);
      float* d = s_q + rr * kRMax + c;
      d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w;
    }
    for (int i = tid; i < kCols * r4; i += kThreads) {
      const int kk = i / r4, c = (i - kk * r4) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (c0 + kk < b) v = *reinterpret_cast<const float4*>(ks + (int64_t)(blk0 + c0 + kk) * r + c);
      float* d = s_k + kk * rp + c;
      d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w;
    }
  } else {
    for (int i = tid; i < kRows * r; i += kThreads) {
      const int rr = i / r, c = i - rr * r;
      s_q[rr * kRMax + c] = (rr < nrows) ? qs[(int64_t)(blk0 + row0 + rr) * r + c] : 0.f;
    }
    for (int i = tid; i < kCols * r; i += kThreads) {
      const int kk = i / r, c = i - kk * r;
      s_k[kk * rp + c] = (c0 + kk < b) ? ks[(int64_t)(blk0 + c0 + kk) * r + c] : 0.f;
    }
  }
  __syncthreads();

  const int col = tid % kCols;                     // key column inside the tile
  const int rg = tid / kCols;                      // rows rg*4 .. rg*4+3
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  const float* kp = s_k + col * rp;
  const float* qp = s_q + (rg * 4) * kRMax;
  for (int c = 0; c < r; ++c) {
    const float kv = kp[c];
#pragma unroll
    for (int e = 0; e < 4; ++e) acc[e] = fmaf(qp[e * kRMax + c], kv, acc[e]);
  }
#pragma unroll
  for (int e = 0; e < 4; ++e) s_t[(rg * 4 + e) * (kCols + 1) + col] = acc[e] * inv_sqrt_r;
  __syncthreads();
  // coalesced store of the raw masked scores (2 rows per warp)
#pragma unroll
  for (int rr2 = 0; rr2 < 2; ++rr2) {
    const int rr = warp * 2 + rr2, gi = row0 + rr;
    if (rr < nrows) {
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int j = c0 + lane + 32 * h;
        if (j < b) Wm[(int64_t)gi * b + j] = (!causal || j <= gi) ? s_t[rr * (kCols + 1) + lane + 32 * h] : 0.f;
      }
    }
  }
}

// One warp per row: A = softmax over the unmasked columns (or the raw scores), W = A^(.s) (or A in
// matrix mode); masked / upper-triangular entries are written as 0.
__global__ void __launch_bounds__(kThreads)
score_rows_kernel(int s, uint32_t flags, const int32_t* __restrict__ cu_blocks, const int64_t* __restrict__ cu_sq,
                  int batch, float* __restrict__ W, float* __restrict__ A) {
  const int lane = threadIdx.x & 31;
  const int gb = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
  if (gb >= __ldg(cu_blocks + batch)) return;
  const int seq = swd::find_seq(cu_blocks, batch, gb);
  const int blk0 = __ldg(cu_blocks + seq);
  const int b = __ldg(cu_blocks + seq + 1) - blk0;
  const int gi = gb - blk0;
  const bool causal = flags & SW_CAUSAL, soft = flags & SW_SCORE_SOFTMAX, matpow = flags & SW_POW_MATRIX;
  float* wrow = W + __ldg(cu_sq + seq) + (int64_t)gi * b;
  float* arow = A ? A + __ldg(cu_sq + seq) + (int64_t)gi * b : nullptr;
  const int hi = causal ? gi + 1 : b;             // unmasked columns [0, hi)
  float m = 0.f, inv_l = 1.f;
  if ((b & 3) == 0 && (reinterpret_cast<uintptr_t>(wrow) & 15u) == 0 &&
      (arow == nullptr || (reinterpret_cast<uintptr_t>(arow) & 15u) == 0)) {
    // 128-bit path: lane owns columns 4*(lane + 32 t) .. +3
    const int hi4 = (hi + 3) >> 2, b4 = b >> 2;
    if (soft) {
      float mx = -INFINITY;
#pragma unroll 8
      for (int q = lane; q < hi4; q += 32) {
        const float4 v = *reinterpret_cast<const float4*>(wrow + 4 * q);
        const int j = 4 * q;
        mx = fmaxf(mx, v.x);
        if (j + 1 < hi) mx = fmaxf(mx, v.y);
        if (j + 2 < hi) mx = fmaxf(mx, v.z);
        if (j + 3 < hi) mx = fmaxf(mx, v.w);
      }
      m = swd::warp_max(mx);
      float e = 0.f;
#pragma unroll 8
      for (int q = lane; q < hi4; q += 32) {
        const float4 v = *reinterpret_cast<const float4*>(wrow + 4 * q);
        const int j = 4 * q;
        e += expf(v.x - m);
        if (j + 1 < hi) e += expf(v.y - m);
        if (j + 2 < hi) e += expf(v.z - m);
        if (j + 3 < hi) e += expf(v.w - m);
      }
      inv_l = 1.f / swd::warp_sum(e);
    }
#pragma unroll 4
    for (int q = lane; q < b4; q += 32) {
      const int j = 4 * q;
      float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
      if (j < hi) {
        const float4 v = *reinterpret_cast<const float4*>(wrow + j);
        a.x = soft ? expf(v.x - m) * inv_l : v.x;
        if (j + 1 < hi) a.y = soft ? expf(v.y - m) * inv_l : v.y;
        if (j + 2 < hi) a.z = soft ? expf(v.z - m) * inv_l : v.z;
        if (j + 3 < hi) a.w = soft ? expf(v.w - m) * inv_l : v.w;
      }
      if (arow) *reinterpret_cast<float4*>(arow + j) = a;
      if (!matpow) { a.x = swd::powi(a.x, s); a.y = swd::powi(a.y, s); a.z = swd::powi(a.z, s); a.w = swd::powi(a.w, s); }
      *reinterpret_cast<float4*>(wrow + j) = a;      // powi(0, s) = 0 for s >= 1: masked entries stay 0
    }
    return;
  }
  if (soft) {
    float mx = -INFINITY;
    for (int j = lane; j < hi; j += 32) mx = fmaxf(mx, wrow[j]);
    m = swd::warp_max(mx);
    float e = 0.f;
    for (int j = lane; j < hi; j += 32) e += expf(wrow[j] - m);
    inv_l = 1.f / swd::warp_sum(e);
  }
  for (int j = lane; j < b; j += 32) {
    float a = 0.f;
    if (j < hi) {
      const float v = wrow[j];
      a = soft ? expf(v - m) * inv_l : v;
    }
    if (arow) arow[j] = a;
    wrow[j] = (j < hi) ? (matpow ? a : swd::powi(a, s)) : 0.f;
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
  const size_t smem = scores_smem_bytes();
  if (int32_t rc = allow_dynamic_smem(score_tile_kernel, smem, "sw_block_scores smem attribute")) return rc;
  dim3 grid(cdiv(L.max_blocks, kCols), cdiv(L.max_blocks, kRows), L.batch);
  count_launch(2);
  score_tile_kernel<<<grid, kThreads, smem, st>>>(qs, ks, r, flags, L.cu_blocks, L.cu_sq, W, 1.0f / sqrtf((float)r));
  score_rows_kernel<<<cdiv(L.total_blocks, kThreads / 32), kThreads, 0, st>>>(s, flags, L.cu_blocks, L.cu_sq, L.batch,
                                                                             W, A);
  return check_launch("sw_block_scores");
}

int32_t launch_block_scores_row(int batch, int block, int max_blocks, const float* q_tok, const float* ks,
                                const int32_t* seqlens, int r, int s, uint32_t flags, float* w_row,
                                cudaStream_t st) {
  if (batch == 0) return SW_OK;
  count_launch();
  block_scores_row_kernel<<<batch, 256, 0, st>>>(q_tok, ks, seqlens, block, max_blocks, r, s, flags,
                                                 w_row, 1.0f / sqrtf((float)r));
  return check_launch("sw_block_scores_row");
}

}  // namespace sw
