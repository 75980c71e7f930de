// sw_block_scores: Alg. 1 Steps 5-6a, eq. PAPER.md:69.
//   S = Q~ K~^T / sqrt(r); block-causal mask (P6); row softmax (P5); W = A^(.s) (P4).
// fp32-class accuracy throughout (the selection is sensitive to ~1e-5 relative score differences): the default
// kernel runs the tile products on mma.sync TF32 with the 3xTF32 hi / lo split (error ~2^-21 relative, not TF32's
// 2^-11), the fallback uses plain fp32 FMA.
// Default, ONE launch: score_fused_kernel (r a power of two >= 4, strip fits in shared memory) -- one CTA per strip
// of 8 query rows keeps the strip's raw scores on chip while the key sketches stream through a cp.async ring, then
// turns each row into A, W = A^s and (for the tensor-core walk) the hi / lo operand images.
// Fallback, two launches: (1) score_tile_kernel - one CTA per (16 query rows x 64 key columns) tile on or below the
// block diagonal writes the raw masked scores S into W; (2) score_rows_kernel - one warp per row reads its row
// twice from L2 (max / sum-exp, then normalise) and writes A and W = A^s in place.
#include "common.cuh"
#include "walk_images.cuh"

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

// ---------------------------------------------------------------------------------------------------
// Fused form: scores, row softmax, power and -- for the tensor-core walk -- the hi / lo
// TF32 operand images of W in ONE launch, with the images of R_prev written by extra CTAs of the same grid.
// One CTA per strip of kFRows = 8 query rows: the strip's raw scores stay in shared memory ([8][b] floats)
// while the key sketches stream through a cp.async double buffer in 64-column tiles (float4 shared-memory reads,
// row stride r + 4 floats: conflict free), then warp w turns row w into A, W = A^s and the image rows.  W is
// written once and never re-read by this step; split_tf32_kernel and its pass over W and R are gone.
constexpr int kFRows = 8;
constexpr int kFCols = 64;
constexpr int kFStagesMax = 8;        // ring of key-sketch tiles (cp.async): 8, 4 or 2 stages, the deepest that fits

// D (16x8, fp32) += A (16x8, tf32, rows g / g + 8) * B (8x8, tf32); the A rows g + 8 are zero here
__device__ __forceinline__ void mma_tf32(float (&c)[4], uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(0u), "r"(a2), "r"(0u), "r"(b0), "r"(b1));
}

struct FusedParams {
  const float *qs, *ks;
  int r, s;
  uint32_t flags;
  const int32_t* cu_blocks;
  const int64_t* cu_sq;
  float *W, *A, *W2;                 // packed outputs (A, W2 may be NULL; W2 = a second copy of W: R^0 = W^0)
  float *whi, *wlo;                  // operand images of W, or NULL
  const float* R_prev;               // packed; split into rhi / rlo by the CTAs behind the strips, or NULL
  float *rhi, *rlo;
  int pitch, n_strips, lds;          // lds: row stride of the score strip in shared memory (floats)
  int stages;                        // 2, 4 or 8
  float inv_sqrt_r;
};

template <int kMaxKs>                  // k-steps of 8 the A fragments are sized for: r <= 8 kMaxKs
__global__ void __launch_bounds__(kThreads, kMaxKs <= 8 ? 2 : 1)
score_fused_kernel(const FusedParams p) {
  extern __shared__ __align__(16) float smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int seq = blockIdx.z;
  const int blk0 = __ldg(p.cu_blocks + seq);
  const int b = __ldg(p.cu_blocks + seq + 1) - blk0;
  const bool causal = p.flags & SW_CAUSAL, soft = p.flags & SW_SCORE_SOFTMAX, matpow = p.flags & SW_POW_MATRIX;
  const bool images = p.whi != nullptr;
  const int rows_all = images ? swimg::pad_rows(b) : b;       // image rows include the zero padding
  const int rbase = images ? swimg::row_base(p.cu_blocks, seq) : 0;

  if ((int)blockIdx.x >= p.n_strips) {
    // ---- operand images of R_prev: one warp per row, 4 float4 loads in flight per lane ---------------------------
    const int i = ((int)blockIdx.x - p.n_strips) * kFRows + warp;
    if (i < rows_all)
      swimg::split_row(p.R_prev + __ldg(p.cu_sq + seq) + (int64_t)i * b, i, b, p.pitch, causal,
                       p.rhi + (int64_t)(rbase + i) * p.pitch, p.rlo + (int64_t)(rbase + i) * p.pitch, lane, 32);
    return;
  }
  const int i0 = blockIdx.x * kFRows;
  if (i0 >= rows_all) return;
  const int r = p.r, r4 = r >> 2, ldk = r + 4, r4_log2 = 31 - __clz(r4);
  float* s_q = smem;                                          // [kFRows][r]
  const int nst = p.stages;
  float* s_k = s_q + kFRows * r;                              // [stages][kFCols][r + 4]
  float* s_S = s_k + nst * kFCols * ldk;                        // [kFRows][lds]
  const int nrows = max(0, min(kFRows, b - i0));

  if (nrows > 0) {
    const int hi_col = causal ? min(b, i0 + kFRows) : b;      // columns some row of the strip can see
    const int nct = (hi_col + kFCols - 1) / kFCols;
    auto load_k = [&](int ct) {                               // tile ct -> ring slot ct % kFStages (or an empty group)
      if (ct < nct) {
        float* dst = s_k + (ct & (nst - 1)) * kFCols * ldk;
        for (int i = tid; i < kFCols * r4; i += kThreads) {
          const int kk = i >> r4_log2, c = (i & (r4 - 1)) * 4;   // (r is a power of two for the SRHT; checked on the host)
          const int j = ct * kFCols + kk;
          const float* src = p.ks + (int64_t)(blk0 + min(j, b - 1)) * r + c;
          const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst + kk * ldk + c);
          const int sz = (j < b) ? 16 : 0;                    // rows past the sequence: zero fill
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
        }
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    };
    auto wait_tile = [&]() {                                  // all but the newest stages - 2 groups have landed
      if (nst == 8) asm volatile("cp.async.wait_group 6;" ::: "memory");
      else if (nst == 4) asm volatile("cp.async.wait_group 2;" ::: "memory");
      else asm volatile("cp.async.wait_group 0;" ::: "memory");
    };
    // stages - 1 tiles in flight
    for (int ct = 0; ct < nst - 1; ++ct) load_k(ct);
    for (int i = tid; i < kFRows * r4; i += kThreads) {
      const int rr = i / r4, c = (i - rr * r4) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (rr < nrows) v = *reinterpret_cast<const float4*>(p.qs + (int64_t)(blk0 + i0 + rr) * r + c);
      *reinterpret_cast<float4*>(s_q + rr * r + c) = v;
    }
    if ((r & 7) == 0) {
      // Tile product on the warp-level tensor cores with 3xTF32 error compensation (as the walk GEMM: x = hi + lo,
      // q k ~= q_lo k_hi + q_hi k_lo + q_hi k_hi, fp32 accumulate; dropped term 2^-22): mma.sync m16n8k8, the 8
      // strip rows in the upper half of M (the lower half is zero), one 8-column n-tile per warp and 64-column
      // tile.  With plain FMAs the strip was bound by shared-memory reads (3 x LDS.128 per 8 FMA): 73 of the
      // 135 us of the b = 2048 selection chain.
      __syncthreads();                                        // s_q is complete
      const int g = lane >> 2, t4 = lane & 3;
      uint32_t ahi[kMaxKs][2], alo[kMaxKs][2];                // A fragments (rows g; rows g + 8 are the zero padding)
#pragma unroll
      for (int ks = 0; ks < kMaxKs; ++ks) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const float x = (8 * ks < r) ? s_q[g * r + 8 * ks + t4 + 4 * h] : 0.f;
          const uint32_t hi = __float_as_uint(x) & 0xffffe000u;
          ahi[ks][h] = hi;
          alo[ks][h] = __float_as_uint(x - __uint_as_float(hi));
        }
      }
      const int n0 = warp * 8;                                // this warp's columns of every tile
      for (int ct = 0; ct < nct; ++ct) {
        wait_tile();
        __syncthreads();                                      // tile ct landed; tile ct - 1 fully consumed
        load_k(ct + nst - 1);
        const float* kp = s_k + (ct & (nst - 1)) * kFCols * ldk + (n0 + g) * ldk + t4;
        float c[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int ks = 0; ks < kMaxKs; ++ks) {
          if (8 * ks < r) {                                   // (warp-uniform)
            const float k0 = kp[8 * ks], k1 = kp[8 * ks + 4];
            const uint32_t b0h = __float_as_uint(k0) & 0xffffe000u, b1h = __float_as_uint(k1) & 0xffffe000u;
            const uint32_t b0l = __float_as_uint(k0 - __uint_as_float(b0h)), b1l = __float_as_uint(k1 - __uint_as_float(b1h));
            mma_tf32(c, alo[ks][0], alo[ks][1], b0h, b1h);    // small terms first
            mma_tf32(c, ahi[ks][0], ahi[ks][1], b0l, b1l);
            mma_tf32(c, ahi[ks][0], ahi[ks][1], b0h, b1h);
          }
        }
        *reinterpret_cast<float2*>(s_S + g * p.lds + ct * kFCols + n0 + 2 * t4) =
            make_float2(c[0] * p.inv_sqrt_r, c[1] * p.inv_sqrt_r);
      }
    } else {
    const int col = tid & (kFCols - 1), rg = tid / kFCols;    // rows 2 rg, 2 rg + 1 of the strip
    for (int ct = 0; ct < nct; ++ct) {
      wait_tile();
      __syncthreads();                                        // tile ct landed; tile ct - 1 fully consumed
      load_k(ct + nst - 1);
      const float* kp = s_k + (ct & (nst - 1)) * kFCols * ldk + col * ldk;
      const float* q0 = s_q + (2 * rg) * r;
      const float* q1 = q0 + r;
      float a0 = 0.f, a1 = 0.f;
      for (int c = 0; c < r; c += 4) {
        const float4 kv = *reinterpret_cast<const float4*>(kp + c);
        const float4 x0 = *reinterpret_cast<const float4*>(q0 + c);
        const float4 x1 = *reinterpret_cast<const float4*>(q1 + c);
        a0 = fmaf(x0.x, kv.x, a0); a0 = fmaf(x0.y, kv.y, a0); a0 = fmaf(x0.z, kv.z, a0); a0 = fmaf(x0.w, kv.w, a0);
        a1 = fmaf(x1.x, kv.x, a1); a1 = fmaf(x1.y, kv.y, a1); a1 = fmaf(x1.z, kv.z, a1); a1 = fmaf(x1.w, kv.w, a1);
      }
      s_S[(2 * rg) * p.lds + ct * kFCols + col] = a0 * p.inv_sqrt_r;
      s_S[(2 * rg + 1) * p.lds + ct * kFCols + col] = a1 * p.inv_sqrt_r;
    }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
  }

  // ---- row phase: warp w owns row i0 + w -------------------------------------------------------------------
  const int i = i0 + warp;
  if (i >= rows_all) return;
  float* ihi = images ? p.whi + (int64_t)(rbase + i) * p.pitch : nullptr;
  float* ilo = images ? p.wlo + (int64_t)(rbase + i) * p.pitch : nullptr;
  const int icols = images ? swimg::row_cols(i, p.pitch, causal) : 0;
  if (i >= b) {                                               // padding row of the images
    for (int j = lane * 4; j < icols; j += 128) {
      *reinterpret_cast<float4*>(ihi + j) = make_float4(0.f, 0.f, 0.f, 0.f);
      *reinterpret_cast<float4*>(ilo + j) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    return;
  }
  const float* srow = s_S + warp * p.lds;
  const int hi = causal ? i + 1 : b;                          // unmasked columns [0, hi)
  float m = 0.f, inv_l = 1.f;
  if (soft) {
    float mx = -INFINITY;
    for (int j = lane; j < hi; j += 32) mx = fmaxf(mx, srow[j]);
    m = swd::warp_max(mx);
    float e = 0.f;
    for (int j = lane; j < hi; j += 32) e += expf(srow[j] - m);
    inv_l = 1.f / swd::warp_sum(e);
  }
  const int64_t off = __ldg(p.cu_sq + seq) + (int64_t)i * b;
  float* wrow = p.W + off;
  float* arow = p.A ? p.A + off : nullptr;
  float* w2row = p.W2 ? p.W2 + off : nullptr;
  const bool vec = (b & 3) == 0 && (reinterpret_cast<uintptr_t>(wrow) & 15u) == 0 &&
                   (arow == nullptr || (reinterpret_cast<uintptr_t>(arow) & 15u) == 0) &&
                   (w2row == nullptr || (reinterpret_cast<uintptr_t>(w2row) & 15u) == 0);
  const int jend = max((b + 3) & ~3, icols);
  for (int j = lane * 4; j < jend; j += 128) {
    float a[4], w[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      a[e] = 0.f;
      if (j + e < hi) a[e] = soft ? expf(srow[j + e] - m) * inv_l : srow[j + e];
      w[e] = matpow ? a[e] : swd::powi(a[e], p.s);            // powi(0, s) = 0 for s >= 1: masked entries stay 0
    }
    if (j < b) {
      if (vec) {
        if (arow) *reinterpret_cast<float4*>(arow + j) = make_float4(a[0], a[1], a[2], a[3]);
        *reinterpret_cast<float4*>(wrow + j) = make_float4(w[0], w[1], w[2], w[3]);
        if (w2row) *reinterpret_cast<float4*>(w2row + j) = make_float4(w[0], w[1], w[2], w[3]);
      } else {
#pragma unroll
        for (int e = 0; e < 4; ++e)
          if (j + e < b) { if (arow) arow[j + e] = a[e]; wrow[j + e] = w[e]; if (w2row) w2row[j + e] = w[e]; }
      }
    }
    if (j < icols) {
      float4 h, l;
      swimg::split4(make_float4(w[0], w[1], w[2], w[3]), h, l);
      *reinterpret_cast<float4*>(ihi + j) = h;
      *reinterpret_cast<float4*>(ilo + j) = l;
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
  if (scores_fused_supported(L, r)) return launch_scores_fused(L, qs, ks, r, s, flags, W, A, nullptr, nullptr, nullptr, st);
  const size_t smem = scores_smem_bytes();
  if (int32_t rc = allow_dynamic_smem(score_tile_kernel, smem, "sw_block_scores smem attribute")) return rc;
  dim3 grid(cdiv(L.max_blocks, kCols), cdiv(L.max_blocks, kRows), L.batch);
  count_launch(2);
  score_tile_kernel<<<grid, kThreads, smem, st>>>(qs, ks, r, flags, L.cu_blocks, L.cu_sq, W, 1.0f / sqrtf((float)r));
  score_rows_kernel<<<cdiv(L.total_blocks, kThreads / 32), kThreads, 0, st>>>(s, flags, L.cu_blocks, L.cu_sq, L.batch,
                                                                             W, A);
  return check_launch("sw_block_scores");
}

static size_t fused_smem_bytes(int max_blocks, int r, int* lds_out, int* stages_out) {
  const int lds = ((max_blocks + kFCols - 1) / kFCols) * kFCols + 4;   // whole 64-column tiles are written
  if (lds_out) *lds_out = lds;
  auto bytes = [&](int st) { return sizeof(float) * ((size_t)kFRows * r + (size_t)st * kFCols * (r + 4) + (size_t)kFRows * lds); };
  // two CTAs per SM (<= 110 KB each) beat a deeper ring with one (b = 2048: 96K against 124K cycles per SM)
  int st = kFStagesMax;
  while (st > 2 && bytes(st) > 110 * 1024) st >>= 1;
  if (stages_out) *stages_out = st;
  return bytes(st);
}

bool scores_fused_supported(const sw_layout& L, int r) {
  return r >= 4 && (r & (r - 1)) == 0 && r <= kRMax && fused_smem_bytes(L.max_blocks, r, nullptr, nullptr) <= 200 * 1024;
}

// W (and A) of sw_block_scores, plus -- when im != NULL -- the operand images of W and, when R_prev != NULL too,
// those of R_prev, in one launch.
int32_t launch_scores_fused(const sw_layout& L, const float* qs, const float* ks, int r, int s, uint32_t flags,
                            float* W, float* A, float* W2, const WalkImages* im, const float* R_prev,
                            cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  FusedParams p;
  p.qs = qs; p.ks = ks; p.r = r; p.s = s; p.flags = flags; p.cu_blocks = L.cu_blocks; p.cu_sq = L.cu_sq;
  p.W = W; p.A = A; p.W2 = W2;
  p.whi = im ? im->w_hi : nullptr; p.wlo = im ? im->w_lo : nullptr;
  p.R_prev = im ? R_prev : nullptr; p.rhi = im ? im->r_hi : nullptr; p.rlo = im ? im->r_lo : nullptr;
  p.pitch = im ? im->pitch : 0;
  p.n_strips = cdiv(im ? swimg::pad_rows(L.max_blocks) : L.max_blocks, kFRows);
  p.inv_sqrt_r = 1.0f / sqrtf((float)r);
  const size_t smem = fused_smem_bytes(L.max_blocks, r, &p.lds, &p.stages);
  void (*kern)(const FusedParams) = (r <= 64) ? score_fused_kernel<8> : score_fused_kernel<kRMax / 8>;
  if (int32_t rc = allow_dynamic_smem(kern, smem, "sw_block_scores(fused) smem attribute")) return rc;
  dim3 grid(p.n_strips * (p.R_prev ? 2 : 1), 1, L.batch);
  count_launch();
  kern<<<grid, kThreads, smem, st>>>(p);
  return check_launch("sw_block_scores(fused)");
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
