// sw_walk_update, tensor-core path for large b: R^k = R^{k-1} W^k (Lemma A.11 PAPER.md:571-576,
// Alg. 1 Step 6 PAPER.md:783-787) as a tcgen05 GEMM with the accumulator in TMEM and TMA-fed operands.
//
// Selection parity needs ~1e-5 relative accuracy (precision note), which one TF32 product
// (2^-11) does not give, so each fp32 operand is split  x = hi + lo,  hi = x with the low 13 mantissa
// bits cleared (exactly a TF32 number), lo = x - hi (exact in fp32, |lo| < 2^-10 |x|), and the product is
//     R W  ~=  R_hi W_hi + R_hi W_lo + R_lo W_hi          (3xTF32; dropped term <= 2^-20 relative)
// accumulated in fp32 in TMEM.  The hi / lo images live in the caller's workspace (walk_images.cuh: all
// sequences of a batch stacked with one row pitch, zero padded, so that ONE tensor map per operand serves a
// varlen batch); they are written by split_tf32_kernel here, or directly by the fused score kernel
// (scores.cu).  Converting inside the GEMM would double the shared-memory traffic of a kernel that is already
// bound by the tensor core's operand reads (SS MMA at M = N = 128 reads 128 B/clk).
//
// GEMM: one CTA per 128x128 output tile (sequence, ti, tj).  With SW_CAUSAL both operands are lower
// triangular, so the reduction of tile (ti, tj) runs over k in [128 tj, 128 (ti+1)) only and tiles with
// tj > ti are zero (written only when asked: the fused selection path fills them itself); tiles are issued
// longest first.  K step = 32 fp32 (128-byte rows):
//   A = R_hi / R_lo [128 x 32]  K-major,  SWIZZLE_128B        (one TMA box each)
//   B = W_hi / W_lo [32 x 128]  MN-major, SWIZZLE_128B_ATOM_32B (four 32x32 TMA boxes each; 32-bit
//       MN-major operands need the 32-byte-atom swizzle, see sm100.cuh)
//   12 x tcgen05.mma.kind::tf32 M=128 N=128 K=8 per step, 3-stage ring of 64 KB.
// The tensor core adds into its fp32 accumulator with truncation, so the error of one long accumulation
// chain grows linearly with its length (measured 2e-5 of the row max at b = 1156); k-step ks therefore
// adds into accumulator ks % 4 (all 512 TMEM columns) and the epilogue sums the four in fp32.
// Warps: 0 = TMA producer, 1 = MMA issuer, 2-5 = epilogue (TMEM -> registers -> global, causal mask).
#include "common.cuh"
#include "sm100.cuh"
#include "walk_images.cuh"

namespace {

using namespace sm100;

constexpr int BM = 128, BN = 128, BK = 32;
constexpr int kStages = 3;
constexpr int kTileBytes = BM * BK * 4;              // 16 KB (A and B tiles have the same size)
constexpr int kStageBytes = 4 * kTileBytes;          // A_hi, A_lo, B_hi, B_lo
constexpr int kThreads = 192;
constexpr int kAcc = 4;                              // TMEM accumulators (k-step ks adds into ks % 4)
constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*align*/ + 256 /*barriers*/;

// x = hi + lo with hi a TF32 number (low 13 mantissa bits zero) and lo = x - hi exact.  Packed per-sequence
// matrices (cu_sq) -> stacked, pitched, zero-padded images.  grid = (padded rows, 2 = R / W, batch).
__global__ void __launch_bounds__(256)
split_tf32_kernel(const float* __restrict__ R, const float* __restrict__ W, float* __restrict__ Rhi,
                  float* __restrict__ Rlo, float* __restrict__ Whi, float* __restrict__ Wlo,
                  const int32_t* __restrict__ cu_blocks, const int64_t* __restrict__ cu_sq, int pitch, int causal) {
  const int i = blockIdx.x, seq = blockIdx.z;
  const float* src = blockIdx.y ? W : R;
  float* hi = blockIdx.y ? Whi : Rhi;
  float* lo = blockIdx.y ? Wlo : Rlo;
  if (src == nullptr) return;
  const int b = __ldg(cu_blocks + seq + 1) - __ldg(cu_blocks + seq);
  if (i >= swimg::pad_rows(b)) return;
  const int64_t irow = (int64_t)(swimg::row_base(cu_blocks, seq) + i) * pitch;
  swimg::split_row(src + __ldg(cu_sq + seq) + (int64_t)i * b, i, b, pitch, causal, hi + irow, lo + irow,
                   threadIdx.x, 256);
}

// kind::tf32, fp32 accumulate: [4,6) D fmt = 1 (f32), [7,10) A fmt = 2 (tf32), [10,13) B fmt = 2,
// [15] A major (0 = K), [16] B major (1 = MN), [17,23) N >> 3, [24,29) M >> 4.
__host__ __device__ constexpr uint32_t idesc_tf32(int M, int N, int b_mn_major) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
         ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void mma_tf32_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                            uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* m, uint32_t bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(c0), "r"(c1) : "memory");
}

struct Params {
  float* out;                     // packed per-sequence matrices (cu_sq)
  const int32_t* cu_blocks;
  const int64_t* cu_sq;
  int causal, zero_upper;         // zero_upper: also write the strictly upper tiles (as zeros)
};

__global__ void __launch_bounds__(kThreads, 1)
walk_tc_kernel(const __grid_constant__ CUtensorMap map_rhi, const __grid_constant__ CUtensorMap map_rlo,
               const __grid_constant__ CUtensorMap map_whi, const __grid_constant__ CUtensorMap map_wlo,
               const Params p) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int seq = blockIdx.y;
  const int b = __ldg(p.cu_blocks + seq + 1) - __ldg(p.cu_blocks + seq);
  const int nt = (b + BM - 1) / BM;
  const int n_work = p.causal ? nt * (nt + 1) / 2 : nt * nt;
  float* out = p.out + __ldg(p.cu_sq + seq);
  const int rbase = swimg::row_base(p.cu_blocks, seq);

  // ---- tile of this CTA: GEMM tiles longest first (by ti - tj), then the zero tiles -------------
  int ti, tj;
  bool zero_tile = false;
  {
    int w = blockIdx.x;
    if (!p.causal) {
      if (w >= n_work) return;
      ti = w / nt; tj = w - ti * nt;
    } else if (w < n_work) {
      int dgap = nt - 1;                     // tiles with ti - tj = dgap: nt - dgap of them
      while (w >= nt - dgap) { w -= nt - dgap; --dgap; }
      tj = w; ti = tj + dgap;
    } else {
      w -= n_work;                           // strictly upper tiles, row-major
      if (!p.zero_upper || w >= nt * (nt - 1) / 2) return;
      zero_tile = true;
      ti = 0;
      while (w >= nt - 1 - ti) { w -= nt - 1 - ti; ++ti; }
      tj = ti + 1 + w;
    }
  }
  const int row0 = ti * BM, col0 = tj * BN;
  const bool vec_out = (b & 3) == 0 && (reinterpret_cast<uintptr_t>(out) & 15u) == 0;
  if (zero_tile) {
    for (int e = threadIdx.x; e < BM * (BN / 4); e += kThreads) {
      const int r = row0 + e / (BN / 4), c = col0 + (e % (BN / 4)) * 4;
      if (r < b) {
        if (vec_out) {
          if (c < b) *reinterpret_cast<float4*>(out + (int64_t)r * b + c) = make_float4(0.f, 0.f, 0.f, 0.f);
        } else {
          for (int f = 0; f < 4; ++f)
            if (c + f < b) out[(int64_t)r * b + c + f] = 0.f;
        }
      }
    }
    return;
  }

  extern __shared__ uint8_t smem_raw[];
  uint8_t* base = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const uint32_t sTiles = smem_u32(base);
  uint64_t* bars = reinterpret_cast<uint64_t*>(base + kStages * kStageBytes);
  const uint32_t bar0 = smem_u32(bars);
  auto FULL = [&](int s) { return bar0 + 8u * s; };
  auto EMPTY = [&](int s) { return bar0 + 8u * (kStages + s); };
  const uint32_t DONE = bar0 + 8u * (2 * kStages);
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(bars + 2 * kStages + 1);

  const int k_begin = p.causal ? col0 : 0;                 // W[m][j] = 0 for m < j
  const int k_end = p.causal ? min(b, row0 + BM) : b;      // R[i][m] = 0 for m > i
  const int nk = (k_end - k_begin + BK - 1) / BK;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&map_rhi); prefetch_tmap(&map_rlo); prefetch_tmap(&map_whi); prefetch_tmap(&map_wlo);
    for (int s = 0; s < kStages; ++s) { mbar_init(FULL(s), 1); mbar_init(EMPTY(s), 1); }
    mbar_init(DONE, 1);
    fence_barrier_init();
  } else if (warp == 2) {
    tmem_alloc<kAcc * BN>(smem_u32((const void*)s_tmem));
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tm = *s_tmem;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      for (int ks = 0; ks < nk; ++ks) {
        const int st = ks % kStages;
        mbar_wait(EMPTY(st), ((ks / kStages) & 1) ^ 1);
        const uint32_t dst = sTiles + st * kStageBytes;
        const int k = k_begin + ks * BK;
        mbar_arrive_expect_tx(FULL(st), kStageBytes);
        tma_load_2d(dst, &map_rhi, FULL(st), k, rbase + row0);
        tma_load_2d(dst + kTileBytes, &map_rlo, FULL(st), k, rbase + row0);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          tma_load_2d(dst + 2 * kTileBytes + c * 4096, &map_whi, FULL(st), col0 + c * 32, rbase + k);
          tma_load_2d(dst + 3 * kTileBytes + c * 4096, &map_wlo, FULL(st), col0 + c * 32, rbase + k);
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (elect_one()) {
      const uint32_t id = idesc_tf32(BM, BN, 1);
      for (int ks = 0; ks < nk; ++ks) {
        const int st = ks % kStages;
        mbar_wait(FULL(st), (ks / kStages) & 1);
        tc_fence_after();
        const uint32_t a_hi = sTiles + st * kStageBytes, a_lo = a_hi + kTileBytes;
        const uint32_t b_hi = a_hi + 2 * kTileBytes, b_lo = a_hi + 3 * kTileBytes;
        // small terms first, the hi*hi term last
#pragma unroll
        for (int t = 0; t < 3; ++t) {
          const uint32_t sa = (t == 0) ? a_lo : a_hi;
          const uint32_t sb = (t == 1) ? b_lo : b_hi;
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
            mma_tf32_ss(tm + (ks & (kAcc - 1)) * BN, desc_kmajor_sw128(sa + kk * 32),
                        desc_mnmajor_sw128_atom32(sb + kk * 1024, 4096, 512), id,
                        (ks >= kAcc || t > 0 || kk > 0) ? 1u : 0u);
        }
        mma_commit(EMPTY(st));
      }
      mma_commit(DONE);
    }
  } else {
    // ===================== epilogue: one thread per output row =====================
    const int q = warp & 3;                               // TMEM lane quadrant this warp may read
    const int r = row0 + q * 32 + lane;
    const int nacc = min(nk, kAcc);
    mbar_wait(DONE, 0);
    tc_fence_after();
#pragma unroll
    for (int ch = 0; ch < 4; ++ch) {
      uint32_t v[32];
      tmem_ld32(tm + ((uint32_t)(q * 32) << 16) + ch * 32, v);
      tmem_wait_ld();
      for (int a = 1; a < nacc; ++a) {                    // fp32 (round-to-nearest) sum of the accumulators
        uint32_t w[32];
        tmem_ld32(tm + ((uint32_t)(q * 32) << 16) + a * BN + ch * 32, w);
        tmem_wait_ld();
#pragma unroll
        for (int e = 0; e < 32; ++e) v[e] = __float_as_uint(__uint_as_float(v[e]) + __uint_as_float(w[e]));
      }
      if (r < b) {
        float* dst = out + (int64_t)r * b + col0 + ch * 32;
#pragma unroll
        for (int e = 0; e < 32; e += 4) {
          const int c = col0 + ch * 32 + e;
          float4 o;
          o.x = (p.causal && c + 0 > r) ? 0.f : __uint_as_float(v[e + 0]);
          o.y = (p.causal && c + 1 > r) ? 0.f : __uint_as_float(v[e + 1]);
          o.z = (p.causal && c + 2 > r) ? 0.f : __uint_as_float(v[e + 2]);
          o.w = (p.causal && c + 3 > r) ? 0.f : __uint_as_float(v[e + 3]);
          if (vec_out) {
            if (c < b) *reinterpret_cast<float4*>(dst + e) = o;     // b % 4 == 0: a float4 is inside or outside
          } else {
            if (c + 0 < b) dst[e + 0] = o.x;
            if (c + 1 < b) dst[e + 1] = o.y;
            if (c + 2 < b) dst[e + 2] = o.z;
            if (c + 3 < b) dst[e + 3] = o.w;
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc<kAcc * BN>(tm);
}

// stacked images [rows, pitch] fp32 -> 2-D map (pitch, rows), box = (32 cols = 128 B, box_rows), 128-byte swizzle
bool make_map_f32(CUtensorMap* map, const float* base, int rows, int pitch, int box_rows, bool atom32) {
  sm100host::EncodeTiledFn fn = sm100host::encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {(cuuint64_t)pitch, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)pitch * 4};
  cuuint32_t box[2] = {32, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, atom32 ? CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B : CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

namespace sw {

bool walk_tc_supported(const sw_layout& L) {
  return L.batch >= 1 && L.max_blocks >= 256 && sm100host::encode_fn() != nullptr;
}

WalkImages walk_images(const sw_layout& L, void* ws_images) {
  WalkImages im;
  im.pitch = swimg::pitch_of(L.max_blocks);
  im.rows = swimg::rows_bound(L.total_blocks, L.batch);
  const size_t n = (size_t)im.rows * im.pitch;
  float* f = reinterpret_cast<float*>(ws_images);
  im.r_hi = f; im.r_lo = f + n; im.w_hi = f + 2 * n; im.w_lo = f + 3 * n;
  return im;
}

size_t walk_tc_ws_bytes(const sw_layout& L) {
  if (!walk_tc_supported(L)) return 0;
  return (size_t)4 * swimg::rows_bound(L.total_blocks, L.batch) * swimg::pitch_of(L.max_blocks) * sizeof(float);
}

int32_t launch_split_tf32(const sw_layout& L, const float* R, const float* W, const WalkImages& im, int causal,
                          cudaStream_t st) {
  dim3 grid(swimg::pad_rows(L.max_blocks), 2, L.batch);
  count_launch();
  split_tf32_kernel<<<grid, 256, 0, st>>>(R, W, im.r_hi, im.r_lo, im.w_hi, im.w_lo, L.cu_blocks, L.cu_sq, im.pitch,
                                          causal);
  return check_launch("sw_walk_update(split)");
}

// One product dst = R * W per sequence on the tensor cores, operands = the hi / lo images in `im`.
int32_t launch_walk_tc(const sw_layout& L, const WalkImages& im, float* dst, int causal, bool zero_upper,
                       cudaStream_t st) {
  CUtensorMap mrh, mrl, mwh, mwl;
  const bool ok = make_map_f32(&mrh, im.r_hi, im.rows, im.pitch, BM, false) &&
                  make_map_f32(&mrl, im.r_lo, im.rows, im.pitch, BM, false) &&
                  make_map_f32(&mwh, im.w_hi, im.rows, im.pitch, BK, true) &&
                  make_map_f32(&mwl, im.w_lo, im.rows, im.pitch, BK, true);
  if (!ok) return fail(SW_ERR_CUDA, "sw_walk_update: cuTensorMapEncodeTiled failed");
  if (int32_t rc = allow_dynamic_smem(walk_tc_kernel, kSmemBytes, "sw_walk_update(tcgen05) smem attribute")) return rc;
  Params p;
  p.out = dst; p.cu_blocks = L.cu_blocks; p.cu_sq = L.cu_sq; p.causal = causal; p.zero_upper = zero_upper ? 1 : 0;
  const int nt = cdiv(L.max_blocks, BM);
  const int tiles = (causal && !zero_upper) ? nt * (nt + 1) / 2 : nt * nt;
  count_launch();
  walk_tc_kernel<<<dim3(tiles, L.batch), kThreads, kSmemBytes, st>>>(mrh, mrl, mwh, mwl, p);
  return check_launch("sw_walk_update(tcgen05)");
}

}  // namespace sw
