// sw_sparse_attn_prefill, sm_100a fast path: block-sparse FlashAttention on tcgen05 tensor cores with
// TMEM accumulators and TMA-gathered K/V tiles.  Alg. 1 Step 8, "zero outside selected
// blocks, renormalized within"; GQA mapping P14.
//
// Work unit (one CTA): a 64-token query tile of one KV-head group (4 q-heads) = 256 query rows, row =
// 4*token + head, processed as two 128-row MMA tiles t = 0, 1.  The selected key blocks of the query
// block are cut into 64-key chunks and consumed two at a time (a 128-key tile):
//     S_t = Q_t K^T      tcgen05.mma  M=128 N=128 K=16 x8   A, B from shared memory (K-major, SW128)
//     P_t = exp2(S_t*c - m)  fp32 online softmax in registers, one thread per row, P written back to
//                            TMEM as bf16 over the S columns
//     O_t += P_t V       tcgen05.mma  M=128 N=128 K=16 x8   A from TMEM, B from shared memory (MN-major)
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512).
// Warps: 0 = TMA producer, 1 = MMA issuer, 2 = TMEM allocator, 3 = chunk-list builder,
//        4-7 = softmax/epilogue of tile 0, 8-11 = softmax/epilogue of tile 1.
// The MMA order  PV0(j) QK0(j+1) PV1(j) QK1(j+1)  lets the softmax of one tile overlap the tensor work
// of the other.  The O rescale is lazy: the running max is only raised (and O multiplied) when it grew
// by more than 2^8, which keeps P within bf16/fp32 range and is exact after the final 1/l.
#include "common.cuh"
#include "sm100.cuh"

namespace {

using namespace sm100;

constexpr int kThreads = 384;
constexpr int kStages = 4;                    // ring of 128-key K or V tiles
constexpr int kTileBytes = 128 * 128 * 2;     // 32 KB: [d-half][128 keys][128 B]
constexpr int kQBytes = 256 * 128 * 2;        // 64 KB: [d-half][256 rows][128 B]
constexpr int kMaxChunks = 4096;              // 64-key chunks per query row the list buffer holds
constexpr int kSmemBytes = kQBytes + kStages * kTileBytes + kMaxChunks * 4 + 1024 /*align*/ + 256 /*barriers*/;
constexpr float kRescaleThreshold = 8.0f;     // log2 units

struct Params {
  const int32_t* cu_seqlens;
  const int32_t* cu_blocks;
  const int32_t* idx;
  const int32_t* count;
  void* out;                     // bf16 or fp32 [total_tokens, h_q, 128]
  float* lse;
  int batch, B, total_slots, tau_max, h_q, causal, out_f32;
  float scale_log2;
};

__device__ __forceinline__ float fmax3(float a, float b, float c) {
  float r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}
__device__ __forceinline__ float ex2(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
template <int N> __device__ __forceinline__ void reg_alloc() {
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N> __device__ __forceinline__ void reg_dealloc() {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

__global__ void __launch_bounds__(kThreads, 1)
attn_prefill_sm100_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                          const __grid_constant__ CUtensorMap map_v, const Params p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* base = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const uint32_t sQ = smem_u32(base);
  const uint32_t sKV = sQ + kQBytes;
  int32_t* s_list = reinterpret_cast<int32_t*>(base + kQBytes + kStages * kTileBytes);
  uint64_t* bars = reinterpret_cast<uint64_t*>(base + kQBytes + kStages * kTileBytes + kMaxChunks * 4);
  // barrier map: 0 q_full | 1..4 full[stage] | 5..8 empty[stage] | 9,10 s_full[t] | 11,12 p_full[t] | 13 o_full
  const uint32_t bar0 = smem_u32(bars);
  auto BAR = [&](int i) { return bar0 + 8u * i; };
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(bars + 16);
  volatile int32_t* s_nchunks = reinterpret_cast<volatile int32_t*>(bars + 17);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- work unit ---------------------------------------------------------------------------
  const int TPB = p.B >> 6;
  const int slot_id = p.total_slots - 1 - (int)blockIdx.x;     // longest rows first
  const int gb = slot_id / TPB, sub = slot_id - gb * TPB;
  const int kvh = blockIdx.y;
  const int seq = swd::find_seq(p.cu_blocks, p.batch, gb);
  const int bi = gb - __ldg(p.cu_blocks + seq);
  const int seq_lo = __ldg(p.cu_seqlens + seq), seq_hi = __ldg(p.cu_seqlens + seq + 1);
  const int q_tok0 = seq_lo + bi * p.B + sub * 64;
  const int q_valid = min(64, seq_hi - q_tok0);
  if (q_valid <= 0) return;
  const int q_last = q_tok0 + q_valid - 1;

  // ---- one-time setup ------------------------------------------------------------------------
  if (warp == 0 && lane == 0) {
    prefetch_tmap(&map_q); prefetch_tmap(&map_k); prefetch_tmap(&map_v);
    mbar_init(BAR(0), 1);
    for (int s = 0; s < kStages; ++s) { mbar_init(BAR(1 + s), 1); mbar_init(BAR(5 + s), 1); }
    mbar_init(BAR(9), 1); mbar_init(BAR(10), 1);
    mbar_init(BAR(11), 4); mbar_init(BAR(12), 4);
    mbar_init(BAR(13), 1);
    fence_barrier_init();
  } else if (warp == 2) {
    tmem_alloc<512>(smem_u32((const void*)s_tmem));
  } else if (warp == 3) {
    // 64-key chunks (token offset of their first key) of the selected blocks that hold a visible key
    const int cnt = __ldg(p.count + gb);
    const int32_t* list = p.idx + (int64_t)gb * p.tau_max;
    const int total = cnt * TPB;
    int n = 0;
    for (int base_i = 0; base_i < total; base_i += 32) {
      const int i = base_i + lane;
      int k0 = -1;
      if (i < total) {
        const int j = __ldg(list + i / TPB);
        if (j >= 0) {
          k0 = seq_lo + j * p.B + (i % TPB) * 64;
          if (k0 >= seq_hi || (p.causal && k0 > q_last)) k0 = -1;
        }
      }
      const unsigned m = __ballot_sync(0xffffffffu, k0 >= 0);
      if (k0 >= 0) {
        const int pos = n + __popc(m & ((1u << lane) - 1));
        if (pos < kMaxChunks) s_list[pos] = k0;
      }
      n += __popc(m);
    }
    if (lane == 0) *s_nchunks = min(n, kMaxChunks);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tm = *s_tmem;
  const int n_chunks = *s_nchunks;
  const int n_iter = (n_chunks + 1) >> 1;

  if (warp < 4) {
  reg_dealloc<64>();                                          // 128*64 + 256*216 <= 64 K registers
  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0 && n_iter > 0) {
      mbar_arrive_expect_tx(BAR(0), kQBytes);
      tma_load_3d(sQ, &map_q, BAR(0), 0, kvh * 4, q_tok0);
      tma_load_3d(sQ + kQBytes / 2, &map_q, BAR(0), 64, kvh * 4, q_tok0);
      for (int it = 0; it < n_iter; ++it) {
        const int nblk = min(2, n_chunks - 2 * it);
#pragma unroll
        for (int kv = 0; kv < 2; ++kv) {
          const int qn = 2 * it + kv;
          const int st = qn % kStages;
          mbar_wait(BAR(5 + st), ((qn / kStages) & 1) ^ 1);
          mbar_arrive_expect_tx(BAR(1 + st), nblk * (kTileBytes / 2));
          const CUtensorMap* m = kv ? &map_v : &map_k;
          const uint32_t dst = sKV + st * kTileBytes;
          for (int h = 0; h < nblk; ++h) {
            const int k0 = s_list[2 * it + h];
            tma_load_3d(dst + h * 8192, m, BAR(1 + st), 0, kvh, k0);
            tma_load_3d(dst + 16384 + h * 8192, m, BAR(1 + st), 64, kvh, k0);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0 && n_iter > 0) {
      const uint32_t id_full = idesc_bf16(128, 128, 0, 0), id_half = idesc_bf16(128, 64, 0, 0);
      const uint32_t id_pv = idesc_bf16(128, 128, 0, 1);
      auto issue_qk = [&](int t, uint32_t sK, int nblk) {
        const uint32_t id = nblk == 2 ? id_full : id_half;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t a = sQ + (kk >> 2) * (kQBytes / 2) + t * 16384 + (kk & 3) * 32;
          const uint32_t b = sK + (kk >> 2) * 16384 + (kk & 3) * 32;
          mma_ss(tm + t * 128, desc_kmajor_sw128(a), desc_kmajor_sw128(b), id, kk > 0);
        }
        mma_commit(BAR(9 + t));
      };
      auto issue_pv = [&](int t, uint32_t sV, int nblk, bool acc) {
        for (int kk = 0; kk < 4 * nblk; ++kk)
          mma_ts(tm + 256 + t * 128, tm + t * 128 + kk * 8, desc_mnmajor_sw128(sV + kk * 2048, 16384, 1024), id_pv,
                 (acc || kk > 0) ? 1u : 0u);
      };
      mbar_wait(BAR(0), 0);
      mbar_wait(BAR(1 + 0), 0);
      tc_fence_after();
      {
        const int nblk = min(2, n_chunks);
        issue_qk(0, sKV, nblk);
        issue_qk(1, sKV, nblk);
        mma_commit(BAR(5 + 0));
      }
      for (int j = 0; j < n_iter; ++j) {
        const int nblk = min(2, n_chunks - 2 * j);
        const int qv = 2 * j + 1, sv = qv % kStages;
        const int qk = 2 * j + 2, sk = qk % kStages;
        const bool more = (j + 1 < n_iter);
        const int nblk_next = more ? min(2, n_chunks - 2 * (j + 1)) : 0;
        mbar_wait(BAR(1 + sv), (qv / kStages) & 1);
        mbar_wait(BAR(11), j & 1);
        tc_fence_after();
        issue_pv(0, sKV + sv * kTileBytes, nblk, j > 0);
        if (more) {
          mbar_wait(BAR(1 + sk), (qk / kStages) & 1);
          tc_fence_after();
          issue_qk(0, sKV + sk * kTileBytes, nblk_next);
        }
        mbar_wait(BAR(12), j & 1);
        tc_fence_after();
        issue_pv(1, sKV + sv * kTileBytes, nblk, j > 0);
        mma_commit(BAR(5 + sv));
        if (more) {
          issue_qk(1, sKV + sk * kTileBytes, nblk_next);
          mma_commit(BAR(5 + sk));
        }
      }
      mma_commit(BAR(13));
    }
  }
  } else {
    reg_alloc<216>();
    // ===================== softmax + epilogue: one thread per query row =====================
    const int t = (warp - 4) >> 2;                       // MMA tile
    const int w4 = warp & 3;                             // TMEM lane quadrant of this warp
    const int row = w4 * 32 + lane;                      // row in the tile
    const int q_pos = q_tok0 + t * 32 + (row >> 2);      // global token index of this row
    const int head = kvh * 4 + (row & 3);
    const uint32_t t_s = tm + ((uint32_t)(w4 * 32) << 16) + t * 128;
    const uint32_t t_o = tm + ((uint32_t)(w4 * 32) << 16) + 256 + t * 128;
    float m_run = -INFINITY, l_run = 0.f;
    const float c = p.scale_log2;

    for (int j = 0; j < n_iter; ++j) {
      const int nblk = min(2, n_chunks - 2 * j);
      mbar_wait(BAR(9 + t), j & 1);
      tc_fence_after();
      uint32_t s[128];
      tmem_ld32(t_s + 0, *reinterpret_cast<uint32_t(*)[32]>(&s[0]));
      tmem_ld32(t_s + 32, *reinterpret_cast<uint32_t(*)[32]>(&s[32]));
      if (nblk == 2) {
        tmem_ld32(t_s + 64, *reinterpret_cast<uint32_t(*)[32]>(&s[64]));
        tmem_ld32(t_s + 96, *reinterpret_cast<uint32_t(*)[32]>(&s[96]));
      }
      tmem_wait_ld();
      if (nblk < 2) {
#pragma unroll
        for (int i = 64; i < 128; ++i) s[i] = 0xff800000u;   // -inf
      }
      // masks: only chunks that touch the diagonal or the end of the sequence
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (h < nblk) {
          const int k0 = s_list[2 * j + h];
          const bool need = (p.causal && k0 + 63 > q_tok0) || (k0 + 64 > seq_hi);
          if (need) {
            const int lim = min(p.causal ? q_pos : 0x7fffffff, seq_hi - 1) - k0;   // visible iff col <= lim
#pragma unroll
            for (int i = 0; i < 64; ++i)
              if (i > lim) s[h * 64 + i] = 0xff800000u;
          }
        }
      }
      float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
      for (int i = 0; i < 128; i += 4) {
        mx0 = fmax3(mx0, __uint_as_float(s[i]), __uint_as_float(s[i + 1]));
        mx1 = fmax3(mx1, __uint_as_float(s[i + 2]), __uint_as_float(s[i + 3]));
      }
      const float m_tile = fmaxf(mx0, mx1) * c;           // c > 0
      // lazy rescale
      float m_new = m_run;
      const bool grow = m_tile > m_run + kRescaleThreshold;   // also true for the first finite tile
      if (grow) m_new = m_tile;
      if (j > 0 && __any_sync(0xffffffffu, grow)) {
        const float f = (m_new == m_run) ? 1.f : ex2(m_run - m_new);   // m_run = -inf -> 0
        l_run *= f;
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          uint32_t o[32];
          tmem_ld32(t_o + ch * 32, o);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
          tmem_st32(t_o + ch * 32, o);
        }
      }
      m_run = m_new;
      const float m_use = (m_run == -INFINITY) ? 0.f : m_run;
      float sum0 = 0.f, sum1 = 0.f;
      uint32_t pk[64];
#pragma unroll
      for (int i = 0; i < 64; ++i) {
        const float a = ex2(fmaf(__uint_as_float(s[2 * i]), c, -m_use));
        const float b = ex2(fmaf(__uint_as_float(s[2 * i + 1]), c, -m_use));
        sum0 += a; sum1 += b;
        pk[i] = pack_bf16(a, b);
      }
      l_run += sum0 + sum1;
      tmem_st32(t_s + 0, *reinterpret_cast<uint32_t(*)[32]>(&pk[0]));
      if (nblk == 2) tmem_st32(t_s + 32, *reinterpret_cast<uint32_t(*)[32]>(&pk[32]));
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(BAR(11 + t));
    }

    // epilogue: O / l -> bf16 -> global
    if (n_iter > 0) {
      mbar_wait(BAR(13), 0);
      tc_fence_after();
    }
    const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
    const bool valid = q_pos <= q_last;
    const int64_t o_off = ((int64_t)q_pos * p.h_q + head) * 128;
    __nv_bfloat16* op = reinterpret_cast<__nv_bfloat16*>(p.out) + o_off;
    float* opf = reinterpret_cast<float*>(p.out) + o_off;
#pragma unroll
    for (int ch = 0; ch < 4; ++ch) {
      uint32_t o[32];
      if (n_iter > 0) {
        tmem_ld32(t_o + ch * 32, o);
        tmem_wait_ld();
      } else {
#pragma unroll
        for (int i = 0; i < 32; ++i) o[i] = 0u;
      }
      if (valid && p.out_f32) {
#pragma unroll
        for (int v = 0; v < 8; ++v)
          *reinterpret_cast<float4*>(opf + ch * 32 + v * 4) =
              make_float4(__uint_as_float(o[4 * v + 0]) * inv, __uint_as_float(o[4 * v + 1]) * inv,
                          __uint_as_float(o[4 * v + 2]) * inv, __uint_as_float(o[4 * v + 3]) * inv);
      } else if (valid) {
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          uint4 w;
          w.x = pack_bf16(__uint_as_float(o[8 * v + 0]) * inv, __uint_as_float(o[8 * v + 1]) * inv);
          w.y = pack_bf16(__uint_as_float(o[8 * v + 2]) * inv, __uint_as_float(o[8 * v + 3]) * inv);
          w.z = pack_bf16(__uint_as_float(o[8 * v + 4]) * inv, __uint_as_float(o[8 * v + 5]) * inv);
          w.w = pack_bf16(__uint_as_float(o[8 * v + 6]) * inv, __uint_as_float(o[8 * v + 7]) * inv);
          *reinterpret_cast<uint4*>(op + ch * 32 + v * 8) = w;
        }
      }
    }
    if (p.lse && valid)
      p.lse[(int64_t)q_pos * p.h_q + head] =
          l_run > 0.f ? (m_run + log2f(l_run)) * 0.6931471805599453f : -INFINITY;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc<512>(tm);
}

}  // namespace

namespace sw {

bool attn_prefill_sm100_supported(const AttnPrefillArgs& a) {
  if (a.d != 128) return false;
  if (a.h_kv <= 0 || a.h_q != 4 * a.h_kv) return false;
  if ((int64_t)a.tau_max * (a.L->block / 64) > kMaxChunks) return false;
  if (!sm100host::encode_fn()) return false;
  return true;
}

int32_t launch_attn_prefill_sm100(const AttnPrefillArgs& a, cudaStream_t st) {
  const sw_layout& L = *a.L;
  if (L.total_blocks == 0 || L.total_tokens == 0) return SW_OK;
  CUtensorMap mq, mk, mv;
  const bool ok = sm100host::make_map_thd(&mq, a.q, L.total_tokens, a.h_q, 128, a.q_stride_tok, a.q_stride_head, 4, 64) &&
                  sm100host::make_map_thd(&mk, a.k, L.total_tokens, a.h_kv, 128, a.k_stride_tok, a.k_stride_head, 1, 64) &&
                  sm100host::make_map_thd(&mv, a.v, L.total_tokens, a.h_kv, 128, a.v_stride_tok, a.v_stride_head, 1, 64);
  if (!ok) return fail(SW_ERR_CUDA, "sw_sparse_attn_prefill: cuTensorMapEncodeTiled failed");
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(attn_prefill_sm100_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes) !=
        cudaSuccess)
      return check_launch("sw_sparse_attn_prefill(sm100) smem attribute");
    attr_set = true;
  }
  Params p;
  p.cu_seqlens = L.cu_seqlens; p.cu_blocks = L.cu_blocks; p.idx = a.idx; p.count = a.count;
  p.out = a.out; p.lse = a.lse; p.out_f32 = (a.out_dtype == SW_F32) ? 1 : 0;
  p.batch = L.batch; p.B = L.block; p.total_slots = L.total_blocks * (L.block / 64); p.tau_max = a.tau_max;
  p.h_q = a.h_q; p.causal = (a.flags & SW_CAUSAL) ? 1 : 0;
  p.scale_log2 = a.softmax_scale * 1.4426950408889634f;
  dim3 grid(p.total_slots, a.h_kv);
  attn_prefill_sm100_kernel<<<grid, kThreads, kSmemBytes, st>>>(mq, mk, mv, p);
  return check_launch("sw_sparse_attn_prefill(sm100)");
}

}  // namespace sw
