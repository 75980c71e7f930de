// sw_sparse_attn_prefill, generic path: block-sparse FlashAttention-style kernel on warp-level
// tensor-core MMA (mma.sync m16n8k16 bf16, fp32 accumulate, fp32 online softmax).  It serves every
// shape the tcgen05 path (attn_prefill_sm100.cu) does not take: d = 64, GQA groups other than 4,
// fp32 I/O (after the bf16 cast pre-pass, P17).  Alg. 1 Step 8.
//
// CTA = 4 warps = one 64-token query tile of one q-head; it walks the selected key blocks of its
// query block (idx/count from sw_select_topk) in 64-key tiles, double-buffered with cp.async.
#include "common.cuh"
#include "mma_sync.cuh"

namespace {

using namespace swmma;

constexpr int kThreads = 128;
constexpr int QT = 64;         // query rows per CTA
constexpr int KT = 64;         // keys per tile


template <int D>
__device__ __forceinline__ void load_tile(uint32_t s_base, const __nv_bfloat16* g, int64_t stride_tok,
                                          int valid_rows) {
  constexpr int CH = D / 8;
  for (int i = threadIdx.x; i < 64 * CH; i += kThreads) {
    const int row = i / CH, ch = i % CH;
    const bool ok = row < valid_rows;
    cp_async16(s_base + tile_off<D>(row, ch), ok ? (const void*)(g + (int64_t)row * stride_tok + ch * 8) : (const void*)g, ok);
  }
}

template <int D, typename OutT>
__global__ void __launch_bounds__(kThreads)
attn_prefill_generic_kernel(const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
                            const __nv_bfloat16* __restrict__ V, int64_t q_st, int64_t q_sh, int64_t k_st,
                            int64_t k_sh, int64_t v_st, int64_t v_sh, int h_q, int h_kv,
                            const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ cu_blocks,
                            int batch, int B, int total_slots, const int32_t* __restrict__ idx,
                            const int32_t* __restrict__ count, int tau_max, float scale_log2, int causal,
                            OutT* __restrict__ out, float* __restrict__ lse) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  constexpr int TILE_BYTES = 64 * D * 2;
  const uint32_t s_q = smem_u32(smem_raw);
  const uint32_t s_k0 = s_q + TILE_BYTES;            // K[2]
  const uint32_t s_v0 = s_k0 + 2 * TILE_BYTES;       // V[2]

  const int TPB = B / 64;                            // 64-token tiles per block
  const int slot_id = total_slots - 1 - blockIdx.x;  // longest rows first
  const int gb = slot_id / TPB, sub = slot_id % TPB;
  const int head = blockIdx.y;
  const int kvh = head / (h_q / h_kv);
  const int seq = swd::find_seq(cu_blocks, batch, gb);
  const int bi = gb - __ldg(cu_blocks + seq);
  const int seq_lo = __ldg(cu_seqlens + seq), seq_hi = __ldg(cu_seqlens + seq + 1);
  const int q_tok0 = seq_lo + bi * B + sub * QT;
  const int q_valid = min(QT, seq_hi - q_tok0);
  if (q_valid <= 0) return;
  const int cnt = __ldg(count + gb);
  const int32_t* list = idx + (int64_t)gb * tau_max;
  const int nslots = cnt * TPB;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t4 = lane & 3;

  // slot -> key tile; returns false when the tile holds no visible key
  auto slot_info = [&](int slot, int& k_tok0, int& k_valid) -> bool {
    const int j = __ldg(list + slot / TPB);
    k_tok0 = seq_lo + j * B + (slot % TPB) * KT;
    k_valid = min(KT, seq_hi - k_tok0);
    if (j < 0 || k_valid <= 0) return false;
    if (causal && k_tok0 > q_tok0 + q_valid - 1) return false;
    return true;
  };
  auto next_active = [&](int slot) {
    int a, b2;
    for (++slot; slot < nslots; ++slot)
      if (slot_info(slot, a, b2)) break;
    return slot;
  };
  auto issue = [&](int slot, int buf) {
    int k_tok0, k_valid;
    slot_info(slot, k_tok0, k_valid);
    load_tile<D>(s_k0 + buf * TILE_BYTES, K + (int64_t)k_tok0 * k_st + (int64_t)kvh * k_sh, k_st, k_valid);
    load_tile<D>(s_v0 + buf * TILE_BYTES, V + (int64_t)k_tok0 * v_st + (int64_t)kvh * v_sh, v_st, k_valid);
  };

  load_tile<D>(s_q, Q + (int64_t)q_tok0 * q_st + (int64_t)head * q_sh, q_st, q_valid);
  cp_async_commit();
  int slot = next_active(-1);
  if (slot < nslots) issue(slot, 0);
  cp_async_commit();

  // Q fragments stay in registers for the whole row
  cp_async_wait<1>();
  __syncthreads();
  uint32_t qf[D / 16][4];
#pragma unroll
  for (int kk = 0; kk < D / 16; ++kk)
    ldsm_x4(qf[kk], s_q + tile_off<D>(warp * 16 + (lane & 15), kk * 2 + (lane >> 4)));

  float o[D / 8][4];
#pragma unroll
  for (int n = 0; n < D / 8; ++n)
#pragma unroll
    for (int e = 0; e < 4; ++e) o[n][e] = 0.f;
  float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
  const int q_pos0 = q_tok0 + warp * 16 + g;         // rows g and g+8 of this warp

  int buf = 0;
  while (slot < nslots) {
    const int nxt = next_active(slot);
    if (nxt < nslots) issue(nxt, buf ^ 1);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();

    int k_tok0, k_valid;
    slot_info(slot, k_tok0, k_valid);
    const uint32_t sk = s_k0 + buf * TILE_BYTES, sv = s_v0 + buf * TILE_BYTES;

    // S = Q K^T  (16 x 64 per warp)
    float s[KT / 8][4];
#pragma unroll
    for (int n = 0; n < KT / 8; ++n)
#pragma unroll
      for (int e = 0; e < 4; ++e) s[n][e] = 0.f;
#pragma unroll
    for (int kk = 0; kk < D / 16; ++kk) {
#pragma unroll
      for (int np = 0; np < KT / 16; ++np) {
        uint32_t bf[4];
        const int mid = lane >> 3;
        ldsm_x4(bf, sk + tile_off<D>(np * 16 + (mid >> 1) * 8 + (lane & 7), kk * 2 + (mid & 1)));
        mma_bf16(s[2 * np], qf[kk], bf[0], bf[1]);
        mma_bf16(s[2 * np + 1], qf[kk], bf[2], bf[3]);
      }
    }
    // mask (only tiles that touch the diagonal or the end of the sequence)
    const bool need_mask = (k_valid < KT) || (causal && (k_tok0 + KT - 1 > q_tok0));
    if (need_mask) {
#pragma unroll
      for (int n = 0; n < KT / 8; ++n)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int kc = n * 8 + t4 * 2 + (e & 1);
          const int qp = q_pos0 + ((e & 2) ? 8 : 0);
          const bool ok = kc < k_valid && (!causal || (k_tok0 + kc) <= qp);
          if (!ok) s[n][e] = -INFINITY;
        }
    }
    // online softmax (fp32), rows g (e = 0,1) and g+8 (e = 2,3)
    float mx[2] = {-INFINITY, -INFINITY};
#pragma unroll
    for (int n = 0; n < KT / 8; ++n) {
      mx[0] = fmaxf(mx[0], fmaxf(s[n][0], s[n][1]));
      mx[1] = fmaxf(mx[1], fmaxf(s[n][2], s[n][3]));
    }
    float corr[2], m_use[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 1));
      mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 2));
      const float m_new = fmaxf(m_run[h], mx[h] * scale_log2);
      m_use[h] = (m_new == -INFINITY) ? 0.f : m_new;
      corr[h] = (m_run[h] == -INFINITY) ? 0.f : exp2f(m_run[h] - m_use[h]);
      m_run[h] = m_new;
      l_run[h] *= corr[h];
    }
    float rs[2] = {0.f, 0.f};
#pragma unroll
    for (int n = 0; n < KT / 8; ++n) {
      s[n][0] = exp2f(s[n][0] * scale_log2 - m_use[0]);
      s[n][1] = exp2f(s[n][1] * scale_log2 - m_use[0]);
      s[n][2] = exp2f(s[n][2] * scale_log2 - m_use[1]);
      s[n][3] = exp2f(s[n][3] * scale_log2 - m_use[1]);
      rs[0] += s[n][0] + s[n][1];
      rs[1] += s[n][2] + s[n][3];
    }
    l_run[0] += rs[0];
    l_run[1] += rs[1];
#pragma unroll
    for (int n = 0; n < D / 8; ++n) {
      o[n][0] *= corr[0]; o[n][1] *= corr[0];
      o[n][2] *= corr[1]; o[n][3] *= corr[1];
    }
    // O += P V
#pragma unroll
    for (int kk = 0; kk < KT / 16; ++kk) {
      uint32_t pa[4];
      pa[0] = pack_bf16(s[2 * kk][0], s[2 * kk][1]);
      pa[1] = pack_bf16(s[2 * kk][2], s[2 * kk][3]);
      pa[2] = pack_bf16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
      pa[3] = pack_bf16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
      for (int np = 0; np < D / 16; ++np) {
        uint32_t bf[4];
        const int mid = lane >> 3;
        ldsm_x4_t(bf, sv + tile_off<D>(kk * 16 + (mid & 1) * 8 + (lane & 7), np * 2 + (mid >> 1)));
        mma_bf16(o[2 * np], pa, bf[0], bf[1]);
        mma_bf16(o[2 * np + 1], pa, bf[2], bf[3]);
      }
    }
    __syncthreads();
    slot = nxt;
    buf ^= 1;
  }

  // finalise: the quad holds partial row sums
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 1);
    l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 2);
  }
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int row = warp * 16 + g + h * 8;
    if (row >= q_valid) continue;
    const float inv = l_run[h] > 0.f ? 1.f / l_run[h] : 0.f;
    const int64_t tok = q_tok0 + row;
    OutT* op = out + (tok * h_q + head) * D;
#pragma unroll
    for (int n = 0; n < D / 8; ++n) {
      const float a = o[n][2 * h] * inv, b2 = o[n][2 * h + 1] * inv;
      const int c = n * 8 + t4 * 2;
      if constexpr (sizeof(OutT) == 2) {
        *reinterpret_cast<__nv_bfloat162*>(op + c) = __floats2bfloat162_rn(a, b2);
      } else {
        *reinterpret_cast<float2*>(op + c) = make_float2(a, b2);
      }
    }
    if (lse && t4 == 0)
      lse[tok * h_q + head] = l_run[h] > 0.f ? (m_run[h] + log2f(l_run[h])) * 0.6931471805599453f : -INFINITY;
  }
}

__global__ void cast_f32_bf16_kernel(const float* __restrict__ src, __nv_bfloat16* __restrict__ dst,
                                     int64_t n8, int heads, int d, int64_t st, int64_t sh) {
  // one thread per 8 consecutive elements of a head row; dst is contiguous [tokens, heads, d]
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n8) return;
  const int ch = d / 8;
  const int64_t row = i / ch;
  const int c = (int)(i % ch);
  const int64_t tok = row / heads;
  const int hd = (int)(row % heads);
  const float* p = src + tok * st + (int64_t)hd * sh + c * 8;
  const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
  uint4 o;
  o.x = pack_bf16(a.x, a.y); o.y = pack_bf16(a.z, a.w);
  o.z = pack_bf16(b.x, b.y); o.w = pack_bf16(b.z, b.w);
  *reinterpret_cast<uint4*>(dst + i * 8) = o;
}

}  // namespace

namespace sw {

int32_t launch_cast_f32_to_bf16(const float* src, __nv_bfloat16* dst, int64_t tokens, int heads, int d,
                                int64_t stride_tok, int64_t stride_head, cudaStream_t st) {
  const int64_t n8 = tokens * heads * (d / 8);
  if (n8 == 0) return SW_OK;
  count_launch();
  cast_f32_bf16_kernel<<<(unsigned)((n8 + 255) / 256), 256, 0, st>>>(src, dst, n8, heads, d, stride_tok,
                                                                     stride_head);
  return check_launch("cast_f32_to_bf16");
}

template <int D, typename OutT>
static int32_t launch_generic_t(const AttnPrefillArgs& a, cudaStream_t st) {
  const sw_layout& L = *a.L;
  const int TPB = L.block / 64;
  const int total_slots = L.total_blocks * TPB;
  const size_t smem = 5 * 64 * D * 2;
  auto kern = attn_prefill_generic_kernel<D, OutT>;
  if (int32_t rc = allow_dynamic_smem(kern, smem, "sw_sparse_attn_prefill(generic) smem attribute")) return rc;
  dim3 grid(total_slots, a.h_q);
  const float scale_log2 = a.softmax_scale * 1.4426950408889634f;
  count_launch();
  kern<<<grid, kThreads, smem, st>>>(a.q, a.k, a.v, a.q_stride_tok, a.q_stride_head, a.k_stride_tok,
                                     a.k_stride_head, a.v_stride_tok, a.v_stride_head, a.h_q, a.h_kv,
                                     L.cu_seqlens, L.cu_blocks, L.batch, L.block, total_slots, a.idx,
                                     a.count, a.tau_max, scale_log2, (a.flags & SW_CAUSAL) ? 1 : 0,
                                     (OutT*)a.out, a.lse);
  return check_launch("sw_sparse_attn_prefill(generic)");
}

int32_t launch_attn_prefill_generic(const AttnPrefillArgs& a, cudaStream_t st) {
  if (a.L->total_blocks == 0) return SW_OK;
  if (a.d == 128 && a.out_dtype == SW_BF16) return launch_generic_t<128, __nv_bfloat16>(a, st);
  if (a.d == 128 && a.out_dtype == SW_F32) return launch_generic_t<128, float>(a, st);
  if (a.d == 64 && a.out_dtype == SW_BF16) return launch_generic_t<64, __nv_bfloat16>(a, st);
  if (a.d == 64 && a.out_dtype == SW_F32) return launch_generic_t<64, float>(a, st);
  return fail(SW_ERR_UNSUPPORTED, "sw_sparse_attn_prefill: head_dim %d", a.d);
}

}  // namespace sw
