// sw_sparse_attn_decode: Alg. 2 Step 7.  One query token per sequence against the
// selected blocks of its KV cache.  HBM-bound (M = h_q/h_kv <= 16 useful rows per KV head), so the
// design is about bytes in flight: the selected blocks of one (sequence, kv head) are split over
// several CTAs (split-KV), every CTA streams its 64-key K and V tiles through a multi-stage
// cp.async ring, and the tiny QK^T / PV products run on mma.sync m16n8k16 with the GQA group in
// the M dimension.  Partial (O, m, l) per split are merged by log-sum-exp in a second kernel.
#include "common.cuh"
#include "mma_sync.cuh"

namespace {

using namespace swmma;

constexpr int kThreads = 128;       // 4 warps, each owns 16 keys of every 64-key tile
constexpr int KT = 64;
constexpr int kStages = 3;


// Partial results: Opart [batch, h_q, nsplit, D] fp32 (unnormalised), ML [batch, h_q, nsplit, 2]
template <int D>
__global__ void __launch_bounds__(kThreads)
attn_decode_kernel(const __nv_bfloat16* Q, int64_t q_sb, int64_t q_sh, const __nv_bfloat16* Kc, const __nv_bfloat16* Vc,
                   int64_t kv_sb, int64_t k_st, int64_t k_sh, int64_t v_st, int64_t v_sh, int h_q, int h_kv,
                   const int32_t* seqlens, int B, const int32_t* idx, const int32_t* count, int tau_max,
                   float scale_log2, int nsplit, const int32_t* table, int table_stride,
                   float* __restrict__ Opart, float* __restrict__ ML) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  constexpr int TILE_BYTES = KT * D * 2;
  constexpr int CH = D / 8;
  const uint32_t s_base = smem_u32(smem_raw);            // [kStages][K tile | V tile]
  const int split = blockIdx.x, kvh = blockIdx.y, seq = blockIdx.z;
  const int grp = h_q / h_kv;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t4 = lane & 3;
  swd::pdl_launch_dependents();                          // (the merge kernel may take its place on the SMs early)
  // the block lists of the selection before this kernel (and whatever else earlier kernels of the stream wrote):
  // no load through these pointers may be scheduled above the wait (common.cuh: pdl_wait)
  swd::pdl_wait(Q, Kc, Vc, seqlens, idx, count, table);
  const int t = seqlens[seq];                            // (plain loads, not __ldg: see pdl_wait)
  const int cnt = count[seq];
  const int32_t* list = idx + (int64_t)seq * tau_max;
  const int TPB = B / KT;
  const int per = (cnt + nsplit - 1) / nsplit;            // selected blocks per split
  const int blk_lo = split * per, blk_hi = min(cnt, blk_lo + per);
  const int nslots = max(0, blk_hi - blk_lo) * TPB;
  // contiguous cache: sequence s at + s * kv_sb; paged cache (table != NULL): one pool of pages of B
  // tokens, logical block j of sequence s lives in page table[s * table_stride + j]
  const __nv_bfloat16* Kb = Kc + (table ? 0 : (int64_t)seq * kv_sb) + (int64_t)kvh * k_sh;
  const __nv_bfloat16* Vb = Vc + (table ? 0 : (int64_t)seq * kv_sb) + (int64_t)kvh * v_sh;
  const int32_t* pages = table ? table + (int64_t)seq * table_stride : nullptr;

  // k_tok0: token offset of the tile in memory; k_valid: keys of it that exist (logical position < t)
  auto slot_info = [&](int slot, int& k_tok0, int& k_valid) {
    const int j = list[blk_lo + slot / TPB];             // (L1-cached after the first touch)
    const int off = (slot % TPB) * KT;
    k_valid = max(0, min(KT, t - (j * B + off)));
    k_tok0 = (pages ? pages[j] : j) * B + off;
  };
  auto issue = [&](int slot, int stage) {
    int k_tok0, k_valid;
    slot_info(slot, k_tok0, k_valid);
    const uint32_t sk = s_base + stage * 2 * TILE_BYTES, sv = sk + TILE_BYTES;
    for (int i = tid; i < KT * CH; i += kThreads) {
      const int row = i / CH, ch = i % CH;
      const bool ok = row < k_valid;
      const int64_t tok = ok ? (k_tok0 + row) : 0;
      cp_async16(sk + tile_off<D>(row, ch), Kb + tok * k_st + ch * 8, ok);
      cp_async16(sv + tile_off<D>(row, ch), Vb + tok * v_st + ch * 8, ok);
    }
  };

  // prologue: fill kStages-1 stages
#pragma unroll
  for (int s = 0; s < kStages - 1; ++s) {
    if (s < nslots) issue(s, s);
    cp_async_commit();
  }

  // Q fragments: rows = heads of the GQA group (row g -> a0/a2, row g+8 -> a1/a3)
  uint32_t qf[D / 16][4];
  {
    const __nv_bfloat16* qb = Q + (int64_t)seq * q_sb + (int64_t)(kvh * grp) * q_sh;
#pragma unroll
    for (int kk = 0; kk < D / 16; ++kk) {
      const int c = kk * 16 + t4 * 2;
      qf[kk][0] = (g < grp) ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)g * q_sh + c) : 0u;
      qf[kk][1] = (g + 8 < grp) ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)(g + 8) * q_sh + c) : 0u;
      qf[kk][2] = (g < grp) ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)g * q_sh + c + 8) : 0u;
      qf[kk][3] = (g + 8 < grp) ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)(g + 8) * q_sh + c + 8) : 0u;
    }
  }

  float o[D / 8][4];
#pragma unroll
  for (int n = 0; n < D / 8; ++n)
#pragma unroll
    for (int e = 0; e < 4; ++e) o[n][e] = 0.f;
  float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};

  for (int slot = 0; slot < nslots; ++slot) {
    const int stage = slot % kStages;
    if (slot + kStages - 1 < nslots) issue(slot + kStages - 1, (slot + kStages - 1) % kStages);
    cp_async_commit();
    cp_async_wait<kStages - 1>();
    __syncthreads();
    int k_tok0, k_valid;
    slot_info(slot, k_tok0, k_valid);
    const uint32_t sk = s_base + stage * 2 * TILE_BYTES, sv = sk + TILE_BYTES;
    const int key0 = warp * 16;                       // this warp's 16 keys inside the tile
    if (key0 < k_valid) {
      float s[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
      for (int kk = 0; kk < D / 16; ++kk) {
        uint32_t bf[4];
        const int mid = lane >> 3;
        ldsm_x4(bf, sk + tile_off<D>(key0 + (mid >> 1) * 8 + (lane & 7), kk * 2 + (mid & 1)));
        mma_bf16(s[0], qf[kk], bf[0], bf[1]);
        mma_bf16(s[1], qf[kk], bf[2], bf[3]);
      }
      if (key0 + 16 > k_valid) {
#pragma unroll
        for (int n = 0; n < 2; ++n)
#pragma unroll
          for (int e = 0; e < 4; ++e)
            if (key0 + n * 8 + t4 * 2 + (e & 1) >= k_valid) s[n][e] = -INFINITY;
      }
      float corr[2], m_use[2];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        float mx = fmaxf(fmaxf(s[0][2 * h], s[0][2 * h + 1]), fmaxf(s[1][2 * h], s[1][2 * h + 1]));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
        const float m_new = fmaxf(m_run[h], mx * scale_log2);
        m_use[h] = (m_new == -INFINITY) ? 0.f : m_new;
        corr[h] = (m_run[h] == -INFINITY) ? 0.f : exp2f(m_run[h] - m_use[h]);
        m_run[h] = m_new;
        l_run[h] *= corr[h];
      }
#pragma unroll
      for (int n = 0; n < 2; ++n) {
        s[n][0] = exp2f(s[n][0] * scale_log2 - m_use[0]);
        s[n][1] = exp2f(s[n][1] * scale_log2 - m_use[0]);
        s[n][2] = exp2f(s[n][2] * scale_log2 - m_use[1]);
        s[n][3] = exp2f(s[n][3] * scale_log2 - m_use[1]);
        l_run[0] += s[n][0] + s[n][1];
        l_run[1] += s[n][2] + s[n][3];
      }
#pragma unroll
      for (int n = 0; n < D / 8; ++n) {
        o[n][0] *= corr[0]; o[n][1] *= corr[0];
        o[n][2] *= corr[1]; o[n][3] *= corr[1];
      }
      uint32_t pa[4];
      pa[0] = pack_bf16(s[0][0], s[0][1]);
      pa[1] = pack_bf16(s[0][2], s[0][3]);
      pa[2] = pack_bf16(s[1][0], s[1][1]);
      pa[3] = pack_bf16(s[1][2], s[1][3]);
#pragma unroll
      for (int np = 0; np < D / 16; ++np) {
        uint32_t bf[4];
        const int mid = lane >> 3;
        ldsm_x4_t(bf, sv + tile_off<D>(key0 + (mid & 1) * 8 + (lane & 7), np * 2 + (mid >> 1)));
        mma_bf16(o[2 * np], pa, bf[0], bf[1]);
        mma_bf16(o[2 * np + 1], pa, bf[2], bf[3]);
      }
    }
    __syncthreads();
  }
  cp_async_wait<0>();

  // merge the 4 warps (disjoint key subsets) through shared memory, then write the split partial
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 1);
    l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 2);
  }
  __syncthreads();
  float* s_o = reinterpret_cast<float*>(smem_raw);              // [4 warps][16 rows][D]
  float* s_ml = s_o + 4 * 16 * D;                               // [4][16][2]
#pragma unroll
  for (int n = 0; n < D / 8; ++n) {
    const int c = n * 8 + t4 * 2;
    s_o[(warp * 16 + g) * D + c] = o[n][0];
    s_o[(warp * 16 + g) * D + c + 1] = o[n][1];
    s_o[(warp * 16 + g + 8) * D + c] = o[n][2];
    s_o[(warp * 16 + g + 8) * D + c + 1] = o[n][3];
  }
  if (t4 == 0) {
    s_ml[((warp * 16 + g) * 2)] = m_run[0];
    s_ml[((warp * 16 + g) * 2) + 1] = l_run[0];
    s_ml[((warp * 16 + g + 8) * 2)] = m_run[1];
    s_ml[((warp * 16 + g + 8) * 2) + 1] = l_run[1];
  }
  __syncthreads();
  for (int i = tid; i < grp * D; i += kThreads) {
    const int row = i / D, c = i % D;
    float m = -INFINITY;
#pragma unroll
    for (int w = 0; w < 4; ++w) m = fmaxf(m, s_ml[(w * 16 + row) * 2]);
    float acc = 0.f, l = 0.f;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const float mw = s_ml[(w * 16 + row) * 2];
      const float f = (mw == -INFINITY) ? 0.f : exp2f(mw - m);
      acc += f * s_o[(w * 16 + row) * D + c];
      l += f * s_ml[(w * 16 + row) * 2 + 1];
    }
    const int head = kvh * grp + row;
    const int64_t pidx = ((int64_t)seq * h_q + head) * nsplit + split;
    Opart[pidx * D + c] = acc;
    if (c == 0) { ML[pidx * 2] = m; ML[pidx * 2 + 1] = l; }
  }
}

template <int D>
__global__ void __launch_bounds__(D)
attn_decode_merge_kernel(const float* Opart, const float* ML, int nsplit, __nv_bfloat16* __restrict__ out,
                         float* __restrict__ lse) {
  const int64_t bh = blockIdx.x;                      // seq * h_q + head
  const int c = threadIdx.x;
  swd::pdl_launch_dependents();                       // the next kernel of the layer loop may start its prologue
  swd::pdl_wait(Opart, ML);                           // the split-KV partials
  float m = -INFINITY;
  for (int s = 0; s < nsplit; ++s) m = fmaxf(m, ML[(bh * nsplit + s) * 2]);
  float acc = 0.f, l = 0.f;
  for (int s = 0; s < nsplit; ++s) {
    const float ms = ML[(bh * nsplit + s) * 2];
    const float f = (ms == -INFINITY) ? 0.f : exp2f(ms - m);
    acc += f * Opart[(bh * nsplit + s) * D + c];
    l += f * ML[(bh * nsplit + s) * 2 + 1];
  }
  out[bh * D + c] = __float2bfloat16(l > 0.f ? acc / l : 0.f);
  if (lse && c == 0) lse[bh] = l > 0.f ? (m + log2f(l)) * 0.6931471805599453f : -INFINITY;
}

}  // namespace

namespace sw {

int decode_num_splits(int batch, int h_kv, int tau_max, int d) {
  // Split-KV factor.  The grid (batch * h_kv * ns CTAs) runs in waves of slots = (CTAs resident per
  // SM) * (SMs); a wave that is mostly empty costs as much as a full one, so pick the ns that
  // minimises  waves * ceil(tau_max / ns)  (time in key blocks per CTA slot), with a 1 % penalty per
  // split for the merge pass.
  const int base = batch * h_kv;
  if (base <= 0 || tau_max <= 0) return 1;
  const int ring = kStages * 2 * KT * d * 2;                   // bytes of shared memory per CTA
  int occ = (227 * 1024) / (ring + 1024);
  if (occ < 1) occ = 1;
  if (occ > 8) occ = 8;
  const int slots = occ * num_sms();
  const int ns_max = tau_max < 64 ? tau_max : 64;
  int best = 1;
  double best_cost = 1e30;
  for (int ns = 1; ns <= ns_max; ++ns) {
    const int waves = (base * ns + slots - 1) / slots;
    const int blocks = (tau_max + ns - 1) / ns;
    const double cost = (double)waves * (blocks + 1) * (1.0 + 0.01 * ns);
    if (cost < best_cost) { best_cost = cost; best = ns; }
  }
  return best;
}

size_t decode_ws_bytes(int batch, int h_q, int d, int nsplit) {
  return (size_t)batch * h_q * nsplit * (d + 2) * sizeof(float);
}

template <int D>
static int32_t launch_decode_t(int batch, int block, const sw_tensor& q, const sw_tensor& kc,
                               const sw_tensor& vc, int64_t stride_batch, const int32_t* seqlens,
                               const int32_t* idx, const int32_t* count, int tau_max, float softmax_scale,
                               void* out, float* lse, void* ws, int nsplit, const int32_t* table,
                               int table_stride, cudaStream_t st) {
  const size_t ring = (size_t)kStages * 2 * KT * D * 2;
  const size_t merge = (size_t)(4 * 16 * D + 4 * 16 * 2) * sizeof(float);
  const size_t smem = ring > merge ? ring : merge;
  if (int32_t rc = allow_dynamic_smem(attn_decode_kernel<D>, smem, "sw_sparse_attn_decode smem attribute")) return rc;
  float* Opart = reinterpret_cast<float*>(ws);
  float* ML = Opart + (size_t)batch * q.heads * nsplit * D;
  dim3 grid(nsplit, kc.heads, batch);
  launch_pdl(attn_decode_kernel<D>, grid, dim3(kThreads), smem, st,
      (const __nv_bfloat16*)q.ptr, q.stride_tok, q.stride_head, (const __nv_bfloat16*)kc.ptr,
      (const __nv_bfloat16*)vc.ptr, stride_batch, kc.stride_tok, kc.stride_head, vc.stride_tok,
      vc.stride_head, q.heads, kc.heads, seqlens, block, idx, count, tau_max,
      softmax_scale * 1.4426950408889634f, nsplit, table, table_stride, Opart, ML);
  count_launch(2);
  launch_pdl(attn_decode_merge_kernel<D>, dim3(batch * q.heads), dim3(D), 0, st, (const float*)Opart, (const float*)ML, nsplit,
             (__nv_bfloat16*)out, lse);
  return check_launch("sw_sparse_attn_decode");
}

int32_t launch_attn_decode(int batch, int block, const sw_tensor& q, const sw_tensor& kc,
                           const sw_tensor& vc, int64_t stride_batch, const int32_t* seqlens,
                           const int32_t* idx, const int32_t* count, int tau_max, float softmax_scale,
                           void* out, float* lse, void* ws, size_t ws_bytes, const int32_t* table,
                           int table_stride, cudaStream_t st) {
  if (batch == 0) return SW_OK;
  const int nsplit = decode_num_splits(batch, kc.heads, tau_max, q.d);
  if (ws == nullptr || ws_bytes < decode_ws_bytes(batch, q.heads, q.d, nsplit))
    return fail(SW_ERR_WORKSPACE, "sw_sparse_attn_decode: workspace %zu < %zu bytes", ws_bytes,
                decode_ws_bytes(batch, q.heads, q.d, nsplit));
  if (q.d == 128)
    return launch_decode_t<128>(batch, block, q, kc, vc, stride_batch, seqlens, idx, count, tau_max,
                                softmax_scale, out, lse, ws, nsplit, table, table_stride, st);
  if (q.d == 64)
    return launch_decode_t<64>(batch, block, q, kc, vc, stride_batch, seqlens, idx, count, tau_max,
                               softmax_scale, out, lse, ws, nsplit, table, table_stride, st);
  return fail(SW_ERR_UNSUPPORTED, "sw_sparse_attn_decode: head_dim %d", q.d);
}

}  // namespace sw
