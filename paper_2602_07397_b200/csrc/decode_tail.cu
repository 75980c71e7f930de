// sw_decode_select, second kernel: Alg. 2 Steps 4-6 on the whole row of one sequence per CTA,
// from what decode_select.cu left in the workspace (the raw score row and the partial sums of r_prev W):
//   A_new = softmax of the score row (P5), W_new = A_new^s, stored as row b_q of the cached W (Step 4);
//   r = sum of the partials (slot order: deterministic) + r_prev[b_q] W_new (Step 5); r_out = r / max|r| (P9);
//   S = TopK(r_out[0..b_q), tau - |forced|) U {b_q} (U {0}) (Step 6; select.cuh, bit-exact given r_out).
// 1024 threads: the row passes and the radix select are chains of block-wide steps, bound by the dependent
// issue latency of each warp -- 32 warps with 2 keys each run them several times faster than 8 warps with 8.
// Launched as a programmatic dependent of the streaming kernel: everything up to griddepcontrol.wait (the chunk
// prefix of the batch, tau, r_prev[b_q]) runs while the streaming kernel's last CTAs drain.
#define SWSEL_THREADS 1024
#include "decode_select.cuh"
#include "select.cuh"

namespace {

using namespace swds;
constexpr int NT = kTailThreads;
static_assert(NT == swsel::kThreads, "select.cuh is compiled for the tail's thread count");

__device__ __forceinline__ float block_max(float v, float* s_red) {
  v = swd::warp_max(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float m = s_red[threadIdx.x & 31];                 // NT / 32 = 32 partial results
  return swd::warp_max(m);
}
__device__ __forceinline__ float block_sum(float v, float* s_red) {
  v = swd::warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float m = s_red[threadIdx.x & 31];
  return swd::warp_sum(m);                           // the same order in every warp
}
__device__ __forceinline__ int block_sum_i(int v, int* s_red) {
  v = swd::warp_sum_i(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  return swd::warp_sum_i(s_red[threadIdx.x & 31]);
}

__global__ void __launch_bounds__(NT, 1)
decode_tail_kernel(const Params p) {
  extern __shared__ __align__(16) float s_row[];     // [mbp]
  __shared__ float s_red[NT / 32];
  __shared__ int s_redi[NT / 32];
  __shared__ unsigned char s_nslot[kMaxTiles + 1];   // partials per column tile
  __shared__ swsel::Scratch scratch;
  const int tid = threadIdx.x, seq = blockIdx.x;
  swd::pdl_launch_dependents();                       // (the attention kernel waits for this one before it reads idx)
  const bool walk = p.r_prev != nullptr, soft = p.flags & SW_SCORE_SOFTMAX;
  const int mb = p.max_blocks;

  // ---- independent of the streaming kernel: chunk prefix of this sequence, T, tau, r_prev[b_q] -------------
  int mine = 0, before = 0;
  for (int sq = tid; sq < p.batch; sq += NT) {
    const int c = seq_info(p.seqlens, sq, p.B).total_chunks(walk);
    mine += c;
    if (sq < seq) before += c;
  }
  const int T = block_sum_i(mine, s_redi);
  const int pref = block_sum_i(before, s_redi);
  const int G = max(1, min(p.g_stream, T));           // CTAs of the streaming kernel that hold chunks
  const SeqInfo si = seq_info(p.seqlens, seq, p.B);
  const int bq = si.bq, hi = bq + 1;
  const int tt = max(0, min(__ldg(p.tau + seq), p.tau_max));
  const float rq = walk ? __ldg(p.r_prev + (int64_t)seq * mb + bq) : 1.f;
  // partials per column tile = CTAs of the streaming kernel that share the tile's chunks
  for (int tl = tid; tl <= si.a; tl += NT) {
    const int nch = si.chunks(tl, walk);
    int ns = 0;
    if (nch > 0) {
      const long long f0 = pref + si.chunks_before(tl, walk);
      ns = cta_of(f0 + nch - 1, T, G) - cta_of(f0, T, G) + 1;
    }
    s_nslot[tl] = (unsigned char)min(ns, 255);
  }
  swd::pdl_wait();                                    // the streaming kernel's scores and partials are visible

  const float* sc = p.ws_scores + (int64_t)seq * p.mbp;
  float lmax = -INFINITY;
  for (int j = tid; j < hi; j += NT) { const float v = __ldcg(sc + j); s_row[j] = v; lmax = fmaxf(lmax, v); }
  float m = 0.f, inv_l = 1.f;
  if (soft) {
    m = block_max(lmax, s_red);
    float e = 0.f;
    for (int j = tid; j < hi; j += NT) e += expf(s_row[j] - m);
    inv_l = 1.f / block_sum(e, s_red);
  } else {
    __syncthreads();                                  // s_nslot
  }
  // W_new = A^s; Alg. 2 Step 4 cache update: the new row becomes row b_q of the cached W,
  // zeros right of the diagonal.  Row b_q is never read while b_q is the current block.
  // Step 5: r[j] = sum_{m < b_q} r_prev[m] W[m][j] + r_prev[b_q] w[j], the partial sums in slot order; the loads of
  // 2 columns x 4 slots are in flight per thread (a dependent load per slot cost 5 us with 256 threads).
  float* wrow = p.W + (int64_t)seq * p.w_stride_seq + (int64_t)bq * mb;
  float lamax = 0.f;
  constexpr int kCols = 2, kSl = 4;
  for (int j0 = 0; j0 < mb; j0 += kCols * NT) {
    float v[kCols];
    int ns[kCols], nsmax = 0;
    const float* pp[kCols];
#pragma unroll
    for (int c = 0; c < kCols; ++c) {
      const int j = j0 + c * NT + tid;
      v[c] = 0.f;
      ns[c] = (j < hi) ? (int)s_nslot[j / kTile] : 0;
      nsmax = max(nsmax, ns[c]);
      pp[c] = p.ws_part + (((int64_t)seq * p.tiles_max + min(j, mb - 1) / kTile) * p.slots) * kTile + (j & (kTile - 1));
    }
    nsmax = __reduce_max_sync(0xffffffffu, nsmax);
    for (int s0 = 0; s0 < nsmax; s0 += kSl) {
      float x[kSl][kCols];
#pragma unroll
      for (int e = 0; e < kSl; ++e)
#pragma unroll
        for (int c = 0; c < kCols; ++c) x[e][c] = (s0 + e < ns[c]) ? __ldcg(pp[c] + (s0 + e) * kTile) : 0.f;
#pragma unroll
      for (int e = 0; e < kSl; ++e)
#pragma unroll
        for (int c = 0; c < kCols; ++c) v[c] += x[e][c];                     // slot order
    }
#pragma unroll
    for (int c = 0; c < kCols; ++c) {
      const int j = j0 + c * NT + tid;
      if (j < mb) {
        float w = 0.f;
        if (j < hi) {
          const float sj = s_row[j];
          w = swd::powi(soft ? expf(sj - m) * inv_l : sj, p.s);
          const float r = fmaf(rq, w, v[c]);
          s_row[j] = r;
          lamax = fmaxf(lamax, fabsf(r));
        }
        wrow[j] = w;
      }
    }
  }
  const float amax = block_max(lamax, s_red);         // (its barriers also publish s_row)
  const bool rescale = (p.flags & SW_ROWNORM) && amax > 0.f;
  float* ro = p.r_out + (int64_t)seq * mb;
  for (int j = tid; j < mb; j += NT) {
    float v = 0.f;
    if (j < hi) { v = rescale ? s_row[j] / amax : s_row[j]; s_row[j] = v; }   // the selection reads r_out's values
    ro[j] = v;
  }
  __syncthreads();
  // Step 6: S = TopK(r[0..b_q), tau - |forced|) U {b_q} (U {0})
  swsel::RowJob J = swsel::make_job(hi, bq, true, p.flags & SW_FORCE_FIRST, tt);
  const float* row = s_row;
  swsel::select_row([row](int j) { return row[j]; }, J, p.idx + (int64_t)seq * p.tau_max, p.tau_max, p.count + seq,
                    scratch);
}

}  // namespace

namespace sw {

int32_t launch_decode_tail(const swds::Params& p, cudaStream_t st) {
  const size_t smem = sizeof(float) * (size_t)p.mbp;
  if (int32_t rc = allow_dynamic_smem(decode_tail_kernel, smem, "sw_decode_select(tail) smem attribute")) return rc;
  count_launch();
  launch_pdl(decode_tail_kernel, dim3(p.batch), dim3(NT), smem, st, p);
  return check_launch("sw_decode_select(tail)");
}

}  // namespace sw
