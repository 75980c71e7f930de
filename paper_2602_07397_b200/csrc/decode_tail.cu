// sw_decode_select, third kernel: Alg. 2 Steps 4-6 on the whole row of one sequence per CTA,
// from what decode_duty.cu (the raw score row) and decode_select.cu (the partial sums of r_prev W) left in the
// workspace:
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
// three integer sums over the block in one pass (two barriers)
__device__ __forceinline__ void block_sum3_i(int& a, int& b, int& c, int (*s_red)[NT / 32]) {
  a = swd::warp_sum_i(a); b = swd::warp_sum_i(b); c = swd::warp_sum_i(c);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { s_red[0][threadIdx.x >> 5] = a; s_red[1][threadIdx.x >> 5] = b; s_red[2][threadIdx.x >> 5] = c; }
  __syncthreads();
  a = swd::warp_sum_i(s_red[0][threadIdx.x & 31]);
  b = swd::warp_sum_i(s_red[1][threadIdx.x & 31]);
  c = swd::warp_sum_i(s_red[2][threadIdx.x & 31]);
}
__device__ __forceinline__ float block_sum(float v, float* s_red) {
  v = swd::warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float m = s_red[threadIdx.x & 31];
  return swd::warp_sum(m);                           // the same order in every warp
}

__global__ void __launch_bounds__(NT, 1)
decode_tail_kernel(const Params p_in) {
  Params p = p_in;                                    // (the pointers to earlier kernels' data pass through pdl_wait)
  extern __shared__ __align__(16) float s_row[];     // [mbp]
  __shared__ float s_red[NT / 32];
  __shared__ int s_redi[3][NT / 32];
  __shared__ unsigned short s_nslot[kMaxTiles + 1];  // partials per stream tile
  __shared__ int s_first[kMaxTiles + 1];             // id of the tile's first partial (decode_select.cuh: part_id)
  __shared__ swsel::Scratch scratch;
  const int tid = threadIdx.x, seq = blockIdx.x;
  swd::pdl_launch_dependents();                       // (the attention kernel waits for this one before it reads idx)
  const bool walk = p.r_prev != nullptr, soft = p.flags & SW_SCORE_SOFTMAX;
  const int mb = p.max_blocks;

  // ---- independent of the streaming kernel: chunk prefix of this sequence, T, tau, r_prev[b_q] -------------
  int mine = 0, before = 0, tbefore = 0;
  for (int sq = tid; sq < p.batch; sq += NT) {
    const SeqInfo o = seq_info(p.seqlens, sq, p.B, mb, walk);
    const int c = o.total_chunks();
    mine += c;
    if (sq < seq) { before += c; tbefore += o.nt; }
  }
  block_sum3_i(mine, before, tbefore, s_redi);
  const int T = mine, pref = before;                  // chunks of the batch / of the sequences before this one
  const int tpref = tbefore;                          // tiles with chunks of the sequences before this one
  const int G = max(1, min(p.g_stream, T));           // CTAs of the streaming kernel that hold chunks
  const SeqInfo si = seq_info(p.seqlens, seq, p.B, mb, walk);
  const int bq = si.bq, hi = bq + 1;
  const int tt = max(0, min(__ldg(p.tau + seq), p.tau_max));   // (tau, seqlens: written before this selection started)
  // partials per stream tile = CTAs of the streaming kernel that share the tile's chunks
  for (int tl = tid; tl < p.tiles_max; tl += NT) {
    const int nch = si.chunks(tl);
    int ns = 0, first = 0;
    if (nch > 0) {
      const long long f0 = pref + si.chunks_before(tl);
      first = cta_of(f0, T, G);
      ns = cta_of(f0 + nch - 1, T, G) - first + 1;
    }
    s_nslot[tl] = (unsigned short)ns;
    s_first[tl] = part_id(first, tpref + tl);
  }
  swd::pdl_wait(p.ws_scores, p.ws_part, p.r_prev);             // the duty kernel's scores and the stream's partials are visible
  if (!seq_live(p.seqlens[seq], p.B, mb)) {
    // idle slot (length outside [1, max_blocks B]): an empty selection and a zero walk row, nothing else is touched
    for (int j = tid; j < mb; j += NT) p.r_out[(int64_t)seq * mb + j] = 0.f;
    for (int j = tid; j < p.tau_max; j += NT) p.idx[(int64_t)seq * p.tau_max + j] = -1;
    if (tid == 0) p.count[seq] = 0;
    return;
  }

  const float rq = walk ? __ldcg(p.r_prev + (int64_t)seq * mb + bq) : 1.f;   // (consumed after the softmax statistics)
  const float* sc = p.ws_scores + (int64_t)seq * p.mbp;
  float lmax = -INFINITY;
  for (int j = tid; j < hi; j += NT) { const float v = __ldcg(sc + j); s_row[j] = v; lmax = fmaxf(lmax, v); }
  float m = 0.f, inv_l = 1.f;
  if (soft) {
    // (max, then sum: merging (max, sum-of-exp) pairs in one reduction costs two expf per shuffle step and was
    // measured slower, 2.8 against 1.5 us)
    m = block_max(lmax, s_red);
    float e = 0.f;
    for (int j = tid; j < hi; j += NT) e += expf(s_row[j] - m);      // (the thread's own entries)
    inv_l = 1.f / block_sum(e, s_red);
  } else {
    __syncthreads();                                  // s_nslot
  }
  // W_new = A^s; Alg. 2 Step 4 cache update: the new row becomes row b_q of the cached W,
  // zeros right of the diagonal.  Row b_q is never read while b_q is the current block.
  // Step 5: r[j] = sum_{m < b_q} r_prev[m] W[m][j] + r_prev[b_q] w[j], the partial sums in slot order; the loads of
  // 2 columns x 8 slots are in flight per thread (a dependent load per slot cost 5 us with 256 threads).
  float* wrow = p.W + (int64_t)seq * p.w_stride_seq + (int64_t)bq * mb;
  float lamax = 0.f;
  constexpr int kCols = 2, kSl = 8;
  for (int j0 = 0; j0 < mb; j0 += kCols * NT) {
    float v[kCols];
    int ns[kCols], nsmax = 0;
    const float* pp[kCols];
#pragma unroll
    for (int c = 0; c < kCols; ++c) {
      const int j = j0 + c * NT + tid;
      v[c] = 0.f;
      const int tl = min(j, mb - 1) / kTileW;
      ns[c] = (j < hi) ? (int)s_nslot[tl] : 0;
      nsmax = max(nsmax, ns[c]);
      pp[c] = p.ws_part + (int64_t)s_first[tl] * kTileW + (j & (kTileW - 1));
    }
    nsmax = __reduce_max_sync(0xffffffffu, nsmax);
    for (int s0 = 0; s0 < nsmax; s0 += kSl) {
      float x[kSl][kCols];
#pragma unroll
      for (int e = 0; e < kSl; ++e)
#pragma unroll
        for (int c = 0; c < kCols; ++c) x[e][c] = (s0 + e < ns[c]) ? __ldcg(pp[c] + (s0 + e) * kTileW) : 0.f;
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
