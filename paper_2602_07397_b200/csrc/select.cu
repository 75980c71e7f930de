// sw_select_topk: Alg. 1 Step 7 / Alg. 2 Step 6.
// One CTA per query block row: forced blocks (diagonal first, then block 0; P7) + an exact
// radix select of the top-(budget - |forced|) remaining candidates on an order-preserving
// uint32 image of the fp32 scores, ties broken by the lower index (P8), then an ordered
// compaction that emits the chosen indices ascending (select.cuh).  Integer work: bit-exact.
#include "common.cuh"
#include "select.cuh"

namespace {

using namespace swsel;

__global__ void __launch_bounds__(kThreads)
select_topk_kernel(const float* __restrict__ R, const int32_t* __restrict__ cu_blocks,
                   const int64_t* __restrict__ cu_sq, int batch, const int32_t* __restrict__ tau,
                   int tau_max, uint32_t flags, int32_t* __restrict__ idx, int32_t* __restrict__ count) {
  const int gb = blockIdx.x;
  const int seq = swd::find_seq(cu_blocks, batch, gb);
  const int blk0 = __ldg(cu_blocks + seq);
  const int b = __ldg(cu_blocks + seq + 1) - blk0;
  const int i = gb - blk0;
  const float* row = R + __ldg(cu_sq + seq) + (int64_t)i * b;
  const int n_cand = (flags & SW_CAUSAL) ? i + 1 : b;
  const int t = max(0, min(__ldg(tau + seq), tau_max));
  __shared__ Scratch scratch;
  RowJob J = make_job(n_cand, i, flags & SW_FORCE_LAST, flags & SW_FORCE_FIRST, t);
  select_row([row](int j) { return __ldg(row + j); }, J, idx + (int64_t)gb * tau_max, tau_max, count + gb, scratch);
}

// Fused form: the per-row max-abs rescale of the walk (P9; selection-invariant) and the
// top-tau of the same row in one launch, in place on the raw product the walk GEMM left in R.  The row is read
// from HBM / L2 once (max-abs), rewritten rescaled -- with zeros right of the diagonal under SW_CAUSAL, which
// the GEMM then does not have to write -- and selected from while it is hot in L1.
__global__ void __launch_bounds__(kThreads)
rescale_select_kernel(float* R, const int32_t* __restrict__ cu_blocks, const int64_t* __restrict__ cu_sq, int batch,
                      const int32_t* __restrict__ tau, int tau_max, uint32_t flags, int32_t* __restrict__ idx,
                      int32_t* __restrict__ count) {
  __shared__ float s_red[kWarps];
  __shared__ Scratch scratch;
  const int gb = blockIdx.x, tid = threadIdx.x;
  const int seq = swd::find_seq(cu_blocks, batch, gb);
  const int blk0 = __ldg(cu_blocks + seq);
  const int b = __ldg(cu_blocks + seq + 1) - blk0;
  const int i = gb - blk0;
  float* row = R + __ldg(cu_sq + seq) + (int64_t)i * b;
  const int n_cand = (flags & SW_CAUSAL) ? i + 1 : b;
  const int t = max(0, min(__ldg(tau + seq), tau_max));
  if (flags & SW_ROWNORM) {
    float m = 0.f;
    for (int j = tid; j < n_cand; j += kThreads) m = fmaxf(m, fabsf(row[j]));
    m = swd::warp_max(m);
    if ((tid & 31) == 0) s_red[tid >> 5] = m;
    __syncthreads();
    m = s_red[0];
#pragma unroll
    for (int w = 1; w < kWarps; ++w) m = fmaxf(m, s_red[w]);
    if (m > 0.f)                                     // all-zero row: untouched (P9)
      for (int j = tid; j < n_cand; j += kThreads) row[j] = row[j] / m;
  }
  for (int j = n_cand + tid; j < b; j += kThreads) row[j] = 0.f;
  __syncthreads();                                   // the rescaled row is visible to the whole CTA
  RowJob J = make_job(n_cand, i, flags & SW_FORCE_LAST, flags & SW_FORCE_FIRST, t);
  const float* crow = row;
  select_row([crow](int j) { return crow[j]; }, J, idx + (int64_t)gb * tau_max, tau_max, count + gb, scratch);
}

__global__ void __launch_bounds__(kThreads)
select_topk_row_kernel(const float* __restrict__ r, const int32_t* __restrict__ seqlens, int B,
                       int max_blocks, const int32_t* __restrict__ tau, int tau_max, uint32_t flags,
                       int32_t* __restrict__ idx, int32_t* __restrict__ count) {
  const int seq = blockIdx.x;
  const int t = __ldg(seqlens + seq);
  const int bq = (t - 1) / B;
  const int nb = (t + B - 1) / B;
  const int n_cand = (flags & SW_CAUSAL) ? bq + 1 : nb;
  const int tt = max(0, min(__ldg(tau + seq), tau_max));
  // the current block is always kept, block 0 with SW_FORCE_FIRST
  __shared__ Scratch scratch;
  const float* row = r + (int64_t)seq * max_blocks;
  RowJob J = make_job(n_cand, bq, true, flags & SW_FORCE_FIRST, tt);
  select_row([row](int j) { return __ldg(row + j); }, J, idx + (int64_t)seq * tau_max, tau_max, count + seq, scratch);
}

}  // namespace

namespace sw {

int32_t launch_select(const sw_layout& L, const float* R, const int32_t* tau, int tau_max,
                      uint32_t flags, int32_t* idx, int32_t* count, cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  count_launch();
  select_topk_kernel<<<L.total_blocks, kThreads, 0, st>>>(R, L.cu_blocks, L.cu_sq, L.batch, tau, tau_max,
                                                          flags, idx, count);
  return check_launch("sw_select_topk");
}

int32_t launch_rescale_select(const sw_layout& L, float* R, const int32_t* tau, int tau_max, uint32_t flags,
                              int32_t* idx, int32_t* count, cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  count_launch();
  rescale_select_kernel<<<L.total_blocks, kThreads, 0, st>>>(R, L.cu_blocks, L.cu_sq, L.batch, tau, tau_max, flags,
                                                             idx, count);
  return check_launch("sw_prefill_select(rescale + select)");
}

int32_t launch_select_row(int batch, int block, int max_blocks, const float* r, const int32_t* seqlens,
                          const int32_t* tau, int tau_max, uint32_t flags, int32_t* idx, int32_t* count,
                          cudaStream_t st) {
  if (batch == 0) return SW_OK;
  count_launch();
  select_topk_row_kernel<<<batch, kThreads, 0, st>>>(r, seqlens, block, max_blocks, tau, tau_max, flags,
                                                     idx, count);
  return check_launch("sw_select_topk_row");
}

}  // namespace sw
