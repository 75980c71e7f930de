// sw_select_topk: Alg. 1 Step 7 / Alg. 2 Step 6.
// One CTA per query block row: forced blocks (diagonal first, then block 0; P7) + an exact
// radix select of the top-(budget - |forced|) remaining candidates on an order-preserving
// uint32 image of the fp32 scores, ties broken by the lower index (P8), then an ordered
// compaction that emits the chosen indices ascending.  Integer work throughout: bit-exact.
#include "common.cuh"

namespace {

constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;

// fp32 -> uint32 whose unsigned order equals the float order; NaN ranks as -inf (P8)
__device__ __forceinline__ uint32_t order_key(float v) {
  if (v != v) v = -INFINITY;
  if (v == 0.f) v = 0.f;               // -0 and +0 compare equal
  uint32_t u = __float_as_uint(v);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

struct RowJob {
  const float* row;      // scores of this query block
  int n_cand;            // candidates are [0, n_cand)
  int f0, f1;            // forced indices (-1 = none), already inside [0, n_cand), f0 != f1
  int need;              // how many non-forced candidates to pick
  int budget;            // total selected
};

__device__ __forceinline__ bool is_forced(const RowJob& J, int j) { return j == J.f0 || j == J.f1; }

// Exact threshold: after the 4 passes `prefix` is the key of the need-th largest non-forced
// candidate and `n_gt` the number of candidates with a strictly larger key.
__device__ void radix_threshold(const RowJob& J, uint32_t* s_hist, uint32_t* s_bcast,
                                uint32_t& prefix_out, int& n_gt_out) {
  const int tid = threadIdx.x;
  uint32_t prefix = 0;
  int remaining = J.need;      // rank (1-based, from the top) still to locate inside the prefix bucket
  int n_gt = 0;
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    for (int i = tid; i < 256; i += kThreads) s_hist[i] = 0;
    __syncthreads();
    const uint32_t mask_hi = (pass == 0) ? 0u : (0xffffffffu << (shift + 8));
    for (int j = tid; j < J.n_cand; j += kThreads) {
      if (is_forced(J, j)) continue;
      uint32_t k = order_key(J.row[j]);
      if ((k & mask_hi) == prefix) atomicAdd(&s_hist[(k >> shift) & 0xffu], 1u);
    }
    __syncthreads();
    if (tid == 0) {
      int cum = 0, bin = 255;
      for (; bin >= 0; --bin) {
        int c = (int)s_hist[bin];
        if (cum + c >= remaining) break;
        cum += c;
      }
      s_bcast[0] = (uint32_t)bin;
      s_bcast[1] = (uint32_t)cum;
    }
    __syncthreads();
    const uint32_t bin = s_bcast[0];
    const int cum = (int)s_bcast[1];
    prefix |= bin << shift;
    n_gt += cum;
    remaining -= cum;
    __syncthreads();
  }
  prefix_out = prefix;
  n_gt_out = n_gt;
}

__device__ void select_row(const RowJob& J, int32_t* __restrict__ out, int tau_max, int32_t* count_out) {
  __shared__ uint32_t s_hist[256];
  __shared__ uint32_t s_bcast[2];
  __shared__ int s_wsel[kWarps], s_weq[kWarps];
  __shared__ int s_base_sel, s_base_eq;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  uint32_t thr = 0;
  int n_gt = 0;
  const int n_free = J.n_cand - (J.f0 >= 0) - (J.f1 >= 0);
  const bool take_all = J.need >= n_free;
  if (!take_all && J.need > 0) radix_threshold(J, s_hist, s_bcast, thr, n_gt);
  const int eq_quota = J.need - n_gt;       // equal-key candidates to take, lowest index first

  if (tid == 0) { s_base_sel = 0; s_base_eq = 0; }
  __syncthreads();
  for (int j0 = 0; j0 < J.n_cand; j0 += kThreads) {
    const int j = j0 + tid;
    bool forced = false, gt = false, eq = false;
    if (j < J.n_cand) {
      forced = is_forced(J, j);
      if (!forced) {
        if (take_all) gt = true;
        else if (J.need > 0) {
          uint32_t k = order_key(J.row[j]);
          gt = k > thr;
          eq = k == thr;
        }
      }
    }
    // rank among equals (index order) decides which equals are taken
    const uint32_t eq_ballot = __ballot_sync(0xffffffffu, eq);
    const int eq_before_lane = __popc(eq_ballot & ((1u << lane) - 1u));
    if (lane == 0) s_weq[warp] = __popc(eq_ballot);
    __syncthreads();
    int eq_before = s_base_eq + eq_before_lane;
    for (int w = 0; w < warp; ++w) eq_before += s_weq[w];
    const bool sel = forced || gt || (eq && eq_before < eq_quota);
    const uint32_t sel_ballot = __ballot_sync(0xffffffffu, sel);
    const int sel_before_lane = __popc(sel_ballot & ((1u << lane) - 1u));
    if (lane == 0) s_wsel[warp] = __popc(sel_ballot);
    __syncthreads();
    int pos = s_base_sel + sel_before_lane;
    for (int w = 0; w < warp; ++w) pos += s_wsel[w];
    if (sel && pos < tau_max) out[pos] = j;
    __syncthreads();
    if (tid == 0) {
      int a = 0, e = 0;
      for (int w = 0; w < kWarps; ++w) { a += s_wsel[w]; e += s_weq[w]; }
      s_base_sel += a;
      s_base_eq += e;
    }
    __syncthreads();
  }
  for (int p = J.budget + tid; p < tau_max; p += kThreads) out[p] = -1;
  if (tid == 0) *count_out = J.budget;
}

__device__ __forceinline__ RowJob make_job(const float* row, int n_cand, int diag, bool force_last,
                                           bool force_first, int tau) {
  RowJob J;
  J.row = row;
  J.n_cand = n_cand;
  J.budget = min(tau, n_cand);
  J.f0 = -1; J.f1 = -1;
  int nf = 0;
  if (force_last && diag >= 0 && diag < n_cand && nf < J.budget) { J.f0 = diag; ++nf; }
  if (force_first && n_cand > 0 && 0 != J.f0 && nf < J.budget) { J.f1 = 0; ++nf; }
  J.need = J.budget - nf;
  return J;
}

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
  RowJob J = make_job(row, n_cand, i, flags & SW_FORCE_LAST, flags & SW_FORCE_FIRST, t);
  select_row(J, idx + (int64_t)gb * tau_max, tau_max, count + gb);
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
  RowJob J = make_job(r + (int64_t)seq * max_blocks, n_cand, bq, true, flags & SW_FORCE_FIRST, tt);
  select_row(J, idx + (int64_t)seq * tau_max, tau_max, count + seq);
}

}  // namespace

namespace sw {

int32_t launch_select(const sw_layout& L, const float* R, const int32_t* tau, int tau_max,
                      uint32_t flags, int32_t* idx, int32_t* count, cudaStream_t st) {
  if (L.total_blocks == 0) return SW_OK;
  select_topk_kernel<<<L.total_blocks, kThreads, 0, st>>>(R, L.cu_blocks, L.cu_sq, L.batch, tau, tau_max,
                                                          flags, idx, count);
  return check_launch("sw_select_topk");
}

int32_t launch_select_row(int batch, int block, int max_blocks, const float* r, const int32_t* seqlens,
                          const int32_t* tau, int tau_max, uint32_t flags, int32_t* idx, int32_t* count,
                          cudaStream_t st) {
  if (batch == 0) return SW_OK;
  select_topk_row_kernel<<<batch, kThreads, 0, st>>>(r, seqlens, block, max_blocks, tau, tau_max, flags,
                                                     idx, count);
  return check_launch("sw_select_topk_row");
}

}  // namespace sw
