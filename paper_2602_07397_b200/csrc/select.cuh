// Block-wide exact top-k of one score row (Alg. 1 Step 7 PAPER.md:788-791, Alg. 2 Step 6
// PAPER.md:832-833; readings P7, P8): forced blocks + radix select of the rest on an
// order-preserving uint32 image of the fp32 scores, ties to the lower index, output ascending.
// Integer work only, hence bit-exact.  Shared by select.cu and decode_select.cu.
//
// One CTA of kThreads threads per row (256 unless the translation unit defines SWSEL_THREADS, a multiple of 256,
// before including this file):
//   * rows of up to 8 * kThreads candidates keep their keys in registers (2, 4 or 8 per thread by row length) and
//     take 3 radix passes of 11 + 11 + 10 bits on one shared histogram of 2048 bins (plain shared-memory atomics; a
//     warp whose keys all hit the same bin sends one add); every thread owns 2048 / kThreads adjacent bins, a
//     block-wide suffix scan of the owners' counts picks the bin: three barriers per pass.  (Four passes of 8 bits
//     with four barriers each took 6 of the 12 us of the decode tail: scores rescaled to [0, 1] share a handful of
//     exponent bytes, so the first pass serialised on two or three bins.)
//   * longer rows re-read their scores: 4 passes of 8 bits, thread b < 256 owns bin b;
//   * one ordered compaction: every thread owns a contiguous index range, a block scan of the
//     (certain, equal-to-threshold) counts gives each range its output offset.
#pragma once

#include <stdint.h>

namespace swsel {

#ifndef SWSEL_THREADS
#define SWSEL_THREADS 256
#endif
constexpr int kThreads = SWSEL_THREADS;
constexpr int kWarps = kThreads / 32;
static_assert(kThreads >= 256 && kThreads % 256 == 0 && kWarps <= 32, "thread b < 256 owns histogram bin b; one lane per warp total");

constexpr int kBins = 2048;                  // register path: digits of 11, 11 and 10 bits
constexpr int kBinsPer = kBins / kThreads;   // adjacent bins owned by a thread
static_assert(kBins % kThreads == 0, "every thread owns the same number of bins");

struct Scratch {
  alignas(16) uint32_t hist[kBins];
  uint32_t warp_tot[kWarps];
  unsigned long long warp_scan[kWarps];
  uint32_t bcast[2];
};

// fp32 -> uint32 whose unsigned order equals the float order; NaN ranks as -inf (P8)
__device__ __forceinline__ uint32_t order_key(float v) {
  if (v != v) v = -INFINITY;
  if (v == 0.f) v = 0.f;               // -0 and +0 compare equal
  uint32_t u = __float_as_uint(v);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// sum of t[w] over the warps w > warp (suffix) or w < warp (prefix): every warp reads the kWarps <= 32 totals once and
// adds them with shuffles -- a loop over the totals is a chain of dependent shared-memory loads (31 of them for the
// first warp of 1024 threads: 0.8 us per radix pass, measured)
__device__ __forceinline__ uint32_t warps_above(const uint32_t* t, int warp, int lane) {
  uint32_t v = (lane < kWarps && lane > warp) ? t[lane] : 0u;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ unsigned long long warps_below(const unsigned long long* t, int warp, int lane) {
  unsigned long long v = (lane < kWarps && lane < warp) ? t[lane] : 0ull;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

struct RowJob {
  int n_cand;            // candidates are [0, n_cand)
  int f0, f1;            // forced indices (-1 = none), already inside [0, n_cand), f0 != f1
  int need;              // how many non-forced candidates to pick
  int budget;            // total selected
};

__device__ __forceinline__ RowJob make_job(int n_cand, int diag, bool force_last, bool force_first, int tau) {
  RowJob J;
  J.n_cand = n_cand;
  J.budget = min(tau, n_cand);
  J.f0 = -1; J.f1 = -1;
  int nf = 0;
  if (force_last && diag >= 0 && diag < n_cand && nf < J.budget) { J.f0 = diag; ++nf; }
  if (force_first && n_cand > 0 && 0 != J.f0 && nf < J.budget) { J.f1 = 0; ++nf; }
  J.need = J.budget - nf;
  return J;
}

__device__ __forceinline__ bool is_forced(const RowJob& J, int j) { return j == J.f0 || j == J.f1; }

// One histogram update per lane (bin 256 = none).  Shared-memory atomics of a warp to distinct bins run in
// parallel and to a few bins fast enough (measured: faster than match.any aggregation, which costs one
// round per distinct value); only the degenerate row whose keys all fall into one bin would serialise
// 32 ways on every update, so a warp that agrees on its bin sends a single add.
__device__ __forceinline__ void hist_add(Scratch& S, uint32_t bin, int lane) {
  const uint32_t b0 = __shfl_sync(0xffffffffu, bin, 0);
  if (__all_sync(0xffffffffu, bin == b0)) {
    if (lane == 0 && b0 < 256u) atomicAdd(&S.hist[b0], 32u);
  } else if (bin < 256u) {
    atomicAdd(&S.hist[bin], 1u);
  }
}

// After the 4 passes `thr` is the key of the need-th largest non-forced candidate and `n_gt` the
// number of non-forced candidates with a strictly larger key.  All threads return the same values.
template <typename Load>
__device__ void radix_threshold(Load load, const RowJob& J, Scratch& S, uint32_t& thr, int& n_gt_out) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t prefix = 0;
  int remaining = J.need;      // rank (1-based, from the top) still to locate inside the prefix bucket
  int n_gt = 0;
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    if (tid < 256) S.hist[tid] = 0;
    __syncthreads();
    const uint32_t mask_hi = (pass == 0) ? 0u : (0xffffffffu << (shift + 8));
    for (int j0 = 0; j0 < J.n_cand; j0 += kThreads) {
      const int j = j0 + tid;
      uint32_t bin = 256u;                              // not a candidate of this pass
      if (j < J.n_cand && !is_forced(J, j)) {
        const uint32_t k = order_key(load(j));
        if ((k & mask_hi) == prefix) bin = (k >> shift) & 0xffu;
      }
      hist_add(S, bin, lane);
    }
    __syncthreads();
    // thread b owns bin b: count, then an inclusive suffix sum over bins b..255
    const uint32_t cnt = (tid < 256) ? S.hist[tid] : 0u;
    uint32_t suf = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_down_sync(0xffffffffu, suf, o);
      if (lane + o < 32) suf += v;
    }
    if (lane == 0) S.warp_tot[warp] = suf;
    __syncthreads();
    suf += warps_above(S.warp_tot, warp, lane);
    const uint32_t above = suf - cnt;                   // candidates in strictly higher bins
    if ((int)above < remaining && (int)suf >= remaining) { S.bcast[0] = (uint32_t)tid; S.bcast[1] = above; }
    __syncthreads();
    prefix |= S.bcast[0] << shift;
    n_gt += (int)S.bcast[1];
    remaining -= (int)S.bcast[1];
  }
  thr = prefix;
  n_gt_out = n_gt;
}

// Register variant for rows of at most kRegKeys * kThreads candidates (b <= 2048 at 256 threads): every thread keeps
// the keys of its contiguous index range [lo, hi) in registers, so the passes and the compaction touch memory only
// for the histogram.  cmask: bit e set = index lo + e is a non-forced candidate.  Three passes (bits 31-21, 20-10,
// 9-0); thread t owns bins [t kBinsPer, (t + 1) kBinsPer) and clears them as it reads them.
constexpr int kRegKeys = 8;
template <int K>
__device__ __forceinline__ void radix_threshold_regs(const uint32_t (&key)[K], uint32_t cmask, const RowJob& J,
                                                     Scratch& S, uint32_t& thr, int& n_gt_out) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t prefix = 0;
  int remaining = J.need;      // rank (1-based, from the top) still to locate inside the prefix bucket
  int n_gt = 0;
#pragma unroll
  for (int b = 0; b < kBinsPer; ++b) S.hist[tid * kBinsPer + b] = 0;
  __syncthreads();
#pragma unroll
  for (int pass = 0; pass < 3; ++pass) {
    const int shift = (pass == 0) ? 21 : (pass == 1) ? 10 : 0;
    const uint32_t dmask = (pass == 2) ? 0x3ffu : 0x7ffu;
    const uint32_t mask_hi = (pass == 0) ? 0u : (pass == 1) ? 0xffe00000u : 0xfffffc00u;
    uint32_t bin[K];
    bool same = true;
#pragma unroll
    for (int e = 0; e < K; ++e) {
      const bool in = ((cmask >> e) & 1u) && (key[e] & mask_hi) == prefix;
      bin[e] = in ? ((key[e] >> shift) & dmask) : (uint32_t)kBins;
      same = same && bin[e] == bin[0];
    }
    // plain shared-memory atomics (distinct bins of a warp run in parallel); only a warp whose keys all fall into
    // one bin -- the degenerate row of equal scores -- would serialise, so it sends a single add
    const uint32_t b0 = __shfl_sync(0xffffffffu, bin[0], 0);
    if (__all_sync(0xffffffffu, same && bin[0] == b0)) {
      if (lane == 0 && b0 < (uint32_t)kBins) atomicAdd(&S.hist[b0], 32u * K);
    } else {
#pragma unroll
      for (int e = 0; e < K; ++e)
        if (bin[e] < (uint32_t)kBins) atomicAdd(&S.hist[bin[e]], 1u);
    }
    __syncthreads();
    // counts of the own bins (cleared for the next pass), then an inclusive suffix sum over the owners t..kThreads-1
    uint32_t cnt[kBinsPer], own = 0;
    if constexpr (kBinsPer % 4 == 0) {                  // 128-bit accesses: 8 words per thread would conflict 8 ways
      uint4* h4 = reinterpret_cast<uint4*>(S.hist + tid * kBinsPer);
#pragma unroll
      for (int b = 0; b < kBinsPer / 4; ++b) {
        const uint4 v = h4[b];
        h4[b] = make_uint4(0u, 0u, 0u, 0u);
        cnt[4 * b] = v.x; cnt[4 * b + 1] = v.y; cnt[4 * b + 2] = v.z; cnt[4 * b + 3] = v.w;
      }
    } else {
#pragma unroll
      for (int b = 0; b < kBinsPer; ++b) {
        cnt[b] = S.hist[tid * kBinsPer + b];
        S.hist[tid * kBinsPer + b] = 0;
      }
    }
#pragma unroll
    for (int b = 0; b < kBinsPer; ++b) own += cnt[b];
    uint32_t suf = own;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_down_sync(0xffffffffu, suf, o);
      if (lane + o < 32) suf += v;
    }
    if (lane == 0) S.warp_tot[warp] = suf;
    __syncthreads();
    suf += warps_above(S.warp_tot, warp, lane);
    uint32_t above = suf - own;                         // candidates in the bins of higher threads
#pragma unroll
    for (int b = kBinsPer - 1; b >= 0; --b) {
      if ((int)above < remaining && (int)(above + cnt[b]) >= remaining) {
        S.bcast[0] = (uint32_t)(tid * kBinsPer + b);
        S.bcast[1] = above;
      }
      above += cnt[b];
    }
    __syncthreads();
    prefix |= S.bcast[0] << shift;
    n_gt += (int)S.bcast[1];
    remaining -= (int)S.bcast[1];
  }
  thr = prefix;
  n_gt_out = n_gt;
}

// Register path: every thread keeps the K keys of its contiguous index range [lo, hi) in registers (rows of at most
// K * kThreads candidates).  K is chosen by the row length (2, 4 or 8): the passes cost K bin computations and
// atomics per thread whatever the row length, and a short row (b = 512: 2 keys per thread) was issue-bound at K = 8.
template <int K, typename Load>
__device__ __forceinline__ void select_row_regs(Load load, const RowJob& J, int32_t* __restrict__ out, int tau_max,
                                              int32_t* __restrict__ count_out, Scratch& S, bool take_all, int lo, int hi) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t thr = 0;
  int n_gt = 0;
  uint32_t key[K];
  uint32_t cmask = 0, fmask = 0;
#pragma unroll
  for (int e = 0; e < K; ++e) {
    const int j = lo + e;
    key[e] = 0;
    if (j < hi) {
      if (is_forced(J, j)) fmask |= 1u << e;
      else { cmask |= 1u << e; key[e] = order_key(load(j)); }
    }
  }
  if (!take_all && J.need > 0) radix_threshold_regs(key, cmask, J, S, thr, n_gt);
  const int eq_quota = J.need - n_gt;
  uint32_t cert = fmask, eqm = 0;                   // bit e: index lo + e is certainly in / equals the threshold
#pragma unroll
  for (int e = 0; e < K; ++e) {
    if ((cmask >> e) & 1u) {
      if (take_all) cert |= 1u << e;
      else if (J.need > 0) {
        if (key[e] > thr) cert |= 1u << e;
        else if (key[e] == thr) eqm |= 1u << e;
      }
    }
  }
  unsigned long long v = ((unsigned long long)__popc(eqm) << 32) | (unsigned)__popc(cert), incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long u = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += u;
  }
  if (lane == 31) S.warp_scan[warp] = incl;
  __syncthreads();
  const unsigned long long base = warps_below(S.warp_scan, warp, lane);
  const unsigned long long excl = base + incl - v;
  int c_before = (int)(excl & 0xffffffffu), e_before = (int)(excl >> 32);
#pragma unroll
  for (int e = 0; e < K; ++e) {
    const bool c = (cert >> e) & 1u, q = (eqm >> e) & 1u;
    const int pos = c_before + min(e_before, eq_quota);
    if ((c || (q && e_before < eq_quota)) && pos < tau_max) out[pos] = lo + e;
    c_before += c; e_before += q;
  }
  for (int p = J.budget + tid; p < tau_max; p += kThreads) out[p] = -1;
  if (tid == 0) *count_out = J.budget;
  __syncthreads();                          // scratch may be reused by the caller
}

// load(j): score of candidate j (global or shared memory).  out: tau_max ints (ascending, -1 padded).
template <typename Load>
__device__ void select_row(Load load, const RowJob& J, int32_t* __restrict__ out, int tau_max,
                           int32_t* __restrict__ count_out, Scratch& S) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t thr = 0;
  int n_gt = 0;
  const int n_free = J.n_cand - (J.f0 >= 0) - (J.f1 >= 0);
  const bool take_all = J.need >= n_free;
  // ordered compaction: thread t owns indices [t*per, (t+1)*per)
  const int per = (J.n_cand + kThreads - 1) / kThreads;
  const int lo = min(tid * per, J.n_cand), hi = min(lo + per, J.n_cand);
  if (per <= 2) { select_row_regs<2>(load, J, out, tau_max, count_out, S, take_all, lo, hi); return; }
  if (per <= 4) { select_row_regs<4>(load, J, out, tau_max, count_out, S, take_all, lo, hi); return; }
  if (per <= kRegKeys) { select_row_regs<kRegKeys>(load, J, out, tau_max, count_out, S, take_all, lo, hi); return; }
  if (!take_all && J.need > 0) radix_threshold(load, J, S, thr, n_gt);
  const int eq_quota = J.need - n_gt;       // equal-key candidates to take, lowest index first

  auto classify = [&](int j, bool& certain, bool& eq) {
    certain = false; eq = false;
    if (is_forced(J, j)) { certain = true; return; }
    if (take_all) { certain = true; return; }
    if (J.need > 0) {
      const uint32_t k = order_key(load(j));
      certain = k > thr;
      eq = k == thr;
    }
  };
  uint32_t n_c = 0, n_e = 0;
  for (int j = lo; j < hi; ++j) {
    bool c, e;
    classify(j, c, e);
    n_c += c; n_e += e;
  }
  unsigned long long v = ((unsigned long long)n_e << 32) | n_c, incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long u = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += u;
  }
  if (lane == 31) S.warp_scan[warp] = incl;
  __syncthreads();
  const unsigned long long base = warps_below(S.warp_scan, warp, lane);
  const unsigned long long excl = base + incl - v;
  int c_before = (int)(excl & 0xffffffffu), e_before = (int)(excl >> 32);
  for (int j = lo; j < hi; ++j) {
    bool c, e;
    classify(j, c, e);
    const int pos = c_before + min(e_before, eq_quota);
    if ((c || (e && e_before < eq_quota)) && pos < tau_max) out[pos] = j;
    c_before += c; e_before += e;
  }
  for (int p = J.budget + tid; p < tau_max; p += kThreads) out[p] = -1;
  if (tid == 0) *count_out = J.budget;
  __syncthreads();                            // scratch may be reused by the caller
}

}  // namespace swsel
