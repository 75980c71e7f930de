// sw_decode_select, the kernel of Alg. 2 Steps 2-4 for one new token per sequence: the
// head-averaged query and its sketch q~_t (Step 3), on the tile that holds b_q the running key-block mean and its
// sketch (Step 2, written to the caches in place), and the raw scores q~_t . k~_j / sqrt(r) of the new row
// (Steps 3-4), left in the workspace for the tail kernel.
//
// This work is a chain of short dependent steps (loads, two block-wide reductions, an in-warp FWHT, 64 dot products
// per tile), a few microseconds whatever one does.  It used to run at the head of the streaming CTAs, where it held
// back the cached-W stream of 256 of the 296 CTAs for ~5 us each (measured: 22 us for the 67 MB of cfg 3).  As its own
// small kernel it runs BESIDE the stream: it is the streaming kernel's programmatic dependent, released once every
// streaming CTA has passed griddepcontrol.wait (= everything before this layer's selection is complete), reads nothing
// the stream writes, and waits for the stream only at its very end so that the tail's wait covers both.
#include "common.cuh"
#include "decode_select.cuh"
#include "sketch_common.cuh"

namespace {

using namespace swds;

// One CTA of 128 threads per (sequence, 64-column tile): all its loads are in flight at once (one round trip through
// a memory system the stream keeps busy: a CTA that walked over four tiles took 17 us beside the stream, this takes
// ~6).  The CTAs are launched behind the streaming kernel's (two per SM, placed first) and several fit beside those.
template <typename TIn, int D>
__global__ void __launch_bounds__(kDutyThreads, 6)
decode_duty_kernel(const Params p_in) {
  Params p = p_in;                                    // (the pointers to earlier kernels' data pass through pdl_wait)
  __shared__ __align__(16) float s_vec[D], s_qt[128], s_kt[128], s_sign[D];
  __shared__ float s_hx[kDutyThreads / D][D];
  __shared__ int32_t s_cols[128];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int seq = blockIdx.y;
  // Released by the streaming kernel after that one's griddepcontrol.wait: everything before this layer's selection
  // is complete, and the streaming kernel writes nothing this kernel reads.  Without a walk state there is no
  // streaming kernel in front and this kernel waits for its predecessors itself.  Either way the first kernel of a
  // selection releases its dependents only AFTER its wait, so nothing later in the stream (the tail's prologue, the
  // next layer's streaming kernel) runs before everything in front of this selection is complete.
  if (!p.streamed) swd::pdl_wait(p.q, p.k, p.seqlens, p.kbar, p.ks);
  swd::pdl_launch_dependents();                       // the tail may become resident (it waits for this kernel)
  const int mb = p.max_blocks;
  const int t = __ldcg(p.seqlens + seq);
  const bool live = seq_live(t, p.B, mb);             // (an idle slot of the batch has no tile: a = -1)
  const int bq = live ? (t - 1) / p.B : 0, a = live ? bq / kDutyTile : -1;   // block of the new token = b_curr
  const int hi = bq + 1;
  constexpr int kGroups = kDutyThreads / D;
  const int q4 = p.r >> 2;                            // float4s per sketch row
  const bool vec_ok = (p.r & 3) == 0 && q4 >= 1 && q4 <= 32 && (q4 & (q4 - 1)) == 0 && kDutyTile * q4 <= kKU * kDutyThreads &&
                      (reinterpret_cast<uintptr_t>(p.ks) & 15u) == 0;
  const int hx = tid % D, hg = tid / D;
  const float* ksb = p.ks + (int64_t)seq * mb * p.r;
  const int part = vec_ok ? (tid & (q4 - 1)) : 0, per_pass = vec_ok ? kDutyThreads / q4 : 1;
  const int colq = vec_ok ? tid / q4 : 0;
  float* sc = p.ws_scores + (int64_t)seq * p.mbp;

  for (int sub = 0; sub < kDutyGroup; ++sub) {
    const int tile = blockIdx.x * kDutyGroup + sub;
    if (tile > a) break;
    const int col0 = tile * kDutyTile;
    const bool need_q = sub == 0, need_k = tile == a; // the tile that holds b_q owns the key-side update of Step 2
    // ---- all loads of the tile, before anything waits on memory: unconditional loads from clamped (always valid)
    // addresses, raw values kept in registers -- a predicated load followed by its convert makes every group of
    // loads wait for the previous one
    TIn qraw[kHeadRegs], kraw[kHeadRegs];
    float4 kv[kKU];
    const TIn* qp = reinterpret_cast<const TIn*>(p.q) + (int64_t)seq * p.q_stride_seq + hx;
    const TIn* kp = reinterpret_cast<const TIn*>(p.k) + (int64_t)seq * p.k_stride_seq + hx;
#pragma unroll
    for (int u = 0; u < kHeadRegs; ++u) {
      const int h = hg + u * kGroups;
      qraw[u] = qp[(int64_t)min(h, p.h_q - 1) * p.q_stride_head];
      kraw[u] = kp[(int64_t)min(h, p.h_kv - 1) * p.k_stride_head];
    }
    const int cnt = (t - 1) % p.B;                    // tokens already in block b_curr
    float* kb = p.kbar + ((int64_t)seq * mb + bq) * D;
    const float kbar_old = kb[tid & (D - 1)];
#pragma unroll
    for (int u = 0; u < kKU; ++u) {
      const int cj = u * per_pass + colq;
      const int j = min(col0 + min(cj, kDutyTile - 1), bq);                    // clamped: always a valid row
      kv[u] = vec_ok ? *reinterpret_cast<const float4*>(ksb + (int64_t)j * p.r + part * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    // ---- head means, running key-block mean, sketches ----------------------------------------------------------
    if (need_q || need_k) {
      if (need_q) {
        if (tid < D) s_sign[tid] = p.signs ? (float)p.signs[tid] : 1.f;
        if (tid < p.r && tid < 128) s_cols[tid] = p.cols[tid];
      }
      float sq = 0.f, sk = 0.f;
#pragma unroll
      for (int u = 0; u < kHeadRegs; ++u) {
        const int h = hg + u * kGroups;
        if (h < p.h_q) sq += (float)qraw[u];
        if (h < p.h_kv) sk += (float)kraw[u];
      }
      if (need_q) for (int h = hg + kHeadRegs * kGroups; h < p.h_q; h += kGroups) sq += (float)qp[(int64_t)h * p.q_stride_head];
      if (need_k) for (int h = hg + kHeadRegs * kGroups; h < p.h_kv; h += kGroups) sk += (float)kp[(int64_t)h * p.k_stride_head];
      if (need_q) {
        s_hx[hg][hx] = sq;
        __syncthreads();
        if (tid < D) {
          float acc = 0.f;
#pragma unroll
          for (int g = 0; g < kGroups; ++g) acc += s_hx[g][tid];
          s_vec[tid] = acc / (float)p.h_q;
        }
        __syncthreads();
        swsk::sketch_tail<D>(s_vec, s_sign, s_cols, p.r, p.scale, s_qt);       // q~_t
        __syncthreads();
      }
      if (need_k) {
        s_hx[hg][hx] = sk;
        __syncthreads();
        if (tid < D) {
          float acc = 0.f;
#pragma unroll
          for (int g = 0; g < kGroups; ++g) acc += s_hx[g][tid];
          const float avg = acc / (float)p.h_kv;
          const float mn = (cnt == 0) ? avg : ((float)cnt * kbar_old + avg) / (float)(cnt + 1);
          kb[tid] = mn;
          s_vec[tid] = mn;
        }
        __syncthreads();
        swsk::sketch_tail<D>(s_vec, s_sign, s_cols, p.r, p.scale, s_kt, p.ks + ((int64_t)seq * mb + bq) * p.r);
        __syncthreads();
      }
    }
    // ---- raw scores of the tile's columns (Steps 3-4; column b_q from the fresh sketch) --------------------------
    if (vec_ok) {
      // q4 adjacent lanes share one column; partial dots meet in a fixed xor butterfly
      const float4 qv = *reinterpret_cast<const float4*>(s_qt + part * 4);
#pragma unroll
      for (int u = 0; u < kKU; ++u) {
        if (u * per_pass >= kDutyTile) break;                                  // warp-uniform
        const int cj = u * per_pass + colq, j = col0 + cj;
        if (j == bq) kv[u] = *reinterpret_cast<const float4*>(s_kt + part * 4);
        float acc = fmaf(qv.w, kv[u].w, fmaf(qv.z, kv[u].z, fmaf(qv.y, kv[u].y, qv.x * kv[u].x)));
        for (int o = q4 >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (part == 0 && cj < kDutyTile && j < hi) sc[j] = acc * p.inv_sqrt_r;
      }
    } else {
      for (int cj = warp; cj < kDutyTile; cj += kDutyThreads / 32) {
        const int j = col0 + cj;
        if (j < hi) {
          const float* kr = (j == bq) ? s_kt : ksb + (int64_t)j * p.r;
          float acc = 0.f;
          for (int c = lane; c < p.r; c += 32) acc = fmaf(s_qt[c], kr[c], acc);
          acc = swd::warp_sum(acc);
          if (lane == 0) sc[j] = acc * p.inv_sqrt_r;
        }
      }
    }
  }
  // The tail kernel waits for this kernel only; one CTA waiting for the streaming kernel here makes "this kernel
  // complete" imply "stream complete".  Only one: a CTA that stays resident keeps the tail (1024 threads, a whole
  // SM's registers) off its SM, and the tail's prologue should run while the last streaming CTAs drain.
  if (blockIdx.x == 0 && blockIdx.y == 0) swd::pdl_wait();
}

}  // namespace

namespace sw {

int32_t launch_decode_duty(const swds::Params& p, cudaStream_t st) {
  void (*kern)(const Params) = nullptr;
  const int d = p.d;
  if (p.dtype == SW_BF16 && d == 128) kern = decode_duty_kernel<__nv_bfloat16, 128>;
  else if (p.dtype == SW_BF16 && d == 64) kern = decode_duty_kernel<__nv_bfloat16, 64>;
  else if (p.dtype == SW_F32 && d == 128) kern = decode_duty_kernel<float, 128>;
  else if (p.dtype == SW_F32 && d == 64) kern = decode_duty_kernel<float, 64>;
  else return fail(SW_ERR_UNSUPPORTED, "sw_decode_select: dtype %d / d %d", p.dtype, d);
  count_launch();
  launch_pdl(kern, dim3(cdiv(cdiv(p.max_blocks, kDutyTile), kDutyGroup), p.batch), dim3(kDutyThreads), 0, st, p);
  return check_launch("sw_decode_select(duty)");
}

}  // namespace sw
