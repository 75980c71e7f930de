// sw_sparse_attn_prefill, sm_100a fast path: block-sparse FlashAttention on tcgen05 tensor cores with
// TMEM accumulators and TMA-gathered K/V tiles.  Alg. 1 Step 8, "zero outside selected
// blocks, renormalized within"; GQA mapping P14.
//
// Work unit (one CTA): a 64-token query tile of one KV-head group (4 q-heads) = 256 query rows, row =
// 4*token + head, processed as two 128-row MMA tiles t = 0, 1.  The selected key blocks of the query
// block are cut into 64-key chunks k = 0..n-1; per tile and chunk:
//     S_t(k) = Q_t K(k)^T     tcgen05.mma  M=128 N=64  K=16 x8   A, B from shared memory (K-major, SW128)
//     P_t(k) = exp2(S*c - m)  fp32 online softmax in registers, one thread per row, P written back to
//                             TMEM as bf16 over the first half of the S columns
//     O_t   += P_t(k) V(k)    tcgen05.mma  M=128 N=128 K=16 x4   A from TMEM, B from shared memory (MN-major)
// TMEM (512 columns): S_t[buf] at t*128 + buf*64 (two S buffers per tile), O_t at 256 + t*128.
// The S buffers decouple the tensor pipe from the softmax warps: QK(k+1) is issued before the softmax
// of chunk k finishes, so a softmax warp never waits for its next S while the tensor pipe works on
// PV(k) / QK(k+2), and the two tiles' softmax warps (one of each per SM sub-partition) run
// concurrently, interleaving their MUFU and FMA work.
// Warps: 0 = TMA producer, 1 = MMA issuer of tile 0, 2 = TMEM allocator, 3 = chunk-list builder, then
//        MMA issuer of tile 1, 4-7 = softmax/epilogue of tile 0, 8-11 = softmax/epilogue of tile 1.
// MMA issue order per tile and chunk k:  PV(k) QK(k+2); the two tiles' streams interleave on the pipe.
// The O rescale is lazy: the running max is only raised (and O multiplied) when it grew by more than
// 2^8, which keeps P within bf16/fp32 range and is exact after the final 1/l; a rescale first waits
// for PV(k-1) of its tile (o_ready barrier).
// A quarter of the exp2 runs on the FMA pipe (ex2_poly2), because MUFU ex2 at 16/clk/SM costs as many
// cycles per chunk as the chunk's MMAs.  The Q tile is requested before the set-up barrier; the bf16
// output leaves through the (then free) Q buffer and one TMA store per d-half and tile.
// kTiles = 1 builds the variant with one 128-row tile per CTA and two CTAs per SM (measured slower).
#include "common.cuh"
#include "sm100.cuh"

namespace {

using namespace sm100;

#ifndef SW_TILES
#define SW_TILES 2
#endif
constexpr int kTiles = SW_TILES;              // 128-row MMA tiles per CTA: 2 (one CTA per SM) or 1 (two CTAs per SM)
constexpr int kQTok = 32 * kTiles;            // query tokens per CTA
constexpr int kThreads = 128 + 128 * kTiles;
constexpr int kStages = 4 * kTiles;           // ring of 64-key K or V tiles
constexpr int kTmemCols = 256 * kTiles;
constexpr int kTileBytes = 64 * 128 * 2;      // 16 KB: [d-half][64 keys][128 B]
constexpr int kQBytes = kTiles * 128 * 128 * 2;   // 32 KB per tile: [d-half][128 kTiles rows][128 B]
constexpr int kMaxChunks = 2048 * kTiles;     // 64-key chunks per query row the list buffer holds
constexpr int kSmemBytes = kQBytes + kStages * kTileBytes + kMaxChunks * 4 + 1024 /*align*/ + 512 /*barriers*/;
constexpr float kRescaleThreshold = 8.0f;     // log2 units
#ifndef SW_EARLY_K
#define SW_EARLY_K 1
#endif
constexpr bool kEarlyK = SW_EARLY_K;          // request the first K tiles before the chunk list is built

// barrier map
constexpr int kBarQ = 0;                      // Q tile landed
constexpr int kBarFull = 1;                   // [kStages] K/V tile landed
constexpr int kBarEmpty = kBarFull + kStages; // [kStages] K/V tile consumed
constexpr int kBarS = kBarEmpty + kStages;    // [t][buf] S ready          (tcgen05.commit)
constexpr int kBarP = kBarS + 4;              // [t][buf] P written         (4 warps arrive)
constexpr int kBarO = kBarP + 4;              // [t] PV(k) done             (tcgen05.commit)
constexpr int kBarDone = kBarO + 2;           // all MMAs done
constexpr int kNumBars = kBarDone + 1;

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
// 2^x on the FMA pipe for a pair of values (x <= ~16): round-to-nearest split x = n + f with the
// 1.5*2^23 magic add, degree-3 minimax polynomial of 2^f on [-0.5, 0.5] (max relative error 7.5e-5,
// well under the bf16 rounding of P), n added into the exponent field.  Takes MUFU work off the
// softmax warps: ex2.approx runs at 16/clk/SM, which at 64 exps per row and key chunk costs exactly
// as many cycles as the chunk's two MMAs.
#ifndef SW_POLY_MASK
#define SW_POLY_MASK 0x88
#endif
// bit q set = column pair q (mod 8) of a row takes the polynomial; which pairs matters as much as how
// many (the compiler's interleaving of the MUFU and FMA streams changes): measured on cfg 2, 0x88
// (pairs 3 and 7) 2.69 ms, 0x80 2.98 ms, 0xA4 2.76 ms, none 2.93 ms
__host__ __device__ constexpr bool use_poly(int pair) { return (SW_POLY_MASK >> (pair % 8)) & 1; }
__device__ __forceinline__ float2 ex2_poly2(float2 x) {
  x.x = fmaxf(x.x, -125.f);
  x.y = fmaxf(x.y, -125.f);
  const float2 magic = make_float2(12582912.f, 12582912.f), nmagic = make_float2(-12582912.f, -12582912.f);
  const float2 t = __fadd2_rn(x, magic);                        // low mantissa bits of t = n = rint(x)
  const float2 nf = __fadd2_rn(t, nmagic);
  const float2 f = __fadd2_rn(x, make_float2(-nf.x, -nf.y));
  float2 pl = __ffma2_rn(f, make_float2(0.055171459913253784f, 0.055171459913253784f),
                         make_float2(0.2426108568906784f, 0.2426108568906784f));
  pl = __ffma2_rn(pl, f, make_float2(0.6932609677314758f, 0.6932609677314758f));
  pl = __ffma2_rn(pl, f, make_float2(0.9999281167984009f, 0.9999281167984009f));
  float2 r;
  r.x = __uint_as_float(__float_as_uint(pl.x) + (__float_as_uint(t.x) << 23));
  r.y = __uint_as_float(__float_as_uint(pl.y) + (__float_as_uint(t.y) << 23));
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

__global__ void __launch_bounds__(kThreads, 3 - kTiles)
attn_prefill_sm100_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                          const __grid_constant__ CUtensorMap map_v, const __grid_constant__ CUtensorMap map_o,
                          const Params p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* base = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const uint32_t sQ = smem_u32(base);
  const uint32_t sKV = sQ + kQBytes;
  int32_t* s_list = reinterpret_cast<int32_t*>(base + kQBytes + kStages * kTileBytes);
  uint64_t* bars = reinterpret_cast<uint64_t*>(base + kQBytes + kStages * kTileBytes + kMaxChunks * 4);
  const uint32_t bar0 = smem_u32(bars);
  auto BAR = [&](int i) { return bar0 + 8u * i; };
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(bars + kNumBars);
  volatile int32_t* s_nchunks = reinterpret_cast<volatile int32_t*>(bars + kNumBars + 1);
  volatile int32_t* s_pre = s_nchunks + 1;                   // K tiles requested during set-up (0, 1 or 2)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- work unit ---------------------------------------------------------------------------
  const int TPB = p.B >> 6;
  const int slot_id = p.total_slots - 1 - (int)blockIdx.x;     // longest rows first
  const int QPB = p.B / kQTok;                                 // query tiles (CTAs) per block
  const int gb = slot_id / QPB, sub = slot_id - gb * QPB;
  const int kvh = blockIdx.y;
  const int seq = swd::find_seq(p.cu_blocks, p.batch, gb);
  const int bi = gb - __ldg(p.cu_blocks + seq);
  const int seq_lo = __ldg(p.cu_seqlens + seq), seq_hi = __ldg(p.cu_seqlens + seq + 1);
  const int q_tok0 = seq_lo + bi * p.B + sub * kQTok;
  const int q_valid = min(kQTok, seq_hi - q_tok0);
  if (q_valid <= 0) return;
  const int q_last = q_tok0 + q_valid - 1;

  // ---- one-time setup ------------------------------------------------------------------------
  if (warp == 0 && lane == 0) {
    prefetch_tmap(&map_q); prefetch_tmap(&map_k); prefetch_tmap(&map_v); prefetch_tmap(&map_o);
    mbar_init(BAR(kBarQ), 1);
    for (int s = 0; s < kStages; ++s) { mbar_init(BAR(kBarFull + s), 1); mbar_init(BAR(kBarEmpty + s), kTiles); }
    for (int i = 0; i < 4; ++i) { mbar_init(BAR(kBarS + i), 1); mbar_init(BAR(kBarP + i), 4); }
    mbar_init(BAR(kBarO), 1); mbar_init(BAR(kBarO + 1), 1);
    mbar_init(BAR(kBarDone), kTiles);
    fence_barrier_init();
    // the Q tile does not depend on the chunk list: request it before the set-up barrier
    mbar_arrive_expect_tx(BAR(kBarQ), kQBytes);
    tma_load_3d(sQ, &map_q, BAR(kBarQ), 0, kvh * 4, q_tok0);
    tma_load_3d(sQ + kQBytes / 2, &map_q, BAR(kBarQ), 64, kvh * 4, q_tok0);
    // The chunk list (built by warp 3, below) starts with the first 64 keys of idx[0] when that block holds a visible
    // key, followed, for 64-token blocks, by those of idx[1] when that one does too: request those K tiles now
    // instead of after the list has been built and the set-up barrier passed -- their latency then overlaps both.
    // The lists are the caller's (any order, hand-built ones included): an entry the list builder drops -- -1, a
    // block past the end of the sequence, a block the causal mask hides entirely -- is not requested here either,
    // and nothing behind it is, so that stage s always holds chunk s of the list.
    if (kEarlyK) {
      const int32_t* list = p.idx + (int64_t)gb * p.tau_max;
      const int cnt = __ldg(p.count + gb);
      const int j0 = __ldg(list), j1 = (p.tau_max > 1) ? __ldg(list + 1) : -1;
      auto listed = [&](int j) {                              // the list builder's predicate on a block's first chunk
        if (j < 0) return false;
        const int k0 = seq_lo + j * p.B;
        return k0 < seq_hi && !(p.causal && k0 > q_last);
      };
      int pre = 0;
      if (cnt > 0 && listed(j0)) {
        mbar_arrive_expect_tx(BAR(kBarFull + 0), kTileBytes);
        tma_load_3d(sKV, &map_k, BAR(kBarFull + 0), 0, kvh, seq_lo + j0 * p.B);
        tma_load_3d(sKV + kTileBytes / 2, &map_k, BAR(kBarFull + 0), 64, kvh, seq_lo + j0 * p.B);
        pre = 1;
        if (TPB == 1 && cnt > 1 && listed(j1)) {
          mbar_arrive_expect_tx(BAR(kBarFull + 1), kTileBytes);
          tma_load_3d(sKV + kTileBytes, &map_k, BAR(kBarFull + 1), 0, kvh, seq_lo + j1 * p.B);
          tma_load_3d(sKV + kTileBytes + kTileBytes / 2, &map_k, BAR(kBarFull + 1), 64, kvh, seq_lo + j1 * p.B);
          pre = 2;
        }
      }
      *s_pre = pre;
    }
  } else if (warp == 2) {
    tmem_alloc<kTmemCols>(smem_u32((const void*)s_tmem));
  } else if (warp == 3) {
    // 64-key chunks (token offset of their first key) of the selected blocks that hold a visible key;
    // the index loads of 128 list entries are issued together (one memory latency per 128 entries)
    const int cnt = __ldg(p.count + gb);
    const int32_t* list = p.idx + (int64_t)gb * p.tau_max;
    const int total = cnt * TPB;
    int n = 0;
    for (int base_i = 0; base_i < total; base_i += 128) {
      int jv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base_i + u * 32 + lane;
        jv[u] = (i < total) ? __ldg(list + i / TPB) : -1;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base_i + u * 32 + lane;
        int k0 = -1;
        if (jv[u] >= 0) {
          k0 = seq_lo + jv[u] * p.B + (i % TPB) * 64;
          if (k0 >= seq_hi || (p.causal && k0 > q_last)) k0 = -1;
        }
        const unsigned m = __ballot_sync(0xffffffffu, k0 >= 0);
        if (k0 >= 0) {
          const int pos = n + __popc(m & ((1u << lane) - 1));
          if (pos < kMaxChunks) s_list[pos] = k0;
        }
        n += __popc(m);
      }
    }
    if (lane == 0) *s_nchunks = min(n, kMaxChunks);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  // warp-uniform copies (shfl from lane 0) so that the compiler keeps descriptors and TMA / MMA
  // operands in uniform registers instead of broadcasting them per instruction
  const uint32_t tm = __shfl_sync(0xffffffffu, *s_tmem, 0);
  const int n = __shfl_sync(0xffffffffu, *s_nchunks, 0);

  if (warp < 4) {
  reg_dealloc<64>();
  if (warp == 0) {
    // ===================== TMA producer =====================
    // tile order = consumption order of the MMA warp: K0 K1 V0 K2 V1 K3 ... V(n-1)
    // (the whole warp runs the loop; one elected lane issues the copies)
    if (n > 0) {
      const bool leader = elect_one();
      const int pre = kEarlyK ? __shfl_sync(0xffffffffu, *s_pre, 0) : 0;
      int c = pre;                                       // (stages 0 .. pre-1 were requested during set-up)
      auto push = [&](const CUtensorMap* m, int chunk) {
        const int st = c % kStages;
        mbar_wait(BAR(kBarEmpty + st), ((c / kStages) & 1) ^ 1);
        const int k0 = __shfl_sync(0xffffffffu, s_list[chunk], 0);
        if (leader) {
          mbar_arrive_expect_tx(BAR(kBarFull + st), kTileBytes);
          const uint32_t dst = sKV + st * kTileBytes;
          tma_load_3d(dst, m, BAR(kBarFull + st), 0, kvh, k0);
          tma_load_3d(dst + kTileBytes / 2, m, BAR(kBarFull + st), 64, kvh, k0);
        }
        __syncwarp();
        ++c;
      };
      if (pre < 1) push(&map_k, 0);
      if (n > 1 && pre < 2) push(&map_k, 1);
      for (int k = 0; k < n; ++k) {
        push(&map_v, k);
        if (k + 2 < n) push(&map_k, k + 2);
      }
    } else {
      mbar_wait(BAR(kBarQ), 0);          // nothing to attend to: let the early Q load land before exit
    }
  } else if (warp == 1 || (warp == 3 && kTiles == 2)) {
    // ===================== MMA issuers: warp 1 -> tile 0, warp 3 -> tile 1 =====================
    // One issuing warp per tile: the barrier waits of one tile overlap the tensor work of the other
    // (tcgen05.mma issue blocks while the pipe's short queue is full, so a single issuing warp exposes
    // every wait).  Warp-uniform control flow; one elected lane issues tcgen05.mma / tcgen05.commit.
    if (n > 0) {
      const int t = warp >> 1;
      const bool leader = elect_one();
      const uint32_t id_qk = idesc_bf16(128, 64, 0, 0);
      const uint32_t id_pv = idesc_bf16(128, 128, 0, 1);
      const uint32_t t_sp = tm + t * 128, t_acc = tm + kTiles * 128 + t * 128;
      const uint32_t sQt = sQ + t * 16384;
      int c = 0;
      auto next_tile = [&](int& stage) -> uint32_t {       // waits for the next tile of the ring
        stage = c % kStages;
        mbar_wait(BAR(kBarFull + stage), (c / kStages) & 1);
        ++c;
        return sKV + stage * kTileBytes;
      };
      auto issue_qk = [&](int buf, uint32_t sK, int stage) {
        if (leader) {
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint32_t a = sQt + (kk >> 2) * (kQBytes / 2) + (kk & 3) * 32;
            const uint32_t b = sK + (kk >> 2) * (kTileBytes / 2) + (kk & 3) * 32;
            mma_ss(t_sp + buf * 64, desc_kmajor_sw128(a), desc_kmajor_sw128(b), id_qk, kk > 0);
          }
          mma_commit(BAR(kBarS + t * 2 + buf));
          mma_commit(BAR(kBarEmpty + stage));
        }
        __syncwarp();
      };
      auto issue_pv = [&](int buf, uint32_t sV, bool acc, int stage) {
        if (leader) {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
            mma_ts(t_acc, t_sp + buf * 64 + kk * 8, desc_mnmajor_sw128(sV + kk * 2048, kTileBytes / 2, 1024),
                   id_pv, (acc || kk > 0) ? 1u : 0u);
          mma_commit(BAR(kBarO + t));
          mma_commit(BAR(kBarEmpty + stage));
        }
        __syncwarp();
      };
      mbar_wait(BAR(kBarQ), 0);
      for (int k = 0; k < 2 && k < n; ++k) {
        int st;
        const uint32_t sK = next_tile(st);
        tc_fence_after();
        issue_qk(k, sK, st);
      }
      for (int k = 0; k < n; ++k) {
        const int buf = k & 1, ph = (k >> 1) & 1;
        const bool more = k + 2 < n;
        // one combined wait: lane 0 on P(k), lane 1 on the V(k) tile, lane 2 on the K(k+2) tile, so the
        // three barrier latencies overlap instead of adding up on the issue path
        const int sv = c % kStages, pv = (c / kStages) & 1;
        const int sk = (c + 1) % kStages, pk = ((c + 1) / kStages) & 1;
        c += more ? 2 : 1;
        uint32_t w_bar = 0, w_par = 0;
        if (lane == 0) { w_bar = BAR(kBarP + t * 2 + buf); w_par = ph; }
        if (lane == 1) { w_bar = BAR(kBarFull + sv); w_par = pv; }
        if (lane == 2 && more) { w_bar = BAR(kBarFull + sk); w_par = pk; }
        {
          SW_WATCHDOG_DECL;
          while (true) {
            const bool ok = (w_bar == 0) || mbar_try_wait(w_bar, w_par);
            if (__all_sync(0xffffffffu, ok)) break;
            SW_WATCHDOG_TICK;
          }
        }
        tc_fence_after();
        issue_pv(buf, sKV + sv * kTileBytes, k > 0, sv);
        if (more) issue_qk(buf, sKV + sk * kTileBytes, sk);
      }
      if (leader) mma_commit(BAR(kBarDone));
      __syncwarp();
    }
  }
  } else {
    reg_alloc<kTiles == 2 ? 200 : 192>();
    // ===================== softmax + epilogue: one thread per query row =====================
    const int t = (warp - 4) >> 2;                       // MMA tile
    const int w4 = warp & 3;                             // TMEM lane quadrant of this warp
    const int row = w4 * 32 + lane;                      // row in the tile
    const int q_pos = q_tok0 + t * 32 + (row >> 2);      // global token index of this row
    const int head = kvh * 4 + (row & 3);
    const uint32_t t_s = tm + ((uint32_t)(w4 * 32) << 16) + t * 128;
    const uint32_t t_o = tm + ((uint32_t)(w4 * 32) << 16) + kTiles * 128 + t * 128;
    float m_run = -INFINITY, l_run = 0.f;
    const float c = p.scale_log2;
    const float2 c2 = make_float2(c, c);

    for (int k = 0; k < n; ++k) {
      const int buf = k & 1, ph = (k >> 1) & 1;
      mbar_wait(BAR(kBarS + t * 2 + buf), ph);
      tc_fence_after();
      uint32_t s[64];
      tmem_ld32(t_s + buf * 64, *reinterpret_cast<uint32_t(*)[32]>(&s[0]));
      tmem_ld32(t_s + buf * 64 + 32, *reinterpret_cast<uint32_t(*)[32]>(&s[32]));
      tmem_wait_ld();
      // masks: only chunks that touch the diagonal or the end of the sequence
      {
        const int k0 = s_list[k];
        const bool need = (p.causal && k0 + 63 > q_tok0) || (k0 + 64 > seq_hi);
        if (need) {
          const int lim = min(p.causal ? q_pos : 0x7fffffff, seq_hi - 1) - k0;   // visible iff col <= lim
#pragma unroll
          for (int i = 0; i < 64; ++i)
            if (i > lim) s[i] = 0xff800000u;
        }
      }
      float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
      for (int i = 0; i < 64; i += 8) {
        mx0 = fmax3(mx0, __uint_as_float(s[i]), __uint_as_float(s[i + 1]));
        mx1 = fmax3(mx1, __uint_as_float(s[i + 2]), __uint_as_float(s[i + 3]));
        mx2 = fmax3(mx2, __uint_as_float(s[i + 4]), __uint_as_float(s[i + 5]));
        mx3 = fmax3(mx3, __uint_as_float(s[i + 6]), __uint_as_float(s[i + 7]));
      }
      const float m_tile = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c;      // c > 0
      // lazy rescale
      float m_new = m_run;
      const bool grow = m_tile > m_run + kRescaleThreshold;   // also true for the first finite tile
      if (grow) m_new = m_tile;
      if (k > 0 && __any_sync(0xffffffffu, grow)) {
        const float f = (m_new == m_run) ? 1.f : ex2(m_run - m_new);   // m_run = -inf -> 0
        l_run *= f;
        mbar_wait(BAR(kBarO + t), (k - 1) & 1);           // PV(k-1) of this tile has landed in O
        tc_fence_after();
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
      const float2 nm2 = make_float2(-m_use, -m_use);
      float2 sum0 = make_float2(0.f, 0.f), sum1 = make_float2(0.f, 0.f);
      uint32_t pk[32];
      // the column pairs of SW_POLY_MASK go through the FMA-pipe polynomial (ex2_poly2) instead of MUFU ex2
#pragma unroll
      for (int i = 0; i < 32; i += 2) {
        const float2 x0 = __ffma2_rn(make_float2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), c2, nm2);
        const float2 x1 = __ffma2_rn(make_float2(__uint_as_float(s[2 * i + 2]), __uint_as_float(s[2 * i + 3])), c2, nm2);
        const float2 e0 = use_poly(i) ? ex2_poly2(x0) : make_float2(ex2(x0.x), ex2(x0.y));
        const float2 e1 = use_poly(i + 1) ? ex2_poly2(x1) : make_float2(ex2(x1.x), ex2(x1.y));
        sum0 = __fadd2_rn(sum0, e0);
        sum1 = __fadd2_rn(sum1, e1);
        pk[i] = pack_bf16(e0.x, e0.y);
        pk[i + 1] = pack_bf16(e1.x, e1.y);
      }
      l_run += (sum0.x + sum0.y) + (sum1.x + sum1.y);
      tmem_st32(t_s + buf * 64, pk);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(BAR(kBarP + t * 2 + buf));
    }

    // epilogue: O / l -> bf16 -> global
    if (n > 0) {
      mbar_wait(BAR(kBarDone), 0);
      tc_fence_after();
    }
    const int n_iter = n;
    // a row that never saw a visible key is 0 (ex2_poly2 returns 2^-125, not 0, for a masked column)
    if (m_run == -INFINITY) l_run = 0.f;
    const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
    const bool valid = q_pos <= q_last;
    const int64_t o_off = ((int64_t)q_pos * p.h_q + head) * 128;
    __nv_bfloat16* op = reinterpret_cast<__nv_bfloat16*>(p.out) + o_off;
    float* opf = reinterpret_cast<float*>(p.out) + o_off;
    // A full 32-token tile goes out as bf16 through shared memory (the Q buffer is free once every
    // MMA has completed) and one TMA store per d-half: row-per-thread global stores took ~6000 cycles
    // per CTA.  Ragged tiles and fp32 output keep the direct stores.
    const bool tile_full = q_tok0 + t * 32 + 31 <= q_last;
    if (n_iter > 0 && tile_full && !p.out_f32) {
      const int R = t * 128 + row;                         // row of the 256-row tile = 4 * token + head
      uint8_t* sO = base + (size_t)R * 128;
#pragma unroll
      for (int ch = 0; ch < 4; ++ch) {
        uint32_t o[32];
        tmem_ld32(t_o + ch * 32, o);
        tmem_wait_ld();
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          uint4 w;
          w.x = pack_bf16(__uint_as_float(o[8 * v + 0]) * inv, __uint_as_float(o[8 * v + 1]) * inv);
          w.y = pack_bf16(__uint_as_float(o[8 * v + 2]) * inv, __uint_as_float(o[8 * v + 3]) * inv);
          w.z = pack_bf16(__uint_as_float(o[8 * v + 4]) * inv, __uint_as_float(o[8 * v + 5]) * inv);
          w.w = pack_bf16(__uint_as_float(o[8 * v + 6]) * inv, __uint_as_float(o[8 * v + 7]) * inv);
          const int c16 = (ch & 1) * 4 + v;                // 16-byte chunk inside the 128-byte row of this d-half
          *reinterpret_cast<uint4*>(sO + (ch >> 1) * (kQBytes / 2) + ((c16 ^ (R & 7)) << 4)) = w;   // SWIZZLE_128B
        }
      }
      fence_proxy_async();
      asm volatile("bar.sync %0, 128;" ::"r"(1 + t) : "memory");
      if (row == 0) {
        tma_store_3d(&map_o, sQ + t * 16384, 0, kvh * 4, q_tok0 + t * 32);
        tma_store_3d(&map_o, sQ + kQBytes / 2 + t * 16384, 64, kvh * 4, q_tok0 + t * 32);
        tma_store_commit();
        tma_store_wait_read<0>();
      }
    } else {
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
    }
    if (p.lse && valid)
      p.lse[(int64_t)q_pos * p.h_q + head] =
          l_run > 0.f ? (m_run + log2f(l_run)) * 0.6931471805599453f : -INFINITY;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc<kTmemCols>(tm);
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
  CUtensorMap mq, mk, mv, mo;
  const bool ok = sm100host::make_map_thd(&mq, a.q, L.total_tokens, a.h_q, 128, a.q_stride_tok, a.q_stride_head, 4, kQTok) &&
                  sm100host::make_map_thd(&mk, a.k, L.total_tokens, a.h_kv, 128, a.k_stride_tok, a.k_stride_head, 1, 64) &&
                  sm100host::make_map_thd(&mv, a.v, L.total_tokens, a.h_kv, 128, a.v_stride_tok, a.v_stride_head, 1, 64);
  if (!ok) return fail(SW_ERR_CUDA, "sw_sparse_attn_prefill: cuTensorMapEncodeTiled failed");
  // output map (bf16 output only): store box = 64 d x 4 heads x 32 tokens = one MMA tile's d-half
  if (a.out_dtype == SW_BF16) {
    if (!sm100host::make_map_thd(&mo, a.out, L.total_tokens, a.h_q, 128, (int64_t)a.h_q * 128, 128, 4, 32))
      return fail(SW_ERR_CUDA, "sw_sparse_attn_prefill: cuTensorMapEncodeTiled failed (output)");
  } else {
    mo = mq;                                   // unused by the fp32 epilogue
  }
  if (int32_t rc = allow_dynamic_smem(attn_prefill_sm100_kernel, kSmemBytes, "sw_sparse_attn_prefill(sm100) smem attribute"))
    return rc;
  Params p;
  p.cu_seqlens = L.cu_seqlens; p.cu_blocks = L.cu_blocks; p.idx = a.idx; p.count = a.count;
  p.out = a.out; p.lse = a.lse; p.out_f32 = (a.out_dtype == SW_F32) ? 1 : 0;
  p.batch = L.batch; p.B = L.block; p.total_slots = L.total_blocks * (L.block / kQTok); p.tau_max = a.tau_max;
  p.h_q = a.h_q; p.causal = (a.flags & SW_CAUSAL) ? 1 : 0;
  p.scale_log2 = a.softmax_scale * 1.4426950408889634f;
  dim3 grid(p.total_slots, a.h_kv);
  count_launch();
  attn_prefill_sm100_kernel<<<grid, kThreads, kSmemBytes, st>>>(mq, mk, mv, mo, p);
  return check_launch("sw_sparse_attn_prefill(sm100)");
}

}  // namespace sw
