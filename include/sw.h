/*
 * sw.h -- C ABI of libsw: the per-layer hot path of Sketch&Walk Attention
 * (arxiv 2602.07397) on one NVIDIA B200 (sm_100a).
 *
 * Citations are lines of /root/reference/PAPER.md ("PAPER.md:<line>") with the
 * section / algorithm they fall in; "P<n>" are the readings listed in DESIGN.md.
 *
 * Conventions (binding for every call)
 *  - Every entry point is extern "C" and returns an int32 status (SW_OK = 0, negative
 *    = error).  No exception crosses the ABI.  sw_last_error() returns a thread-local,
 *    NUL-terminated description of the last failure on the calling thread.
 *  - OWNERSHIP: the caller owns every buffer (inputs, outputs, workspace).  The library
 *    never allocates or frees device memory, never synchronises the device or the
 *    stream, and launches only on the stream passed in.  Pointers documented "dev" are
 *    device pointers; everything else (structs, scalars) is host memory read during the
 *    call.  Workspace sizes come from sw_workspace_bytes() (pure host function).
 *  - VALIDATION happens on the host before any launch; on error nothing is launched and
 *    outputs are untouched.  There is no CPU fallback and no backend dispatch: on a
 *    device that is not sm_100 every compute call returns SW_ERR_ARCH.
 *  - LAYOUT: token tensors are [tokens, heads, d] with d contiguous (strides in
 *    elements).  A batch of sequences is packed along the token axis (varlen, P16);
 *    sequence s owns tokens [cu_seqlens[s], cu_seqlens[s+1]), blocks
 *    [cu_blocks[s], cu_blocks[s+1]) with b_s = ceil(n_s / B), and a
 *    b_s x b_s row-major matrix at element offset cu_sq[s] of the packed W / A / R
 *    buffers.  Block indices are 0-based and local to their sequence.
 *  - All floating point state of the selection path (sketches, scores, walk) is fp32;
 *    attention operands are bf16 with fp32 accumulation and fp32 online softmax.
 */
#ifndef SW_H_
#define SW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Bumped whenever a signature or a workspace layout changes (101: sw_decode_select takes ws / ws_bytes, the
 * SW_OP_WALK_UPDATE workspace holds the operand images, sw_sparse_attn_decode_static added).  A caller built against
 * another header compares its SW_VERSION with sw_version() of the library it loaded and refuses to run on a mismatch
 * (the Python binding does). */
#define SW_VERSION 101            /* 0.1.1 */

#if defined(__GNUC__)
#define SW_API __attribute__((visibility("default")))
#else
#define SW_API
#endif

typedef void* sw_stream_t;        /* a cudaStream_t (NULL = legacy default stream) */

enum sw_status {
  SW_OK = 0,
  SW_ERR_INVALID_ARG = -1,        /* null pointer, bad shape, r not a power of two <= d, ...  */
  SW_ERR_UNSUPPORTED = -2,        /* dtype / head_dim / block size / feature not implemented  */
  SW_ERR_WORKSPACE = -3,          /* workspace missing or too small                           */
  SW_ERR_CUDA = -4,               /* launch error (text in sw_last_error)                     */
  SW_ERR_ARCH = -5                /* current device is not compute capability 10.x            */
};

enum sw_dtype { SW_BF16 = 0, SW_F32 = 1 };

enum sw_flags {
  SW_CAUSAL = 1,         /* P6: block-causal mask on scores, candidates j <= i, token-causal
                            inside the diagonal block                                         */
  SW_SCORE_SOFTMAX = 2,  /* P5: A = row softmax of the masked scores; off = raw signed scores  */
  SW_POW_MATRIX = 4,     /* P4: (A)^s is the s-fold matrix product; off = element-wise power   */
  SW_FORCE_FIRST = 8,    /* always keep key block 0                          */
  SW_FORCE_LAST = 16,    /* ... and the diagonal ("last") key block of the query block         */
  SW_ROWNORM = 32        /* P9: divide each row of R by its max-abs after the update           */
};
#define SW_DEFAULT_FLAGS (SW_CAUSAL | SW_SCORE_SOFTMAX | SW_FORCE_FIRST | SW_FORCE_LAST | SW_ROWNORM)

enum sw_op {              /* for sw_workspace_bytes */
  SW_OP_SKETCH = 0, SW_OP_BLOCK_SCORES = 1, SW_OP_WALK_UPDATE = 2, SW_OP_SELECT_TOPK = 3,
  SW_OP_ATTN_PREFILL = 4, SW_OP_ATTN_DECODE = 5
};

/* A [tokens, heads, d] tensor in device memory, d contiguous. */
typedef struct {
  const void* ptr;        /* dev; 16-byte aligned                                              */
  int32_t dtype;          /* SW_BF16 | SW_F32                                                  */
  int32_t heads, d;       /* d in {64, 128}                                                    */
  int64_t stride_tok;     /* elements between consecutive tokens (multiple of 8)               */
  int64_t stride_head;    /* elements between consecutive heads  (multiple of 8)               */
} sw_tensor;

/* Packed varlen batch description (host struct; the cu_* arrays live on the device). */
typedef struct {
  int32_t batch;          /* number of sequences                                               */
  int32_t block;          /* B, tokens per block: 64 or 128 (PAPER.md:202 uses 64)             */
  int32_t total_tokens;   /* cu_seqlens[batch]                                                 */
  int32_t total_blocks;   /* cu_blocks[batch]                                                  */
  int32_t max_blocks;     /* max_s b_s                                                         */
  const int32_t* cu_seqlens;  /* dev [batch+1] token offsets                                   */
  const int32_t* cu_blocks;   /* dev [batch+1] block offsets                                   */
  const int64_t* cu_sq;       /* dev [batch+1] element offsets of each b_s x b_s matrix        */
} sw_layout;

/* ---------------------------------------------------------------------------------------
 * (1) Sketch -- Small-World Sketching, Alg. 1 Steps 1-4, sec 2.2
 *     (PAPER.md:55-65), SRHT of Lemma A.6.
 *   xbar_i  = mean over the valid tokens of block i and over all heads of x   (P12, P14)
 *   sketch[i, c] = scale * sum_x xbar_i[x] * signs[x] * (-1)^popcount(x & cols[c])   (P1, P2)
 * x: bf16 or fp32.  signs: dev int8[d] of +-1, NULL = all +1.  cols: dev int32[r], values in
 * [0, d).  r: power of two, 1 <= r <= d.  scale: normally 1/sqrt(r).
 * sketch: dev fp32 [total_blocks, r] (written).  mean: dev fp32 [total_blocks, d] or NULL.
 * ------------------------------------------------------------------------------------- */
SW_API int32_t sw_sketch(const sw_layout* L, const sw_tensor* x, const int8_t* signs, const int32_t* cols,
                  int32_t r, float scale, float* sketch, float* mean, sw_stream_t stream);

/* Q and K of one layer in ONE launch (bit-identical to two sw_sketch calls: the same kernel body, the query
 * blocks first and the key blocks behind them in one grid).  q: [total_tokens, h_q, d], k: [total_tokens, h_kv, d],
 * same dtype and d.  qs / ks: dev fp32 [total_blocks, r] (written).  qbar / kbar: dev fp32 [total_blocks, d] or
 * NULL. */
SW_API int32_t sw_sketch_qk(const sw_layout* L, const sw_tensor* q, const sw_tensor* k, const int8_t* signs,
                     const int32_t* cols, int32_t r, float scale, float* qs, float* ks, float* qbar, float* kbar,
                     sw_stream_t stream);

/* Sketch fused upstream ("custom CUDA kernels for block aggregation").  The
 * token-space sketch is a plain sum, so whatever kernel produces (or copies) Q / K can leave the per-block sums
 * behind and the 10 240 bytes per token that sw_sketch re-reads disappear:
 *   sums[i, x] = sum over the heads and the valid tokens of block i of x[token, head, x]     (Steps 1-3, unscaled)
 * sw_sketch_from_pooled finishes Alg. 1 Steps 3-4 from such sums: divide by heads * (valid
 * tokens of the block) (P12), sign flip, FWHT, column pick, scale -- the same arithmetic as sw_sketch after its
 * pooling loop.  sums: dev fp32 [total_blocks, d]; heads: how many heads were summed; sketch / mean as sw_sketch.
 * sw_copy_pool is one such producer: it copies x (bf16 or fp32, strided) into the packed bf16 tensor dst
 * [total_tokens, heads, d] (a KV-cache append, or the bf16 cast pre-pass of P17) and writes sums as a
 * by-product of the same pass. */
SW_API int32_t sw_sketch_from_pooled(const sw_layout* L, const float* sums, int32_t heads, int32_t d,
                              const int8_t* signs, const int32_t* cols, int32_t r, float scale, float* sketch,
                              float* mean, sw_stream_t stream);
SW_API int32_t sw_copy_pool(const sw_layout* L, const sw_tensor* x, void* dst, float* sums, sw_stream_t stream);

/* Decode form, Alg. 2 Steps 2-3: one new token per sequence.
 * x: [batch, heads, d] (stride_tok = stride between sequences).  seqlens: dev int32[batch],
 * length INCLUDING the new token (t).  Block b_curr = (t-1)/B gets the running mean
 *   mean[b_curr] <- (c * mean[b_curr] + x_avg) / (c + 1),  c = (t-1) mod B
 * mean:   dev fp32 [batch, max_blocks, d]  (in/out, row b_curr updated)
 * sketch: dev fp32 [batch, max_blocks, r]  (in/out, row b_curr recomputed from the new mean)
 * tok_sketch: dev fp32 [batch, r] or NULL: sketch of the head-averaged token itself
 *             (q~_t of PAPER.md:815).  mean/sketch may be NULL when only tok_sketch is wanted. */
SW_API int32_t sw_sketch_append(int32_t batch, int32_t block, int32_t max_blocks, const sw_tensor* x,
                         const int32_t* seqlens, const int8_t* signs, const int32_t* cols, int32_t r,
                         float scale, float* mean, float* sketch, float* tok_sketch,
                         sw_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * (2) Block scores -- Alg. 1 Steps 5-6a, eq. PAPER.md:69.
 *   S = qs ks^T / sqrt(r)                          (P3: divided by sqrt(r) once)
 *   SW_CAUSAL: entries j > i are masked            (P6)
 *   SW_SCORE_SOFTMAX: A[i,:] = softmax of the unmasked S[i,:], masked -> 0; else A = S, masked -> 0
 *   W = A^(element-wise s)   (or W = A with SW_POW_MATRIX: the walk then multiplies s times)
 * qs, ks: dev fp32 [total_blocks, r], 16-byte aligned (SW_ERR_INVALID_ARG otherwise; also for
 * sw_prefill_select).  W: dev fp32 packed sum_s b_s^2 (written in full, zeros
 * where masked).  A: same shape or NULL.  s >= 1.
 * ------------------------------------------------------------------------------------- */
SW_API int32_t sw_block_scores(const sw_layout* L, const float* qs, const float* ks, int32_t r, int32_t s,
                        uint32_t flags, float* W, float* A, sw_stream_t stream);

/* Decode form, Alg. 2 Steps 3-4: the new query row of W for block
 * b_q = (t-1)/B against key blocks 0..b_q of the same sequence.
 * q_tok: dev fp32 [batch, r].  ks: dev fp32 [batch, max_blocks, r].
 * w_row: dev fp32 [batch, max_blocks] (entries > b_q written as 0).  Needs !SW_POW_MATRIX and SW_CAUSAL
 * (SW_ERR_UNSUPPORTED otherwise): all decode row-mode calls are defined under the block-causal mask only.
 * Without it Alg. 2 Step 4(ii) rewrites column b_curr of the cached scores for every
 * earlier query block, which changes the softmax of all those rows; the row-vector form does not carry that
 * (under SW_CAUSAL the column is masked and the update is a no-op, P11). */
SW_API int32_t sw_block_scores_row(int32_t batch, int32_t block, int32_t max_blocks, const float* q_tok,
                            const float* ks, const int32_t* seqlens, int32_t r, int32_t s,
                            uint32_t flags, float* w_row, sw_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * (3) Walk -- Sketch-Determined Walk, sec 2.3 eq. PAPER.md:77, Lemma A.11,
 *     Alg. 1 Step 6.
 *   R_out = R_prev * W        (R_prev = NULL is the identity: R^0 = W^0, P10)
 *   SW_POW_MATRIX: R_out = R_prev * W^s as s successive products (W must then be A)
 *   SW_ROWNORM: each row of R_out is divided by its max-abs (P9)
 *   SW_CAUSAL: both operands are lower triangular; the strictly upper part of R_out is 0.
 * R_prev, W, R_out: dev fp32 packed (cu_sq).  R_out must not alias R_prev or W.
 * ws: dev scratch (128-byte aligned) of sw_workspace_bytes(SW_OP_WALK_UPDATE, ...) bytes = one ping-pong matrix
 * (batch * max_blocks^2 floats; required with SW_POW_MATRIX and s > 1, else SW_ERR_WORKSPACE) followed
 * by the hi/lo operand images of the tensor-core kernel (max_blocks >= 256; any batch: the sequences are
 * stacked with one row pitch, ~4 (total_blocks + 128 (batch + 1)) max_blocks floats).  ws may be NULL or
 * shorter otherwise: the fp32 SIMT kernel then runs (see sw_set_walk_kernel).  Both kernels keep ~fp32
 * accuracy (the tcgen05 one by 3xTF32 splitting).
 * ------------------------------------------------------------------------------------- */
SW_API int32_t sw_walk_update(const sw_layout* L, const float* R_prev, const float* W, int32_t s,
                       uint32_t flags, float* R_out, void* ws, size_t ws_bytes, sw_stream_t stream);

/* Decode form, Alg. 2 Step 5 as a row vector: only row b_q of R is ever
 * consumed by Step 6, and row b_q of R_prev*W depends only on row b_q of R_prev, so
 *   r_out = r_prev * W',   W' = W_cache with row b_q replaced by w_row,  r_prev = NULL -> e_{b_q}.
 * W_cache: dev fp32, sequence s at W_cache + s*stride_seq, row-major [max_blocks, max_blocks]
 * (rows < b_q are read).  w_row, r_prev, r_out: dev fp32 [batch, max_blocks].
 * Cache update of Alg. 2 Step 4 ("update cached A^"): w_row is also stored as row b_q
 * of W_cache (zeros right of the diagonal), so that when the token completes block b_q the cache holds
 * that block's row for the following steps -- the row the literal algorithm leaves behind (P11).
 * Needs SW_CAUSAL (see sw_block_scores_row). */
SW_API int32_t sw_walk_update_row(int32_t batch, int32_t block, int32_t max_blocks, const float* r_prev,
                           float* W_cache, int64_t stride_seq, const float* w_row,
                           const int32_t* seqlens, uint32_t flags, float* r_out, sw_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * (4) Top-tau selection -- Alg. 1 Step 7; first and last key block always
 *     kept.
 *   candidates of query block i: j <= i (SW_CAUSAL) or all j;  budget = min(tau_s, #candidates)
 *   forced = {i} (SW_FORCE_LAST) then {0} (SW_FORCE_FIRST), inside the budget (P7)
 *   the rest = top-(budget - |forced|) of the other candidates by (R[i,j] desc, j asc);
 *   NaN ranks as -inf (P8).  Output ascending.
 * R: dev fp32 packed.  tau: dev int32[batch].  tau_max >= max tau.
 * idx: dev int32 [total_blocks, tau_max] (padded with -1).  count: dev int32 [total_blocks].
 * Bit-exact: comparisons are done on an order-preserving integer image of the fp32 scores.
 * ------------------------------------------------------------------------------------- */
SW_API int32_t sw_select_topk(const sw_layout* L, const float* R, const int32_t* tau, int32_t tau_max,
                       uint32_t flags, int32_t* idx, int32_t* count, sw_stream_t stream);

/* Prefill selection, fused -- Alg. 1 Steps 5-7: exactly the sequence
 *   sw_block_scores(qs, ks -> W, A); sw_walk_update(R_prev, W -> R_out); sw_select_topk(R_out -> idx, count)
 * with the same arguments and the same results up to fp32 summation order, in at most three launches
 * (SURVEY 8(f) item 1): (1) score tiles, row softmax and power in one kernel that keeps a strip of rows on chip
 * and, for the tensor-core walk, writes W directly as the hi / lo TF32 operand images next to the fp32 W (the
 * images of R_prev come from extra CTAs of the same grid); (2) the walk GEMM (tcgen05 3xTF32 for
 * max_blocks >= 512, any batch; fp32 SIMT below), which leaves the raw product in R_out; (3) the per-row
 * max-abs rescale (P9) and the top-tau of the same row in one kernel, in place.  R_prev = NULL: R_out = W
 * (P10) and launch (2) is skipped.  W: dev fp32 packed (written; what a decode cache keeps).  A: optional.
 * ws: as sw_walk_update (sw_workspace_bytes(SW_OP_WALK_UPDATE)); without it the SIMT GEMM runs.  With
 * SW_POW_MATRIX and s > 1 (s successive products) the three plain calls are issued instead. */
SW_API int32_t sw_prefill_select(const sw_layout* L, const float* qs, const float* ks, int32_t r, int32_t s,
                          uint32_t flags, const float* R_prev, float* R_out, float* W, float* A,
                          const int32_t* tau, int32_t tau_max, int32_t* idx, int32_t* count, void* ws,
                          size_t ws_bytes, sw_stream_t stream);

/* Decode form, Alg. 2 Step 6: S = TopK(r[0..b_q), tau-1) U {b_q}, block 0
 * also forced with SW_FORCE_FIRST.  r: dev fp32 [batch, max_blocks].
 * idx: dev int32 [batch, tau_max], count: dev int32 [batch]. */
SW_API int32_t sw_select_topk_row(int32_t batch, int32_t block, int32_t max_blocks, const float* r,
                           const int32_t* seqlens, const int32_t* tau, int32_t tau_max,
                           uint32_t flags, int32_t* idx, int32_t* count, sw_stream_t stream);

/* Decode selection, fused -- Alg. 2 Steps 2-6 in three launches: exactly the sequence
 *   sw_sketch_append(k_new -> kbar, ks); sw_sketch_append(q -> q~_t); sw_block_scores_row;
 *   sw_walk_update_row (with SW_ROWNORM: r_out / max|r_out|, P9); sw_select_topk_row
 * with the same arguments and the same results up to fp32 summation order (the selected indices are
 * bit-exact given the same r_out).  The cached W is read once, by the whole grid whatever the batch.
 * q: [batch, h_q, d], k_new: [batch, h_kv, d] (bf16 or fp32, same dtype).  kbar [batch, max_blocks, d]
 * and ks [batch, max_blocks, r] are updated in place for block b_curr, and the new row of W is stored
 * as row b_q of W_cache (as sw_walk_update_row does), so consecutive decode steps -- across block
 * boundaries too -- need no other cache maintenance than appending K/V.  r_prev (NULL = e_{b_q}),
 * r_out: dev fp32 [batch, max_blocks].  Needs !SW_POW_MATRIX and SW_CAUSAL (see sw_block_scores_row).
 * ws: dev scratch of sw_decode_select_workspace_bytes(batch, max_blocks) bytes (SW_ERR_WORKSPACE if smaller):
 * the raw score row and the partial sums of the W stream, handed from the first kernel to the second (no state is
 * kept between calls; calls that share a workspace must not overlap).  batch <= 512.  seqlens[s] must lie in
 * [1, max_blocks * block]; a value outside that range marks an IDLE SLOT of the batch: nothing of sequence s is read
 * or updated (kbar, ks, W_cache untouched), count[s] = 0, its idx row is -1 and its r_out row 0.  Three launches chained as
 * programmatic dependents: the streaming kernel (the cached-W stream of Step 5 over the whole grid; skipped when
 * r_prev is NULL), beside it the kernel of Steps 2-4 (sketches, running key mean, raw score row), then the
 * per-sequence tail (softmax, W_new, rescale, select).  No kernel of the chain reads anything an earlier kernel of
 * the stream may have written before its griddepcontrol.wait. */
SW_API int32_t sw_decode_select(int32_t batch, int32_t block, int32_t max_blocks, const sw_tensor* q,
                         const sw_tensor* k_new, const int32_t* seqlens, const int8_t* signs,
                         const int32_t* cols, int32_t r, float scale, int32_t s, uint32_t flags,
                         float* kbar, float* ks, float* W_cache, int64_t stride_seq,
                         const float* r_prev, float* r_out, const int32_t* tau, int32_t tau_max,
                         int32_t* idx, int32_t* count, void* ws, size_t ws_bytes, sw_stream_t stream);
SW_API size_t sw_decode_select_workspace_bytes(int32_t batch, int32_t max_blocks);

/* ---------------------------------------------------------------------------------------
 * (5) Block-sparse attention, prefill -- Alg. 1 Step 8; "zero outside selected
 *     blocks, renormalized within".
 *   For q-head u (kv head u / (h_q/h_kv), P14) and query token t of block i:
 *   o_t = softmax_k( q_t . k * softmax_scale ) v  over the tokens k of the blocks idx[i, 0..count[i])
 *   with position(k) <= position(t) when SW_CAUSAL.
 * q: [total_tokens, h_q, d]; k, v: [total_tokens, h_kv, d]; all bf16, or all fp32 (P17: fp32
 * operands are rounded to bf16 by a cast pre-pass into ws).  out: dev, same dtype as q,
 * [total_tokens, h_q, d] contiguous.  lse: dev fp32 [total_tokens, h_q] (natural log) or NULL.
 * idx/count as written by sw_select_topk, or built by the caller: block indices local to the sequence, in any order,
 * each block at most once.  Entries that are -1, lie past the last block of the sequence, or (under SW_CAUSAL) name a
 * block j > i that the mask hides entirely are skipped wherever they stand in the list.
 * ------------------------------------------------------------------------------------- */
SW_API int32_t sw_sparse_attn_prefill(const sw_layout* L, const sw_tensor* q, const sw_tensor* k,
                               const sw_tensor* v, const int32_t* idx, const int32_t* count,
                               int32_t tau_max, float softmax_scale, uint32_t flags, void* out,
                               float* lse, void* ws, size_t ws_bytes, sw_stream_t stream);

/* ---------------------------------------------------------------------------------------
 * (6) Block-sparse attention, decode -- Alg. 2 Step 7: one query token per
 *     sequence against the selected blocks of its KV cache (the last block may be partial),
 *     split over the selected blocks across CTAs and merged by log-sum-exp.
 * q: [batch, h_q, d] bf16.  kcache/vcache: sequence s at ptr + s*stride_batch elements, laid
 * out [t_s, h_kv, d] bf16.  seqlens: dev int32[batch], INCLUDING the new token.
 * idx: dev int32 [batch, tau_max], count: dev int32[batch].  out: dev bf16 [batch, h_q, d].
 * lse: dev fp32 [batch, h_q] or NULL.  ws: sw_workspace_bytes(SW_OP_ATTN_DECODE, ...) bytes.
 * ------------------------------------------------------------------------------------- */
SW_API int32_t sw_sparse_attn_decode(int32_t batch, int32_t block, const sw_tensor* q,
                              const sw_tensor* kcache, const sw_tensor* vcache, int64_t stride_batch,
                              const int32_t* seqlens, const int32_t* idx, const int32_t* count,
                              int32_t tau_max, float softmax_scale, void* out, float* lse,
                              void* ws, size_t ws_bytes, sw_stream_t stream);

/* Paged KV cache: the same computation with K and V in one pool of pages of ``block`` tokens.
 * kpool/vpool: [num_pages * block, h_kv, d] bf16 (page p = tokens [p*block, (p+1)*block)); logical block j of
 * sequence s lives in page block_table[s * table_stride + j] (dev int32; entries of the selected blocks
 * must be valid pages, others are never read).  Selected blocks are gathered page by page, so nothing is
 * copied.  Everything else as sw_sparse_attn_decode. */
SW_API int32_t sw_sparse_attn_decode_paged(int32_t batch, int32_t block, const sw_tensor* q,
                                    const sw_tensor* kpool, const sw_tensor* vpool, int64_t num_pages,
                                    const int32_t* block_table, int32_t table_stride,
                                    const int32_t* seqlens, const int32_t* idx, const int32_t* count,
                                    int32_t tau_max, float softmax_scale, void* out, float* lse,
                                    void* ws, size_t ws_bytes, sw_stream_t stream);

/* sw_sparse_attn_decode for callers that have no device memory to spare for a workspace and no way to get some:
 * a serving process whose memory pool was carved up completely at start-up, a plug-in that receives tensors from
 * its host framework but no allocator, a latency-critical thread that must never reach cudaMalloc (which
 * synchronises the whole device and may take arbitrarily long).  Same arguments, same kernels and bit-identical
 * results as sw_sparse_attn_decode (contiguous cache), minus ws / ws_bytes: the split-KV partials go into a fixed
 * array of SW_STATIC_SCRATCH_BYTES that is part of libsw's device image.  The call allocates and frees nothing
 * (no cudaMalloc / cudaFree, no allocating library routine); q, the caches, the lists and out are still the
 * caller's.
 *  - LIMIT: sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau_max) must be <= SW_STATIC_SCRATCH_BYTES, otherwise
 *    SW_ERR_WORKSPACE is returned (message in sw_last_error) and nothing is launched.  (cfg 3 of BASELINE.json,
 *    batch 8 x 32 heads x d = 128 at tau = 410, needs about 1.2 MB.)
 *  - COST: the array occupies SW_STATIC_SCRATCH_BYTES of device memory on every GPU that loads this part of the
 *    library, until the process exits, used or not.
 *  - FIRST CALL PER DEVICE: the first call made with a given device current looks up that device's address of the
 *    array (cudaGetSymbolAddress; this may load the module on that device).  Make that first call during start-up,
 *    outside any stream capture.
 *  - SHARING: all calls on a device use the same array and it keeps whatever the last call left in it.  Nothing in
 *    it needs clearing (every slot that is read is written first, by the same call), but two calls whose kernels
 *    can be on the GPU at the same time -- different streams, or different host threads -- race on it and give
 *    wrong results without any error.  Keep all calls on one stream, or order them with events. */
#define SW_STATIC_SCRATCH_BYTES (4u << 20)
SW_API int32_t sw_sparse_attn_decode_static(int32_t batch, int32_t block, const sw_tensor* q,
                                     const sw_tensor* kcache, const sw_tensor* vcache, int64_t stride_batch,
                                     const int32_t* seqlens, const int32_t* idx, const int32_t* count,
                                     int32_t tau_max, float softmax_scale, void* out, float* lse,
                                     sw_stream_t stream);

/* Bytes of device scratch ``op`` needs for this problem (pure host functions; 0 = none).
 * SW_OP_WALK_UPDATE: see sw_walk_update.  SW_OP_ATTN_PREFILL: only for
 * dtype = SW_F32 (the bf16 cast copies, P17).  SW_OP_ATTN_DECODE: the split-KV partials
 * (batch = L->batch; or call sw_decode_workspace_bytes without a layout). */
SW_API size_t sw_workspace_bytes(int32_t op, const sw_layout* L, int32_t h_q, int32_t h_kv, int32_t d,
                          int32_t tau_max, int32_t dtype);
SW_API size_t sw_decode_workspace_bytes(int32_t batch, int32_t h_q, int32_t h_kv, int32_t d, int32_t tau_max);

/* Number of KV splits sw_sparse_attn_decode will use (host-only; for reporting). */
SW_API int32_t sw_decode_num_splits(int32_t batch, int32_t h_kv, int32_t d, int32_t tau_max);

/* Kernel choice of sw_sparse_attn_prefill (process-wide; for tests and benchmarks -- both kernels
 * are CUDA kernels of this library, there is no non-GPU path).
 *   SW_PREFILL_AUTO (default): the tcgen05/TMEM/TMA kernel when the problem fits it (d = 128, bf16
 *                    or cast fp32 operands, h_q = 4 h_kv), else the generic mma.sync kernel.
 *   SW_PREFILL_GENERIC: always the generic kernel.
 *   SW_PREFILL_TCGEN05: the tcgen05 kernel; sw_sparse_attn_prefill returns SW_ERR_UNSUPPORTED when
 *                    the problem does not fit it.
 * Returns the previous setting, or SW_ERR_INVALID_ARG for an unknown value (setting unchanged).
 * sw_get_prefill_kernel_used(): which kernel the last sw_sparse_attn_prefill of this thread launched
 * (SW_PREFILL_GENERIC / SW_PREFILL_TCGEN05; 0 = none yet). */
enum sw_prefill_kernel { SW_PREFILL_AUTO = 0, SW_PREFILL_GENERIC = 1, SW_PREFILL_TCGEN05 = 2 };
SW_API int32_t sw_set_prefill_kernel(int32_t which);
SW_API int32_t sw_get_prefill_kernel_used(void);

/* Kernel choice of sw_walk_update (process-wide; for tests and benchmarks -- both are CUDA kernels of
 * this library).
 *   SW_WALK_AUTO (default): the tcgen05 3xTF32 GEMM when max_blocks >= 512 and the workspace holds its
 *                    operand images, else the fp32 SIMT GEMM.
 *   SW_WALK_SIMT: always the SIMT kernel.
 *   SW_WALK_TCGEN05: the tcgen05 kernel (max_blocks >= 256); SW_ERR_UNSUPPORTED / SW_ERR_WORKSPACE when the
 *                    problem or the workspace does not fit it.
 * Returns the previous setting, or SW_ERR_INVALID_ARG.  sw_get_walk_kernel_used(): the kernel the last
 * sw_walk_update of this thread launched (SW_WALK_SIMT / SW_WALK_TCGEN05; 0 = none yet). */
enum sw_walk_kernel { SW_WALK_AUTO = 0, SW_WALK_SIMT = 1, SW_WALK_TCGEN05 = 2 };
SW_API int32_t sw_set_walk_kernel(int32_t which);
SW_API int32_t sw_get_walk_kernel_used(void);

SW_API const char* sw_last_error(void);
SW_API int32_t sw_version(void);
/* Number of CUDA kernels this library has launched in the calling process so far (all streams, all calls).
 * Host-only counter for benchmarks that report how many of the library's kernels a timed region ran. */
SW_API uint64_t sw_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SW_H_ */
