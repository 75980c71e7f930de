// sw_sparse_attn_decode_static: the decode attention of attn_decode.cu (Alg. 2 Step 7) for callers
// that cannot hand the library a scratch buffer.
//
// Who that is: code that runs where device memory may not be allocated any more -- a serving loop whose memory
// pool was sized and handed out in full at start-up, a plug-in that is given tensors by its host framework but no
// allocator, a real-time thread for which cudaMalloc (a device-wide synchronising call of unbounded duration) is
// off limits.  Such a caller still owns q, the caches, the block lists and the output; the only thing it lacks is
// the few hundred kilobytes in which the split-KV kernel leaves its partial results for the merge kernel.
//
// Here that scratch is a fixed array in the library's own device image.  It costs SW_STATIC_SCRATCH_BYTES of HBM on
// every GPU on which a kernel of this file's module is loaded, for the life of the process, whether used or not;
// that is why it is modest and why problems that need more are refused instead of served some other way.
#include <mutex>

#include "common.cuh"

namespace {

// The scratch itself.  NOTE for anyone editing the host code below: in host code the identifier g_static_scratch
// is only a handle by which the runtime finds the array; it is NOT a device address.  Passing it (or &g_static_scratch[0])
// to a kernel makes the kernel fault, or, on a system where the GPU can reach host memory, read and write some
// unrelated host bytes without any error.  The device address comes from cudaGetSymbolAddress, below.
static __device__ __align__(256) unsigned char g_static_scratch[SW_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
void* g_scratch_addr[kMaxDevices] = {};   // device address of g_static_scratch on device i (0 = not asked yet)

// Once per device, with that device current: ask the runtime where this device's copy of the array lives.
// (Every device has its own copy at its own address, so the answer cannot be shared between devices.)
int32_t static_scratch(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
    cudaGetLastError();
    return sw::fail(SW_ERR_CUDA, "sw_sparse_attn_decode_static: no current device, or device ordinal >= %d", kMaxDevices);
  }
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (g_scratch_addr[dev] == nullptr) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || p == nullptr) {
      cudaGetLastError();
      return sw::fail(SW_ERR_CUDA, "sw_sparse_attn_decode_static: cudaGetSymbolAddress on device %d: %s", dev,
                      cudaGetErrorString(e));
    }
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return SW_OK;
}

}  // namespace

using namespace sw;

extern "C" SW_API int32_t sw_sparse_attn_decode_static(int32_t batch, int32_t block, const sw_tensor* q,
                                                const sw_tensor* kcache, const sw_tensor* vcache,
                                                int64_t stride_batch, const int32_t* seqlens, const int32_t* idx,
                                                const int32_t* count, int32_t tau_max, float softmax_scale,
                                                void* out, float* lse, sw_stream_t stream) {
  // the argument checks of sw_sparse_attn_decode
  SW_REQUIRE(batch >= 0, SW_ERR_INVALID_ARG, "batch = %d", batch);
  SW_REQUIRE(block == 64 || block == 128, SW_ERR_UNSUPPORTED, "block size %d not in {64,128}", block);
  if (int32_t rc = validate_tensor(q, "q")) return rc;
  if (int32_t rc = validate_tensor(kcache, "kcache")) return rc;
  if (int32_t rc = validate_tensor(vcache, "vcache")) return rc;
  SW_REQUIRE(q->dtype == SW_BF16 && kcache->dtype == SW_BF16 && vcache->dtype == SW_BF16, SW_ERR_UNSUPPORTED,
             "decode attention takes bf16 q and caches");
  SW_REQUIRE(q->d == kcache->d && q->d == vcache->d, SW_ERR_UNSUPPORTED, "head_dim mismatch");
  SW_REQUIRE(kcache->heads == vcache->heads && q->heads % kcache->heads == 0 && q->heads / kcache->heads <= 16,
             SW_ERR_UNSUPPORTED, "GQA group h_q/h_kv = %d/%d must be an integer <= 16", q->heads, kcache->heads);
  SW_REQUIRE(seqlens && idx && count && out, SW_ERR_INVALID_ARG, "NULL argument");
  SW_REQUIRE(tau_max >= 1 && stride_batch % 8 == 0, SW_ERR_INVALID_ARG, "tau_max / stride_batch");
  if (int32_t rc = check_arch()) return rc;
  // the one extra rule: the partials must fit the fixed array
  const size_t need = decode_ws_bytes(batch, q->heads, q->d, decode_num_splits(batch, kcache->heads, tau_max, q->d));
  SW_REQUIRE(need <= (size_t)SW_STATIC_SCRATCH_BYTES, SW_ERR_WORKSPACE,
             "sw_sparse_attn_decode_static: this problem needs %zu bytes of scratch, the built-in array holds %zu "
             "(SW_STATIC_SCRATCH_BYTES); use sw_sparse_attn_decode with a caller-owned workspace",
             need, (size_t)SW_STATIC_SCRATCH_BYTES);
  if (batch == 0) return SW_OK;
  void* scratch = nullptr;
  if (int32_t rc = static_scratch(&scratch)) return rc;
  // Nothing in the array has to be cleared between calls: the split-KV kernel writes every (sequence, head, split)
  // slot the merge kernel reads, empty splits included (as m = -inf, l = 0), before the merge kernel starts.
  return launch_attn_decode(batch, block, *q, *kcache, *vcache, stride_batch, seqlens, idx, count, tau_max,
                            softmax_scale, out, lse, scratch, (size_t)SW_STATIC_SCRATCH_BYTES, nullptr, 0,
                            (cudaStream_t)stream);
}
