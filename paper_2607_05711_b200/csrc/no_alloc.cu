// no_alloc.cu -- ft_quantize_blockwise_static: the fused quantize + down-projection pass (a0 + a1 / a3)
// for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving loops, harnesses
// that forbid cudaMalloc).  The pass needs scratch -- control words (tensor amax, grid barrier, exit counter) and the
// fp32 partial-H slots that k_finalize_h sums -- which ft_quantize_blockwise takes from a caller-allocated workspace.
// Here the scratch is a file-scope device array of FT_STATIC_SCRATCH_BYTES (8 MiB): every GPU that loads the library
// holds it until the process exits.  The kernels are the same (launch_quantize_fused), so are the results.
//
// In host code `g_static_scratch` is a host-side stand-in for the symbol, NOT a device address: the device address
// comes from cudaGetSymbolAddress, once per device, with that device current (below), and that pointer is what the
// kernels get.
//
// Every call on a device shares the one array, and the array keeps what the last call left: the control words are
// cleared at the start of every call (a memset node on the caller's stream), the slots are fully written before they
// are read.  Two calls that overlap on the GPU (different streams, no dependency) RACE on the array: serialise them.
#include "common.cuh"

namespace ft {

int device_check();
int launch_quantize_fused(const void* x, int64_t rows, int64_t cols, const float* amax_t, const ft_proj* proj,
                          ft_qtensor* out, void* workspace, bool after_kernel, bool* finalize_last,
                          const SumJob* side_job, cudaStream_t st);

constexpr size_t STATIC_SCRATCH_BYTES = (size_t)8 << 20;
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

// what one call touches: control words, (unused) Hs region, one slot per CTA and row tile (common.cuh: ws_layout)
static size_t static_scratch_needed(int64_t rows, int r_t) { return ws_layout(rows, r_t).wg_off; }

// device address of the array on the CURRENT device, looked up once per device
static int static_scratch_ptr(void** out) {
  static void* ptrs[FT_MAX_DEVICES] = {};
  int dev = 0;
  FT_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= FT_MAX_DEVICES) return FT_ERR_INVALID_ARG;
  if (ptrs[dev] == nullptr) {
    void* p = nullptr;
    FT_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
    if (p == nullptr) return FT_ERR_CUDA;
    ptrs[dev] = p;   // racing first callers store the same value
  }
  *out = ptrs[dev];
  return FT_OK;
}

}  // namespace ft

using namespace ft;

extern "C" {

size_t ft_static_scratch_bytes(void) { return STATIC_SCRATCH_BYTES; }

size_t ft_static_scratch_needed(int64_t rows, int32_t r_t) {
  if (rows < 1 || r_t < 0) return 0;
  return static_scratch_needed(rows, r_t);
}

int ft_quantize_blockwise_static(const void* x_bf16, int64_t rows, int64_t cols, const float* tensor_amax,
                                 const ft_proj* proj, ft_qtensor* out, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  if (!x_bf16 || !out || !out->codes || !out->sf || !out->tensor_dec_scale) return FT_ERR_INVALID_ARG;
  if (out->block_rows != 1 || (out->sf_layout != FT_SF_ROWMAJOR && out->sf_layout != FT_SF_TILE128x4))
    return FT_ERR_INVALID_ARG;
  if (out->rows != rows || out->cols != cols) return FT_ERR_INVALID_ARG;
  if (rows < 1 || cols < 64 || cols % 64 != 0) return FT_ERR_UNSUPPORTED_SHAPE;
  if (!aligned16(x_bf16) || !aligned16(out->codes) || (reinterpret_cast<uintptr_t>(out->sf) & 3)) return FT_ERR_INVALID_ARG;
  int r_t = 0;
  if (proj) {
    r_t = proj->r_t;
    if (r_t < 16 || r_t > 128 || r_t % 16 != 0) return FT_ERR_UNSUPPORTED_SHAPE;
    if (!proj->down || !aligned16(proj->down)) return FT_ERR_INVALID_ARG;
    if (proj->out && !aligned16(proj->out)) return FT_ERR_INVALID_ARG;
    if (proj->out_scaled && (!aligned16(proj->out_scaled) || !proj->other_dec_scale)) return FT_ERR_INVALID_ARG;
  }
  // beyond the static array: refused on the host, nothing is launched (the caller falls back to
  // ft_quantize_blockwise with a workspace of its own)
  if (static_scratch_needed(rows, r_t) > STATIC_SCRATCH_BYTES) return FT_ERR_WORKSPACE_TOO_SMALL;
  int rc = device_check();
  if (rc != FT_OK) return rc;
  void* scratch = nullptr;
  rc = static_scratch_ptr(&scratch);
  if (rc != FT_OK) return rc;
  // the control words must be zero when the kernels start; the array is shared and keeps the last call's contents
  FT_CUDA_TRY(cudaMemsetAsync(scratch, 0, WS_CTL_BYTES, st));
  return launch_quantize_fused(x_bf16, rows, cols, tensor_amax, proj, out, scratch, false, nullptr, nullptr, st);
}

}  // extern "C"
