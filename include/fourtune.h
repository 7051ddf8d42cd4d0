/* fourtune.h -- C ABI of the B200 (sm_100a) W4A4G4 triple-branch linear layer.
 *
 * The operation is the hot path of FourTune (arxiv 2607.05711); citations are
 * lines of PAPER.md plus the section / equation they fall in, and readings
 * Q1..Q5 / O-n of DESIGN.md where the paper is silent.
 *
 *   forward  (sec. 3.1, Eq. 2 recovered from Eq. 3):
 *       Y  = GEMM4(Q(X), Q(R)) + X L1 L2 + X A B
 *   dgrad    (sec. 3.2, Eq. 3):
 *       dX = GEMM4(Q(G), Q(R)^T) + G L_stab^T + G (A B)^T
 *   wgrad    (Eq. 4):   dB = (X A)^T G ,  dA = X^T (G B^T)
 *   Q(.) is the NVFP4 block quantizer: E2M1 codes, one
 *   E4M3 scale per block, one FP32 scale per tensor (Q1-Q5).
 *
 * Shapes:  X [M x K], G and Y [M x N], R [N x K].
 * The two low-rank factors are stored "feature-major":
 *       D_f = [L1 | A]        : [K x r_t]   (row k, r_t contiguous)
 *       U_t = [L2 ; B]^T      : [N x r_t]   (row n, r_t contiguous)
 * r_t = r_s + r; columns 0..r_s-1 are the frozen stabilizer, r_s..r_t-1 the
 * trainable LoRA adapter.  With this storage forward and backward are the same
 * kernels with (X, K, D_f, U_t) and (G, N, U_t, D_f) swapped.
 *
 * Conventions for EVERY call
 *  - all data pointers are DEVICE pointers unless the comment says "host";
 *    the structs themselves are host memory, read during the call only.
 *  - the caller owns every buffer; the library never allocates, frees or keeps
 *    a pointer after the call returns.  Scratch comes from `workspace`, a device buffer of at least
 *    ft_workspace_bytes() bytes whose first 4 KB hold control words that must be ZERO when a call starts:
 *    zero-fill the buffer once (or call ft_workspace_init); every call leaves them zero again (the kernels
 *    put each word back when they are done with it), so no clearing runs per call.  One workspace serves any
 *    number of stream-ordered calls of any shapes, but not two calls that run concurrently.
 *  - `stream` is a cudaStream_t passed as void*; all work is enqueued on it and
 *    the call returns without synchronising.  No device scalar is read by the
 *    host (tensor scales stay on the device).
 *  - return value: FT_OK or a negative ft_status; on error nothing (or only
 *    part of the work) was enqueued.  Shapes are validated on the host before
 *    the first launch.  Inputs must be finite (NaN/Inf: undefined results).
 *  - bf16 matrices are row-major and dense (leading dimension = #columns),
 *    16-byte aligned.
 */
#ifndef FOURTUNE_H_
#define FOURTUNE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  FT_OK = 0,
  FT_ERR_INVALID_ARG = -1,       /* NULL pointer, misaligned pointer, bad enum */
  FT_ERR_UNSUPPORTED_SHAPE = -2, /* dimension not a multiple of the block / tile */
  FT_ERR_WORKSPACE_TOO_SMALL = -3,
  FT_ERR_CUDA = -4,              /* a CUDA runtime/driver call failed: see ft_last_cuda_error */
  FT_ERR_ARCH = -5               /* device is not compute capability 10.x */
} ft_status;

/* scale-factor layouts (Q5) */
#define FT_SF_ROWMAJOR 0  /* sf[row / block_rows][col / 16], dense                          */
#define FT_SF_TILE128x4 1 /* per-row scales in 512-byte tiles of 128 rows x 4 blocks, the
                             layout tcgen05.cp moves to tensor memory unchanged:
                             off(r, c) = ((r/128) * ceil(nblk/4) + c/4) * 512
                                         + (r%32)*16 + ((r%128)/32)*4 + c%4
                             rows padded to 128, blocks to 4 (padding bytes are 0).  With
                             block_rows = 16 row r carries the scale of block r/16.      */

#define FT_ROUND_NEAREST_EVEN 0 /* reading O-6: what every layer call uses                                  */
#define FT_ROUND_STOCHASTIC 1   /* reading O-6': the E2M1 codes by stochastic rounding, the
                                   scales unchanged; ft_quantize_blockwise only (see there)              */

/* A quantized tensor Q(T) of a logical [rows x cols] matrix, blocked along cols. */
typedef struct {
  uint8_t* codes;          /* [rows x cols/2]; byte j of a row = element 2j in bits 0-3,
                              element 2j+1 in bits 4-7 (Q5); E2M1, bit 3 = sign (Q1)   */
  uint8_t* sf;             /* E4M3 block scales (Q2), ft_sf_bytes() bytes, layout below  */
  float* tensor_dec_scale; /* one float: g_dec = 1 / (2688 / amax_t)  (Q3)               */
  int64_t rows, cols;
  int32_t block_rows;      /* 1 (activations, gradients) or 16 (weights, 16x16 blocks)  */
  int32_t sf_layout;       /* FT_SF_ROWMAJOR or FT_SF_TILE128x4                          */
  /* optional, weights only (NULL / 0 otherwise): the same scales once more, cut to the GEMM's output-tile
   * width `ntile` (224 or 240, or 192 for the FC1 of ft_mlp_fwd): for row tile nt = row / ntile and K=64 step ks two 512-byte groups -- rows
   * nt*ntile + 0..127 and + 128..ntile-1 of the tile, each in the (r%32)*16 + (r/32)*4 + c%4 order of
   * FT_SF_TILE128x4, rows past the tile or the tensor zero -- at ((nt * cols/64 + ks) * 2 + half) * 512.
   * ft_sf_ntile_bytes() bytes, filled by ft_pack_weight.  With it ft_gemm4 / ft_linear_* may run 256 x ntile
   * tiles, whose block scales have tensor-memory columns of their own. */
  uint8_t* sf_ntile;
  int32_t ntile;
  int32_t reserved_;
} ft_qtensor;

/* Optional low-rank down-projection fused into the quantize pass (PAPER.md:110,
 * "fuse ... quantization and down-projection"):  H = X * down  (fp32 accumulate). */
typedef struct {
  const void* down;          /* bf16 [cols x r_t]                                        */
  void* out;                 /* bf16 [rows x r_t] = bf16(H); may be NULL                 */
  void* out_scaled;          /* bf16 [rows x r_t] = bf16(H * fl(1 / alpha)), alpha = g_dec(this
                                tensor) * *other_dec_scale (O-10'); may be NULL */
  const float* other_dec_scale; /* g_dec of the operand this tensor will meet in GEMM4;
                                required iff out_scaled != NULL                          */
  int32_t r_t;               /* 16..128, multiple of 16                                  */
} ft_proj;

/* Frozen parts of one layer plus the current adapter. */
typedef struct {
  ft_qtensor r_kmajor; /* Q(R)   as [N x K], 16x16 blocks, sf TILE128x4 (forward operand) */
  ft_qtensor r_nmajor; /* Q(R)^T as [K x N]: the SAME codes and scales re-packed
                          (PAPER.md:102), sf TILE128x4 (dgrad operand)                    */
  const void* D_f;     /* bf16 [K x r_t] = [L1 | A]                                       */
  const void* U_t;     /* bf16 [N x r_t] = [L2 ; B]^T                                     */
  int64_t K, N;
  int32_t r_s, r;      /* r_t = r_s + r: 0, or a multiple of 16 up to 128                 */
} ft_layer;

/* ---- a0: tensor amax (Q3).  *amax_out = max |x_i| over n bf16 values.
 * (ft_quantize_blockwise / ft_linear_* with tensor_amax == NULL find the amax themselves: inside
 * the quantize kernel when the tensor fits the SMs' shared memory, with this kernel otherwise.) */
int ft_tensor_amax(const void* x_bf16, int64_t n, float* amax_out, void* stream);

/* ---- a1/a3/a6: Q(.) of DESIGN.md Q3-Q5 (+ optional fused down-projection).
 * x_bf16 [rows x cols]; blocks are out->block_rows x 16 along cols.
 * tensor_amax: device float holding amax_t; NULL => the library computes it: inside the same
 *   kernel (one HBM read of x in total) when x is at most ~29 MB, by an extra pass otherwise.
 *   The fused projection keeps fp32 partial sums of H (one per CTA and 128-row tile) in the
 *   workspace and adds them in a fixed order: the same bits on every run for a given shape.
 *   workspace may be NULL only if tensor_amax != NULL and proj == NULL.
 * proj: NULL => quantize only.  Requires out->block_rows == 1 if non-NULL.
 * Requirements: cols % 64 == 0; rows % 16 == 0 if block_rows == 16; any rows >= 1
 *   otherwise.  out->rows/cols must equal rows/cols.  workspace >= ft_workspace_bytes(rows, cols, 0, r_t).
 * round_mode FT_ROUND_NEAREST_EVEN: seed and offset are ignored.
 * round_mode FT_ROUND_STOCHASTIC (PAPER.md:59 writes Round(W / s) without naming the mode; O-6'):
 *   x_i * enc_b goes to the E2M1 neighbour above with probability (|v| - lo) / (hi - lo), else to the one below:
 *   hi iff u_i * (hi - lo) < |v| - lo, u_i = (word >> 8) * 2^-24 with word = output[idx % 4] of
 *   Philox4x32-10(counter = (lo, hi, 0, 0) of offset + idx / 4, key = (lo, hi) of seed), idx = row * cols + col.
 *   Counter-based: a caller that quantizes a tensor in row slices passes offset + first_row * cols / 4 and gets
 *   the bits of the whole-tensor call.  Requires out->block_rows == 1 and proj == NULL (a plain kernel, not the
 *   fused one: the mode is a variant for gradients, not the hot path). */
int ft_quantize_blockwise(const void* x_bf16, int64_t rows, int64_t cols,
                          const float* tensor_amax, const ft_proj* proj,
                          ft_qtensor* out, int32_t round_mode, uint64_t seed, uint64_t offset,
                          void* workspace, size_t workspace_bytes, void* stream);

/* ---- ft_quantize_blockwise without a caller workspace and without any device allocation: for callers that cannot
 * call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).  The scratch the
 * pass needs (control words + the fp32 partial sums of the fused projection) lives in a static device array of
 * ft_static_scratch_bytes() = 8 MiB inside the library, held by every GPU that loads the library until the process
 * exits.  Same kernels, same results, same arguments as ft_quantize_blockwise with block_rows == 1 and
 * FT_ROUND_NEAREST_EVEN (tensor_amax == NULL: the library finds it).  x, proj->down in; out (codes,
 * sf, tensor_dec_scale), proj->out, proj->out_scaled are the caller's device buffers.
 * Limit: ft_static_scratch_needed(rows, r_t) <= ft_static_scratch_bytes(): any size without a projection; with one,
 *   rows <= 5450 at r_t = 64 (the 4608-token FLUX activations fit), rows <= 27 000 at r_t = 32, never for r_t >= 96
 *   (the partial sums take 192 slots of 128 x r_t floats).  Beyond it the call returns FT_ERR_WORKSPACE_TOO_SMALL
 *   and launches nothing (use ft_quantize_blockwise with a workspace).
 * The call allocates nothing (no cudaMalloc / cudaFree, no allocating library routine); it enqueues one 4 KB memset
 *   node (the control words) and the kernels on `stream`.
 * All calls on a device share the one array: calls that may OVERLAP on the GPU (different streams without a
 *   dependency between them) race on it -- serialise them.  Not interchangeable with a caller workspace inside one
 *   layer call: ft_linear_* still take theirs. */
int ft_quantize_blockwise_static(const void* x_bf16, int64_t rows, int64_t cols, const float* tensor_amax,
                                 const ft_proj* proj, ft_qtensor* out, void* stream);
size_t ft_static_scratch_bytes(void);
size_t ft_static_scratch_needed(int64_t rows, int32_t r_t);

/* ---- a6 helper: build Q(R)^T ([K x N], N contiguous) from Q(R) ([N x K]) by
 * moving nibbles and scales; nothing is re-quantized.
 * r_kmajor: block_rows 16, sf_layout FT_SF_ROWMAJOR (S[N/16][K/16]).
 * Outputs: r_nmajor (codes [K x N/2], sf TILE128x4 over K rows, same tensor scale
 * value copied), and, if r_kmajor_tiled != NULL, the TILE128x4 expansion of the
 * forward operand's scales (its codes/tensor_dec_scale pointers are not written;
 * point them at r_kmajor's buffers).  For each of the two outputs whose sf_ntile is non-NULL and whose ntile
 * is 224, 240 or 192, the tile-cut copy of the scales as well.  N % 64 == 0 and K % 64 == 0. */
int ft_pack_weight(const ft_qtensor* r_kmajor, ft_qtensor* r_kmajor_tiled,
                   ft_qtensor* r_nmajor, void* stream);

/* ---- single-copy weights ("the same 4-bit weights serve forward and backward",
 * :197 one 4-bit copy per layer): codes_t [K x N/2 bytes] = the codes of Q(R)^T rebuilt from r_kmajor->codes
 * ([N x K/2 bytes]) -- the 4-bit elements transposed, nothing re-quantized; the same bytes ft_pack_weight writes to
 * r_nmajor->codes.  A caller that keeps ONE copy of the codes per layer points every layer's r_nmajor.codes at one
 * scratch buffer of max_layers(N K / 2) bytes and calls this before that layer's backward (same stream); the two
 * scale layouts (1/8 of the codes) stay per layer.  The tensor core takes 4-bit operands K-major only, and a
 * transposition inside the dgrad main loop would put ordinary warps and one more hand-off per stage on a chain that
 * runs at the tensor core's rate: a separate HBM-bound pass it is.  N % 64 == 0, K % 64 == 0; both pointers 16-byte aligned. */
int ft_weight_transpose_codes(const ft_qtensor* r_kmajor, uint8_t* codes_t, void* stream);

/* ---- a0+a1+a2: forward.  x_bf16 [M x K] -> y_bf16 [M x N].
 * h_saved_bf16 [M x r_t] receives bf16(X D_f) (columns r_s.. are X A, reused by
 * ft_lora_wgrad); ignored if r_t == 0.
 * qx_scratch: caller-allocated Q(X) buffers (codes M*K/2 bytes, sf
 *   ft_sf_bytes(M, K, FT_SF_TILE128x4), tensor_dec_scale 1 float); filled here,
 *   rows/cols/block_rows/sf_layout are set by the call.
 * Requirements: K % 64 == 0, N % 64 == 0, M >= 1. */
int ft_linear_fwd(const ft_layer* L, const void* x_bf16, int64_t M, void* y_bf16,
                  void* h_saved_bf16, ft_qtensor* qx_scratch, void* workspace,
                  size_t workspace_bytes, void* stream);

/* ---- a0+a3+a4: input gradient.  g_bf16 [M x N] -> dx_bf16 [M x K].
 * p_saved_bf16 [M x r_t] receives bf16(G U_t) (columns r_s.. are G B^T). */
int ft_linear_bwd_dgrad(const ft_layer* L, const void* g_bf16, int64_t M, void* dx_bf16,
                        void* p_saved_bf16, ft_qtensor* qg_scratch, void* workspace,
                        size_t workspace_bytes, void* stream);

/* ---- a2 / a4 alone: out[M x N] = bf16( alpha * ( GEMM4(a, b) + lr_a_scaled * lr_b^T ) ),
 * alpha = *a->tensor_dec_scale * *b->tensor_dec_scale.
 * a: Q(X) [M x K] (block_rows 1), b: Q(R) [N x K]; both sf TILE128x4, K % 64 == 0, N % 64 == 0.
 * lr_a_scaled: bf16 [M x r_t] = bf16(H * fl(1 / alpha)) as written by ft_quantize_blockwise's
 * out_scaled; lr_b: bf16 [N x r_t]; r_t = 0 (both may be NULL) skips the low-rank term.
 * ft_linear_fwd / ft_linear_bwd_dgrad are ft_tensor_amax + ft_quantize_blockwise + this. */
int ft_gemm4(const ft_qtensor* a, const ft_qtensor* b, const void* lr_a_scaled, const void* lr_b,
             int32_t r_t, void* out_bf16, void* stream);

/* ---- a5: LoRA weight gradients (Eq. 4), fp32.
 * dA  [K x r]  = X^T  * P[:, r_s:]      dBt [N x r] = G^T * H[:, r_s:]  (= dB^T)
 * h_saved / p_saved are the [M x r_t] outputs of the two calls above.
 * accumulate: 0 overwrite, 1 add to the existing contents.  Partial sums over slices of M are added in a fixed
 * order (the same bits on every run), over distributed shared memory inside a thread-block cluster: no clear
 * kernel, no atomics on the data. */
int ft_lora_wgrad(const ft_layer* L, const void* x_bf16, const void* g_bf16, int64_t M,
                  const void* h_saved_bf16, const void* p_saved_bf16, float* dA,
                  float* dBt, int32_t accumulate, void* stream);

/* ---- a5 with 4-bit saved activations (O-12'): Eq. 4
 * with the X of dA = X^T (G B^T) taken as dequant(Q(X)) = E2M1(code) * sf * g_dec -- the qx_scratch
 * that ft_linear_fwd filled -- so the caller keeps 0.5625 instead of 2 bytes per activation element
 * between forward and backward (the activation side of PAPER.md:197-207) and may free or reuse x_bf16
 * as soon as ft_linear_fwd has run.
 * qx: Q(X) [M x K], block_rows 1, sf FT_SF_TILE128x4, all three pointers device memory.
 * dBt = G^T * H[:, r_s:] exactly as in ft_lora_wgrad (it never reads X).  Everything else as there.
 * The dequantized operand is exact in bf16 (E2M1 x E4M3 has six significant bits); g_dec multiplies
 * the fp32 sums. */
int ft_lora_wgrad_q4(const ft_layer* L, const ft_qtensor* qx, const void* g_bf16, int64_t M,
                     const void* h_saved_bf16, const void* p_saved_bf16, float* dA,
                     float* dBt, int32_t accumulate, void* stream);

/* ---- a0+a3+a4+a5 in one call: the whole backward of the layer (Eq. 3 and Eq. 4).
 * Same results as ft_linear_bwd_dgrad followed by ft_lora_wgrad, different schedule: the pass
 * over G that computes dBt = G^T (X A) also finds max |G|, so the separate amax pass of the
 * quantizer disappears (G is read twice instead of three times); dA = X^T (G B^T) runs last
 * because it needs P.  Arguments as in the two calls above. */
int ft_linear_bwd(const ft_layer* L, const void* x_bf16, const void* g_bf16, int64_t M,
                  const void* h_saved_bf16, void* dx_bf16, void* p_saved_bf16, float* dA, float* dBt,
                  int32_t accumulate, ft_qtensor* qg_scratch, void* workspace, size_t workspace_bytes,
                  void* stream);

/* ---- ft_linear_bwd with 4-bit saved activations: the same schedule, dA taken from qx = Q(X) as in
 * ft_lora_wgrad_q4 (O-12').  qx and qg_scratch must be different buffers. */
int ft_linear_bwd_q4(const ft_layer* L, const ft_qtensor* qx, const void* g_bf16, int64_t M,
                     const void* h_saved_bf16, void* dx_bf16, void* p_saved_bf16, float* dA, float* dBt,
                     int32_t accumulate, ft_qtensor* qg_scratch, void* workspace, size_t workspace_bytes,
                     void* stream);

/* ---- NEXT-1, MLP fusion (sec. 3.3 "MLP Fusion"; reading O-16): the forward of
 * FC1 -> GeLU -> FC2 with the FC1 GEMM's epilogue doing GeLU and FC2's quantize + down-projection, so that neither
 * Y1 = FC1(X) nor Z = gelu(Y1) ([M x N1] bf16 each) is written to global memory.
 *   fc1: K -> N1, its r_kmajor.sf_ntile cut to 192-wide tiles (ntile == 192); fc2: N1 -> N2.
 *   x_bf16 [M x K] -> y2_bf16 [M x N2].
 *   z_amax, y1_amax: device floats, the tensor amax the quantizers of Z and of Y1 use (delayed scaling: normally the
 *     value the previous step left in z_amax_next / y1_amax_next; a GEMM epilogue cannot know max |Z| before its
 *     last tile).  z_amax_next, y1_amax_next: device floats (or both NULL) that receive THIS step's max |Z|, max |Y1|.
 *   Outputs kept for backward: h1_saved [M x r_t1] = bf16(X D_f1), h2_saved [M x r_t2] = bf16(Z D_f2),
 *     qx = Q(X), qz = Q(Z) (FC2's activation operand; its dA uses it, ft_linear_bwd_q4), qy1 = Q(Y1) (the
 *     pre-activation, consumed by ft_gelu_bwd_q4); all three caller-allocated like qx_scratch of ft_linear_fwd.
 *   z_debug_bf16, y1_debug_bf16: NULL, or both [M x N1] bf16 buffers that receive copies of Z and Y1 (parity tests:
 *     the staged comparison of DESIGN.md O-11 needs the bits the quantizers consumed).
 *   workspace >= ft_mlp_workspace_bytes(M, K, N1, r_t1, r_t2), control words zero (as for every call).
 * Requirements: K % 64 == 0, N1 % 192 == 0, N2 % 64 == 0, 16 <= r_t2 <= 112, fc1->N == fc2->K == N1.
 * The GeLU is the tanh form evaluated in fp32 on bf16(Y1), as y sigmoid(2 t) with the hardware's exp2 and
 * reciprocal approximations (2^-22 relative); Z = bf16(gelu). */
int ft_mlp_fwd(const ft_layer* fc1, const ft_layer* fc2, const void* x_bf16, int64_t M,
               const float* z_amax, const float* y1_amax, float* z_amax_next, float* y1_amax_next,
               void* y2_bf16, void* h1_saved_bf16, void* h2_saved_bf16,
               ft_qtensor* qx, ft_qtensor* qz, ft_qtensor* qy1, void* z_debug_bf16, void* y1_debug_bf16,
               void* workspace, size_t workspace_bytes, void* stream);
size_t ft_mlp_workspace_bytes(int64_t M, int64_t K, int64_t N1, int32_t r_t1, int32_t r_t2);
/* Byte offset of FC2's pre-scaled intermediate Hs2 [M x r_t2] inside the workspace of ft_mlp_fwd (FC1's Hs1 is at
 * ft_workspace_hs_offset(M, r_t1)). */
size_t ft_mlp_workspace_hs2_offset(int64_t M, int32_t r_t1);

/* ---- GeLU backward of the fused MLP: dy1_bf16 [M x N1] = bf16( dz_bf16 * gelu'(dequant(qy1)) ), qy1 = the Q(Y1)
 * ft_mlp_fwd saved (reading O-16).  dz and dy1 may be the same buffer. */
int ft_gelu_bwd_q4(const void* dz_bf16, const ft_qtensor* qy1, void* dy1_bf16, void* stream);

/* ---- sizes and diagnostics (host only, no CUDA calls) */
size_t ft_sf_bytes(int64_t rows, int64_t cols, int32_t block_rows, int32_t layout);
size_t ft_sf_ntile_bytes(int64_t rows, int64_t cols, int32_t ntile);   /* ft_qtensor::sf_ntile */
/* The tile width worth packing ft_qtensor::sf_ntile for, for a weight operand [N x K] that will meet M tokens
 * (with a low-rank term of rank r_t): 224 or 240, or 0 if the GEMM will use its 256-wide tiles anyway (which need
 * no tile-cut scales).  Host only (the library's cost model of its own schedule on the current device); any of the
 * three choices gives the same results, only the speed differs. */
int32_t ft_gemm_best_ntile(int64_t M, int64_t N, int64_t K, int32_t r_t);
size_t ft_workspace_bytes(int64_t M, int64_t K, int64_t N, int32_t r_t);
/* Zero the control words at the head of a workspace (one 4 KB memset on `stream`).  Needed once per buffer,
 * before its first use, unless the caller zero-filled it; never per call.  Also the way to recover a workspace
 * after a call was aborted by a CUDA error. */
int ft_workspace_init(void* workspace, size_t workspace_bytes, void* stream);
/* Byte offset, inside the workspace handed to ft_linear_fwd / ft_linear_bwd_dgrad / ft_linear_bwd, of the
 * pre-scaled low-rank intermediate Hs = bf16(H * fl(1 / alpha)) [M x r_t] that the quantize pass leaves for
 * the GEMM (O-10'); valid from the call's completion until the next call that uses the
 * workspace.  Exported so that the staged comparison of DESIGN.md O-11 can read the bits the GEMM consumed. */
size_t ft_workspace_hs_offset(int64_t M, int32_t r_t);
const char* ft_error_string(int status);
int ft_last_cuda_error(void); /* cudaError_t / CUresult of the last FT_ERR_CUDA, thread-local */
int ft_version(void);
#ifdef __cplusplus
}
#endif
#endif /* FOURTUNE_H_ */
