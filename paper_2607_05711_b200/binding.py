"""Thin Python binding of include/fourtune.h: argument marshalling only.  Every step of
the hot path runs in the CUDA kernels of libfourtune.so; PyTorch supplies device memory and
the stream.  There is no CPU fallback: a missing library raises at import of the symbols.

Function names and argument order follow the C header.  Tensors are torch CUDA tensors;
`QTensor` / `Layer` mirror ft_qtensor / ft_layer.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfourtune.so")

FT_SF_ROWMAJOR, FT_SF_TILE128x4 = 0, 1
FT_ROUND_NEAREST_EVEN, FT_ROUND_STOCHASTIC = 0, 1


class FtError(RuntimeError):
    pass


class _QT(C.Structure):
    _fields_ = [("codes", C.c_void_p), ("sf", C.c_void_p), ("tensor_dec_scale", C.c_void_p),
                ("rows", C.c_int64), ("cols", C.c_int64), ("block_rows", C.c_int32), ("sf_layout", C.c_int32),
                ("sf_ntile", C.c_void_p), ("ntile", C.c_int32), ("reserved_", C.c_int32)]


class _Proj(C.Structure):
    _fields_ = [("down", C.c_void_p), ("out", C.c_void_p), ("out_scaled", C.c_void_p),
                ("other_dec_scale", C.c_void_p), ("r_t", C.c_int32)]


class _Layer(C.Structure):
    _fields_ = [("r_kmajor", _QT), ("r_nmajor", _QT), ("D_f", C.c_void_p), ("U_t", C.c_void_p),
                ("K", C.c_int64), ("N", C.c_int64), ("r_s", C.c_int32), ("r", C.c_int32)]


_lib = None


def lib():
    """Load libfourtune.so (building it is `python -m paper_2607_05711_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FtError("libfourtune.so not built: run `python -m paper_2607_05711_b200.build` "
                          "(there is no fallback path)")
        L = C.CDLL(LIB_PATH)
        vp, i64, i32, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_size_t
        L.ft_tensor_amax.argtypes = [vp, i64, vp, vp]
        L.ft_quantize_blockwise.argtypes = [vp, i64, i64, vp, C.POINTER(_Proj), C.POINTER(_QT), i32, C.c_uint64, C.c_uint64,
                                            vp, sz, vp]
        L.ft_pack_weight.argtypes = [C.POINTER(_QT), C.POINTER(_QT), C.POINTER(_QT), vp]
        L.ft_quantize_blockwise_static.argtypes = [vp, i64, i64, vp, C.POINTER(_Proj), C.POINTER(_QT), vp]
        L.ft_static_scratch_bytes.restype = sz
        L.ft_static_scratch_needed.argtypes = [i64, i32]
        L.ft_static_scratch_needed.restype = sz
        L.ft_weight_transpose_codes.argtypes = [C.POINTER(_QT), vp, vp]
        L.ft_linear_fwd.argtypes = [C.POINTER(_Layer), vp, i64, vp, vp, C.POINTER(_QT), vp, sz, vp]
        L.ft_linear_bwd_dgrad.argtypes = [C.POINTER(_Layer), vp, i64, vp, vp, C.POINTER(_QT), vp, sz, vp]
        L.ft_gemm4.argtypes = [C.POINTER(_QT), C.POINTER(_QT), vp, vp, i32, vp, vp]
        L.ft_lora_wgrad.argtypes = [C.POINTER(_Layer), vp, vp, i64, vp, vp, vp, vp, i32, vp]
        L.ft_lora_wgrad_q4.argtypes = [C.POINTER(_Layer), C.POINTER(_QT), vp, i64, vp, vp, vp, vp, i32, vp]
        L.ft_linear_bwd.argtypes = [C.POINTER(_Layer), vp, vp, i64, vp, vp, vp, vp, vp, i32, C.POINTER(_QT), vp, sz, vp]
        L.ft_linear_bwd_q4.argtypes = [C.POINTER(_Layer), C.POINTER(_QT), vp, i64, vp, vp, vp, vp, vp, i32, C.POINTER(_QT), vp, sz, vp]
        L.ft_sf_bytes.argtypes = [i64, i64, i32, i32]
        L.ft_sf_bytes.restype = sz
        L.ft_mlp_fwd.argtypes = [C.POINTER(_Layer), C.POINTER(_Layer), vp, i64, vp, vp, vp, vp, vp, vp, vp, C.POINTER(_QT),
                                 C.POINTER(_QT), C.POINTER(_QT), vp, vp, vp, sz, vp]
        L.ft_mlp_workspace_bytes.argtypes = [i64, i64, i64, i32, i32]
        L.ft_mlp_workspace_bytes.restype = sz
        L.ft_mlp_workspace_hs2_offset.argtypes = [i64, i32]
        L.ft_mlp_workspace_hs2_offset.restype = sz
        L.ft_gelu_bwd_q4.argtypes = [vp, C.POINTER(_QT), vp, vp]
        L.ft_sf_ntile_bytes.argtypes = [i64, i64, i32]
        L.ft_gemm_best_ntile.argtypes = [i64, i64, i64, i32]
        L.ft_gemm_best_ntile.restype = i32
        L.ft_sf_ntile_bytes.restype = sz
        L.ft_workspace_bytes.argtypes = [i64, i64, i64, i32]
        L.ft_workspace_bytes.restype = sz
        L.ft_workspace_init.argtypes = [vp, sz, vp]
        L.ft_workspace_hs_offset.argtypes = [i64, i32]
        L.ft_workspace_hs_offset.restype = sz
        L.ft_error_string.argtypes = [C.c_int]
        L.ft_error_string.restype = C.c_char_p
        L.ft_debug_set_gemm_tile_n.argtypes = [C.c_int]
        L.ft_debug_set_quantize_mode.argtypes = [C.c_int]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        L = lib()
        raise FtError("fourtune: %s (status %d, cuda error %d)" %
                      (L.ft_error_string(rc).decode(), rc, L.ft_last_cuda_error()))


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _bf16(t):
    assert t.is_cuda and t.dtype == torch.bfloat16 and t.is_contiguous(), "need contiguous CUDA bf16"
    return t


def ft_sf_bytes(rows, cols, block_rows, layout):
    return lib().ft_sf_bytes(rows, cols, block_rows, layout)


def ft_workspace_bytes(M, K, N, r_t):
    return lib().ft_workspace_bytes(M, K, N, r_t)


def ft_workspace_init(workspace, stream=None):
    """Zero the control words at the head of a workspace (once per buffer; torch.zeros does the same)."""
    _check(lib().ft_workspace_init(_ptr(workspace), workspace.numel(), _stream(stream)))
    return workspace


def new_workspace(M, K, N, r_t, device="cuda"):
    """A workspace for one layer, control words initialised."""
    ws = torch.empty(ft_workspace_bytes(M, K, N, r_t), dtype=torch.uint8, device=device)
    return ft_workspace_init(ws)


def workspace_hs(workspace, M, r_t):
    """View of the pre-scaled low-rank intermediate Hs [M x r_t] (bf16) that the last ft_linear_* call left in
    `workspace` (ft_workspace_hs_offset of the header): what the GEMM consumed, for the staged comparison O-11."""
    off = lib().ft_workspace_hs_offset(M, r_t)
    return workspace[off:off + M * r_t * 2].view(torch.bfloat16).view(M, r_t)


class QTensor:
    """ft_qtensor with its buffers owned by torch."""

    def __init__(self, rows, cols, block_rows=1, sf_layout=FT_SF_TILE128x4, device="cuda"):
        self.rows, self.cols, self.block_rows, self.sf_layout = rows, cols, block_rows, sf_layout
        self.codes = torch.empty((rows, cols // 2), dtype=torch.uint8, device=device)
        self.sf = torch.zeros(ft_sf_bytes(rows, cols, block_rows, sf_layout), dtype=torch.uint8, device=device)
        self.tensor_dec_scale = torch.zeros(1, dtype=torch.float32, device=device)
        self.sf_ntile, self.ntile = None, 0      # weights only: scales cut to the GEMM's tile width

    def with_ntile(self, ntile=224):
        self.ntile = ntile
        self.sf_ntile = torch.zeros(lib().ft_sf_ntile_bytes(self.rows, self.cols, ntile), dtype=torch.uint8,
                                    device=self.codes.device)
        return self

    def c(self):
        return _QT(self.codes.data_ptr(), self.sf.data_ptr(), self.tensor_dec_scale.data_ptr(),
                   self.rows, self.cols, self.block_rows, self.sf_layout,
                   None if self.sf_ntile is None else self.sf_ntile.data_ptr(), self.ntile, 0)

    def sync_from(self, q):
        self.rows, self.cols, self.block_rows, self.sf_layout = q.rows, q.cols, q.block_rows, q.sf_layout


def ft_tensor_amax(x, out=None, stream=None):
    _bf16(x)
    out = torch.empty(1, dtype=torch.float32, device=x.device) if out is None else out
    _check(lib().ft_tensor_amax(_ptr(x), x.numel(), _ptr(out), _stream(stream)))
    return out


def ft_quantize_blockwise(x, out, tensor_amax=None, down=None, h_out=None, hs_out=None,
                          other_dec_scale=None, workspace=None, stream=None, round_mode=FT_ROUND_NEAREST_EVEN,
                          seed=0, offset=0):
    """x [rows x cols] bf16 -> out (QTensor).  down [cols x r_t] enables the fused projection.
    round_mode=FT_ROUND_STOCHASTIC: stochastic rounding of the codes from the Philox stream (seed, offset)."""
    _bf16(x)
    rows, cols = x.shape
    if workspace is None:
        workspace = new_workspace(rows, cols, 0, 0 if down is None else down.shape[1], x.device)
    proj = None
    if down is not None:
        _bf16(down)
        proj = _Proj(down.data_ptr(), None if h_out is None else h_out.data_ptr(),
                     None if hs_out is None else hs_out.data_ptr(),
                     None if other_dec_scale is None else other_dec_scale.data_ptr(), down.shape[1])
    q = out.c()
    _check(lib().ft_quantize_blockwise(_ptr(x), rows, cols, _ptr(tensor_amax),
                                       None if proj is None else C.byref(proj), C.byref(q),
                                       round_mode, seed, offset, _ptr(workspace), workspace.numel(),
                                       _stream(stream)))
    return out


def ft_quantize_blockwise_static(x, out, tensor_amax=None, down=None, h_out=None, hs_out=None, other_dec_scale=None,
                                 stream=None):
    """ft_quantize_blockwise on the library's static scratch array: no workspace argument, no device allocation."""
    _bf16(x)
    rows, cols = x.shape
    proj = None
    if down is not None:
        _bf16(down)
        proj = _Proj(down.data_ptr(), None if h_out is None else h_out.data_ptr(),
                     None if hs_out is None else hs_out.data_ptr(),
                     None if other_dec_scale is None else other_dec_scale.data_ptr(), down.shape[1])
    q = out.c()
    _check(lib().ft_quantize_blockwise_static(_ptr(x), rows, cols, _ptr(tensor_amax),
                                              None if proj is None else C.byref(proj), C.byref(q), _stream(stream)))
    return out


class Layer:
    """ft_layer: Q(R) in both orientations plus the low-rank factors D_f [K x r_t], U_t [N x r_t]."""

    def __init__(self, R_bf16, D_f, U_t, r_s, r, stream=None, ntile=224, tokens=None):
        """ntile: width of the tile-cut copy of the forward operand's scales (224 or 240; 192 for the FC1 of ft_mlp_fwd).
        tokens: the M this layer will run at; given, the library's cost model (ft_gemm_best_ntile) picks the widths
        for both operands (same results either way, only the GEMM's tile schedule differs)."""
        _bf16(R_bf16)
        N, K = R_bf16.shape
        self.N, self.K, self.r_s, self.r = N, K, r_s, r
        self.D_f, self.U_t = D_f, U_t
        if r_s + r > 0:
            _bf16(D_f), _bf16(U_t)
            assert D_f.shape == (K, r_s + r) and U_t.shape == (N, r_s + r)
        dev = R_bf16.device
        # a6: offline quantize (16x16 blocks, row-major S) then re-pack both orientations
        self.q_rowmajor = QTensor(N, K, 16, FT_SF_ROWMAJOR, dev)
        ft_quantize_blockwise(R_bf16, self.q_rowmajor, stream=stream)
        nt_bwd = ntile if ntile in (224, 240) else 224
        if tokens is not None:
            ntile = lib().ft_gemm_best_ntile(tokens, N, K, r_s + r) or 224
            nt_bwd = lib().ft_gemm_best_ntile(tokens, K, N, r_s + r) or 224
        self.r_kmajor = QTensor(N, K, 16, FT_SF_TILE128x4, dev).with_ntile(ntile)
        self.r_kmajor.codes = self.q_rowmajor.codes
        self.r_kmajor.tensor_dec_scale = self.q_rowmajor.tensor_dec_scale
        self.r_nmajor = QTensor(K, N, 16, FT_SF_TILE128x4, dev).with_ntile(nt_bwd)
        qk, qkt, qn = self.q_rowmajor.c(), self.r_kmajor.c(), self.r_nmajor.c()
        _check(lib().ft_pack_weight(C.byref(qk), C.byref(qkt), C.byref(qn), _stream(stream)))

    def c(self):
        return _Layer(self.r_kmajor.c(), self.r_nmajor.c(),
                      None if self.D_f is None else self.D_f.data_ptr(),
                      None if self.U_t is None else self.U_t.data_ptr(), self.K, self.N, self.r_s, self.r)


def ft_weight_transpose_codes(layer, codes_t, stream=None):
    """Single-copy weights (NEXT-5): rebuild the codes of Q(R)^T from layer.r_kmajor into codes_t (uint8, K*N/2)."""
    q = layer.r_kmajor.c()
    _check(lib().ft_weight_transpose_codes(C.byref(q), _ptr(codes_t), _stream(stream)))
    return codes_t


def ft_linear_fwd(layer, x, y, h_saved, qx, workspace, stream=None):
    _bf16(x)
    L, q = layer.c(), qx.c()
    _check(lib().ft_linear_fwd(C.byref(L), _ptr(x), x.shape[0], _ptr(y), _ptr(h_saved), C.byref(q),
                               _ptr(workspace), workspace.numel(), _stream(stream)))
    qx.sync_from(q)
    return y


def ft_linear_bwd_dgrad(layer, g, dx, p_saved, qg, workspace, stream=None):
    _bf16(g)
    L, q = layer.c(), qg.c()
    _check(lib().ft_linear_bwd_dgrad(C.byref(L), _ptr(g), g.shape[0], _ptr(dx), _ptr(p_saved), C.byref(q),
                                     _ptr(workspace), workspace.numel(), _stream(stream)))
    qg.sync_from(q)
    return dx


def ft_gemm4(a, b, lr_a_scaled, lr_b, out, stream=None):
    qa, qb = a.c(), b.c()
    r_t = 0 if lr_a_scaled is None else lr_a_scaled.shape[1]
    _check(lib().ft_gemm4(C.byref(qa), C.byref(qb), _ptr(lr_a_scaled), _ptr(lr_b), r_t, _ptr(out),
                          _stream(stream)))
    return out


def ft_lora_wgrad(layer, x, g, h_saved, p_saved, dA, dBt, accumulate=False, stream=None):
    L = layer.c()
    _check(lib().ft_lora_wgrad(C.byref(L), _ptr(x), _ptr(g), x.shape[0], _ptr(h_saved), _ptr(p_saved),
                               _ptr(dA), _ptr(dBt), 1 if accumulate else 0, _stream(stream)))
    return dA, dBt


def ft_lora_wgrad_q4(layer, qx, g, h_saved, p_saved, dA, dBt, accumulate=False, stream=None):
    """ft_lora_wgrad with dequant(Q(X)) -- the QTensor ft_linear_fwd filled -- in place of the bf16 X."""
    L, q = layer.c(), qx.c()
    _check(lib().ft_lora_wgrad_q4(C.byref(L), C.byref(q), _ptr(g), g.shape[0], _ptr(h_saved), _ptr(p_saved),
                                  _ptr(dA), _ptr(dBt), 1 if accumulate else 0, _stream(stream)))
    return dA, dBt


def ft_linear_bwd(layer, x, g, h_saved, dx, p_saved, dA, dBt, qg, workspace, accumulate=False, stream=None):
    """dgrad + LoRA wgrad in one call (one pass over g serves dBt and the tensor amax)."""
    _bf16(x), _bf16(g)
    L, q = layer.c(), qg.c()
    _check(lib().ft_linear_bwd(C.byref(L), _ptr(x), _ptr(g), g.shape[0], _ptr(h_saved), _ptr(dx), _ptr(p_saved),
                               _ptr(dA), _ptr(dBt), 1 if accumulate else 0, C.byref(q), _ptr(workspace),
                               workspace.numel(), _stream(stream)))
    qg.sync_from(q)
    return dx, dA, dBt


def ft_linear_bwd_q4(layer, qx, g, h_saved, dx, p_saved, dA, dBt, qg, workspace, accumulate=False, stream=None):
    """ft_linear_bwd with dA taken from the saved Q(X) instead of the bf16 X."""
    _bf16(g)
    L, qi, q = layer.c(), qx.c(), qg.c()
    _check(lib().ft_linear_bwd_q4(C.byref(L), C.byref(qi), _ptr(g), g.shape[0], _ptr(h_saved), _ptr(dx), _ptr(p_saved),
                                  _ptr(dA), _ptr(dBt), 1 if accumulate else 0, C.byref(q), _ptr(workspace),
                                  workspace.numel(), _stream(stream)))
    qg.sync_from(q)
    return dx, dA, dBt


def new_mlp_workspace(M, K, N1, r_t1, r_t2, device="cuda"):
    ws = torch.empty(lib().ft_mlp_workspace_bytes(M, K, N1, r_t1, r_t2), dtype=torch.uint8, device=device)
    return ft_workspace_init(ws)


def mlp_workspace_hs2(workspace, M, r_t1, r_t2):
    off = lib().ft_mlp_workspace_hs2_offset(M, r_t1)
    return workspace[off:off + M * r_t2 * 2].view(torch.bfloat16).view(M, r_t2)


def ft_mlp_fwd(fc1, fc2, x, z_amax, y1_amax, y2, h1, h2, qx, qz, qy1, workspace, z_amax_next=None, y1_amax_next=None,
               z_debug=None, y1_debug=None, stream=None):
    """FC1 -> GeLU -> FC2 with the FC1 GEMM's epilogue doing GeLU and FC2's quantize + down-projection (NEXT-1)."""
    _bf16(x)
    L1, L2, a, b, c = fc1.c(), fc2.c(), qx.c(), qz.c(), qy1.c()
    _check(lib().ft_mlp_fwd(C.byref(L1), C.byref(L2), _ptr(x), x.shape[0], _ptr(z_amax), _ptr(y1_amax),
                            _ptr(z_amax_next), _ptr(y1_amax_next), _ptr(y2), _ptr(h1), _ptr(h2), C.byref(a), C.byref(b),
                            C.byref(c), _ptr(z_debug), _ptr(y1_debug), _ptr(workspace), workspace.numel(), _stream(stream)))
    qx.sync_from(a), qz.sync_from(b), qy1.sync_from(c)
    return y2


def ft_gelu_bwd_q4(dz, qy1, out, stream=None):
    q = qy1.c()
    _check(lib().ft_gelu_bwd_q4(_ptr(dz), C.byref(q), _ptr(out), _stream(stream)))
    return out


# test / bench hooks of include/fourtune_debug.h (not part of the product interface)
def debug_set_gemm_tile_n(bn):
    _check(lib().ft_debug_set_gemm_tile_n(bn))


def debug_set_quantize_mode(mode):
    _check(lib().ft_debug_set_quantize_mode(mode))
