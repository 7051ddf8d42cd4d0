"""Oracle: the FourTune triple-branch linear layer -- TEST INFRASTRUCTURE.

Shapes (PAPER.md:77,94,106 use W in R^{m x n}, Y = X W):
    X : M x K      activations (bf16)
    R : N x K      residual weight, K contiguous (paper's R^T), quantized 16x16
    G : M x N      output gradient dL/dY (bf16)
    D_f = [L1 | A] : K x r_t    down-projection (stabilizer cols 0..r_s, LoRA after)
    U_f = [L2 ; B] : r_t x N    up-projection
    r_t = r_s + r

Passages followed:
  Eq. 1  W ~= R + L_stab, L_stab = L1 L2           -> prepare_weight
  Eq. 2 (lost in extraction between PAPER.md:86 and 88; recovered from the
         prose, Fig. 3b at PAPER.md:65, and as the unique forward whose input
         gradient is Eq. 3):
         Y = GEMM_4bit(Q(X), Q(R)) + X L1 L2 + X A B                 -> forward
  Eq. 3     dX = GEMM_4bit(Q(G), Q(R)^T) + G L_stab^T + G (AB)^T
                                                                     -> dgrad
  Eq. 4    dB = (XA)^T G ,  dA = X^T (G B^T)          -> wgrad
  Q(R)^T is the same codes and scales as Q(R), re-indexed.

Readings: O-10 the low-rank branches consume the bf16 X / G (not the
dequantized codes); H = X D_f and P = G U_f^T are stored in bf16.  O-10' ("pre-
scaled" variant, what the CUDA epilogue computes): H' = bf16(H_exact / alpha),
Y = bf16(alpha * (acc4 + H' U_f)), alpha = g_dec_X * g_dec_R, so that the
low-rank product can be accumulated in the same accumulator as the unscaled
4-bit sum.  Both variants are implemented; they differ only in where the one
bf16 rounding of the rank-r_t intermediate happens.

All sums are float64.  No blocking, fusion or reordering.

Pins (tests/test_oracle_layer.py): brute-force Python triple loops on tiny
shapes, r_s = r = 0 reducing to a float64 matmul of the dequantized operands,
B = 0 / A = 0 degenerate cases, the exact-linearity adjoint identity
<Y,G> = <X,dX> and the directional derivative for Eq. 4 on grid-exact data.
"""
import numpy as np

from . import nvfp4
from .nvfp4 import bf16_round_from_f64


def prepare_weight(W, r_s):
    """Eq. 1 under reading O-13: float64 SVD of W [N x K]; with W^T = V S U^T in
    the paper's orientation, L1 = bf16(V_r sqrt(S_r)) [K x r_s],
    L2 = bf16(sqrt(S_r) U_r^T) [r_s x N], R = bf16(W - (L1 L2)^T) using the
    ROUNDED L1, L2.  No smoothing.  Returns float32 arrays of bf16 values."""
    W = np.asarray(W, dtype=np.float64)
    N, K = W.shape
    if r_s == 0:
        return (nvfp4.bf16_round(W.astype(np.float32)),
                np.zeros((K, 0), np.float32), np.zeros((0, N), np.float32))
    # W = Uw diag(s) Vh  with Uw [N x q], Vh [q x K]
    Uw, s, Vh = np.linalg.svd(W, full_matrices=False)
    rs = np.sqrt(s[:r_s])
    L1 = bf16_round_from_f64(Vh[:r_s, :].T * rs[None, :])       # K x r_s
    L2 = bf16_round_from_f64(rs[:, None] * Uw[:, :r_s].T)       # r_s x N
    R = bf16_round_from_f64(W - (L1.astype(np.float64) @ L2.astype(np.float64)).T)
    return R, L1, L2


def quantize_weight(R):
    """a6: Q(R) with 16x16 blocks."""
    return nvfp4.quantize_blockwise(R, block_rows=16, block_cols=16)


def _alpha(qa, qr):
    return np.float64(np.float32(qa["g_dec"]) * np.float32(qr["g_dec"]))   # one float32 multiply


def forward(X, qR, D_f, U_f, prescale=False, H_given=None, x_amax=None, out_bf16=True):
    """F: H = bf16(X D_f);  Y = bf16( sum_k dq(X)[m,k] dq(R)[n,k] + sum_j H[m,j] U_f[j,n] ).

    prescale=True follows O-10': the returned H is still bf16(X D_f) (saved for
    wgrad) and Hs = bf16((X D_f) / alpha) feeds the up-projection.
    H_given: use these bf16 values in place of the oracle's own H (prescale
    False) or Hs (prescale True) -- the staged comparison of DESIGN.md O-11.
    Returns dict(Y, H, Hs, qX, alpha)."""
    X = np.asarray(X, dtype=np.float32)
    qX = nvfp4.quantize_blockwise(X, block_rows=1, block_cols=16, amax_t=x_amax)
    alpha = _alpha(qX, qR)
    Hex = X.astype(np.float64) @ np.asarray(D_f, np.float64)              # M x r_t, float64
    H = bf16_round_from_f64(Hex)
    Hs = bf16_round_from_f64(Hex / alpha)
    U = np.asarray(U_f, np.float64)
    if prescale:
        Hin = Hs if H_given is None else np.asarray(H_given, np.float32)
        acc = nvfp4.dequantize_unscaled(qX) @ nvfp4.dequantize_unscaled(qR).T
        Yex = alpha * (acc + Hin.astype(np.float64) @ U)
    else:
        Hin = H if H_given is None else np.asarray(H_given, np.float32)
        Yex = nvfp4.dequantize(qX) @ nvfp4.dequantize(qR).T + Hin.astype(np.float64) @ U
    Y = bf16_round_from_f64(Yex) if out_bf16 else Yex
    return {"Y": Y, "H": H, "Hs": Hs, "qX": qX, "alpha": alpha, "Y_exact": Yex}


def dgrad(G, qR, D_f, U_f, prescale=False, P_given=None, g_amax=None, out_bf16=True):
    """B: P = bf16(G U_f^T);  dX = bf16( sum_n dq(G)[m,n] dq(R)[n,k] + sum_j P[m,j] D_f[k,j] ).
    G is quantized in 1x16 blocks along N, the dgrad reduction dim (O-2)."""
    G = np.asarray(G, dtype=np.float32)
    qG = nvfp4.quantize_blockwise(G, block_rows=1, block_cols=16, amax_t=g_amax)
    alpha = _alpha(qG, qR)
    Pex = G.astype(np.float64) @ np.asarray(U_f, np.float64).T            # M x r_t
    P = bf16_round_from_f64(Pex)
    Ps = bf16_round_from_f64(Pex / alpha)
    Dt = np.asarray(D_f, np.float64).T                                    # r_t x K
    if prescale:
        Pin = Ps if P_given is None else np.asarray(P_given, np.float32)
        acc = nvfp4.dequantize_unscaled(qG) @ nvfp4.dequantize_unscaled(qR)
        dXex = alpha * (acc + Pin.astype(np.float64) @ Dt)
    else:
        Pin = P if P_given is None else np.asarray(P_given, np.float32)
        dXex = nvfp4.dequantize(qG) @ nvfp4.dequantize(qR) + Pin.astype(np.float64) @ Dt
    dX = bf16_round_from_f64(dXex) if out_bf16 else dXex
    return {"dX": dX, "P": P, "Ps": Ps, "qG": qG, "alpha": alpha, "dX_exact": dXex}


def wgrad(X, G, H, P, r_s):
    """W (Eq. 4): dB[j,n] = sum_m H[m, r_s+j] G[m,n];  dA[k,j] = sum_m X[m,k] P[m, r_s+j].
    H[:, r_s:] = bf16(X A) saved from forward, P[:, r_s:] = bf16(G B^T) from dgrad;
    X is the bf16 X saved from forward (O-12).  float64 sums, float32 results."""
    X = np.asarray(X, np.float64)
    G = np.asarray(G, np.float64)
    H_l = np.asarray(H, np.float64)[:, r_s:]
    P_l = np.asarray(P, np.float64)[:, r_s:]
    dB = (H_l.T @ G).astype(np.float32)
    dA = (X.T @ P_l).astype(np.float32)
    return {"dA": dA, "dB": dB}


def wgrad_saved4(qX, G, H, P, r_s):
    """W with 4-bit saved activations (reading O-12' in DESIGN.md): Eq. 4
     with the X of `dA = X^T (G B^T)` taken as dequant(Q(X)) -- the codes and scales
    the forward pass produced anyway -- instead of the bf16 X, so that the layer keeps 0.5625
    instead of 2 bytes per activation element between forward and backward (the activation side
    of the memory figures at PAPER.md:197-207; the paper does not say which X its Eq. 4 uses).
        dA[k,j] = sum_m (E2M1(code[m,k]) * sf[m,k/16] * g_dec) * P[m, r_s+j]
    dB is unchanged (it never touches X).  float64 sums, float32 results."""
    return wgrad(nvfp4.dequantize(qX), G, H, P, r_s)


# ---------------------------------------------------------------- NEXT-1: MLP fusion (sec. 3.3)
# "we fuse the first fully connected (FC1) GEMM with the subsequent FC2 quantization kernel.  This approach allows
#  intermediate results to be consumed immediately without materializing large tensors in global memory".
# The paper names GeLU and says nothing else; reading O-16 of DESIGN.md pins the rest:
#   * GeLU is the tanh form (FLUX's MLP), evaluated on the bf16-rounded FC1 output Y1, and rounded to bf16: Z;
#   * Q(Z) (1x16 blocks along FC2's reduction dim) takes its tensor amax from the CALLER (delayed scaling: the
#     value of the previous step; the epilogue of a GEMM cannot know max|Z| before its last tile), and so does the
#     second quantized tensor the block keeps, Q(Y1), the pre-activation that GeLU's backward consumes;
#   * FC2's low-rank branches consume the bf16 Z (O-10 unchanged): H2 = bf16(Z D_f2);
#   * backward: dY1 = bf16( dZ * gelu'(dequant(Q(Y1))) ), dZ the bf16 dgrad of FC2; FC2's dA uses dequant(Q(Z))
#     (reading O-12', since the bf16 Z is never materialized).
# The fused forward is BY DEFINITION the composition of the two layer forwards with that quantizer in between:
# mlp_forward below is written as that composition, so "fused == unfused" holds by construction and the CUDA
# kernel is what has to match it.

def _gelu_sigmoid(y):
    """0.5 (1 + tanh t) = 1 / (1 + exp(-2 t)), t = sqrt(2/pi) (y + 0.044715 y^3), float64.  The same function as
    the tanh expression, written so that it does not cancel: 1 + tanh(t) loses all its digits in float64 once
    t < -18 (y < -5.3), where the value is 1e-16 .. 1e-37 -- still a normal bf16 number."""
    y = np.asarray(y, dtype=np.float64)
    t = np.sqrt(2.0 / np.pi) * (y + 0.044715 * y * y * y)
    with np.errstate(over="ignore"):
        return 1.0 / (1.0 + np.exp(-2.0 * t))


def gelu_tanh(y):
    """GeLU, tanh form: 0.5 y (1 + tanh( sqrt(2/pi) (y + 0.044715 y^3) )) = y sigmoid(2 t), float64."""
    return np.asarray(y, dtype=np.float64) * _gelu_sigmoid(y)


def gelu_tanh_grad(y):
    """d/dy of gelu_tanh, float64: with s = sigmoid(2 t),  s + y s (1 - s) 2 sqrt(2/pi) (1 + 3 * 0.044715 y^2)."""
    y = np.asarray(y, dtype=np.float64)
    s = _gelu_sigmoid(y)
    return s + y * s * (1.0 - s) * 2.0 * np.sqrt(2.0 / np.pi) * (1.0 + 3.0 * 0.044715 * y * y)


def mlp_forward(X, qR1, D1, U1, qR2, D2, U2, z_amax, y1_amax, Y1_given=None, Z_given=None, H1s_given=None,
                H2s_given=None):
    """FC1 -> GeLU -> FC2 under reading O-16 (pre-scaled low-rank intermediates, O-10').
    *_given: bf16 values produced by the CUDA path that replace the oracle's own at that point (the staged
    comparison of DESIGN.md O-11: each stage is checked on its own, then fed forward bit for bit).
    Returns Y1, Z (bf16), qZ, qY1, Y2, and the two layer dicts."""
    f1 = forward(X, qR1, D1, U1, prescale=True, H_given=H1s_given)
    Y1 = f1["Y"] if Y1_given is None else np.asarray(Y1_given, np.float32)
    Z = bf16_round_from_f64(gelu_tanh(Y1)) if Z_given is None else np.asarray(Z_given, np.float32)
    qY1 = nvfp4.quantize_blockwise(Y1, block_rows=1, block_cols=16, amax_t=y1_amax)
    f2 = forward(Z, qR2, D2, U2, prescale=True, x_amax=z_amax, H_given=H2s_given)
    return {"Y1": Y1, "Z": Z, "qZ": f2["qX"], "qY1": qY1, "Y2": f2["Y"], "fc1": f1, "fc2": f2}


def gelu_backward_saved4(dZ, qY1):
    """dY1 = bf16( dZ * gelu'(dequant(Q(Y1))) ): GeLU's backward on the 4-bit saved pre-activation (O-16)."""
    return bf16_round_from_f64(np.asarray(dZ, np.float64) * gelu_tanh_grad(nvfp4.dequantize(qY1)))
