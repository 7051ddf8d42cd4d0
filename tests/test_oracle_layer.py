"""Pins for oracle/layer.py (CPU only): brute force, degenerate layers, adjoint identities."""
import numpy as np
import pytest

from oracle import layer, nvfp4
from paper_2607_05711_b200 import synth


def _tiny_layer(seed, M, K, N, r_s, r):
    d = synth.layer_inputs(seed, M, K, N, max(r, 1))
    R, L1, L2 = layer.prepare_weight(d["W"], r_s)
    A, B = d["A"][:, :r], d["B"][:r, :]
    D_f = np.concatenate([L1, A], axis=1).astype(np.float32)
    U_f = np.concatenate([L2, B], axis=0).astype(np.float32)
    return d["X"], d["dY"], R, D_f, U_f, d["W"]


# ---------------------------------------------------------------- Eq. 1 / O-13
def test_prepare_weight_split():
    rng = synth.make_rng(11)
    W = synth.normal(rng, (96, 64), 0.02)
    # plant a rank-2 high-magnitude component (the "outliers" of PAPER.md:80)
    u = rng.standard_normal((96, 2)).astype(np.float32)
    v = rng.standard_normal((2, 64)).astype(np.float32)
    W = synth.to_bf16_f32(W + 0.5 * (u @ v) / 8)
    R, L1, L2 = layer.prepare_weight(W, 4)
    assert L1.shape == (64, 4) and L2.shape == (4, 96) and R.shape == W.shape
    rec = R.astype(np.float64) + (L1.astype(np.float64) @ L2.astype(np.float64)).T
    # R absorbs the bf16 rounding of L1, L2: reconstruction is exact up to one bf16 rounding of R
    assert np.max(np.abs(rec - W)) <= np.max(np.abs(R)) * 2.0 ** -8
    # Eckart-Young: the residual's spectral norm is the 5th singular value of W (up to rounding)
    s = np.linalg.svd(W.astype(np.float64), compute_uv=False)
    sR = np.linalg.svd(R.astype(np.float64), compute_uv=False)
    assert abs(sR[0] - s[4]) < 0.02 * s[4] + 1e-3
    # stabilizer makes the residual easier to quantize than W (stand-in for Fig. 8 / Table 5)
    rel = lambda a: np.linalg.norm(nvfp4.dequantize(nvfp4.quantize_blockwise(a, 16)) - a)
    assert rel(R) < rel(W)
    # r_s = 0 -> R = W
    R0, L10, L20 = layer.prepare_weight(W, 0)
    assert np.array_equal(R0, W) and L10.shape == (64, 0) and L20.shape == (0, 96)


# ------------------------------------------------------- P-7: brute force loops
def _brute_forward(X, R, D_f, U_f):
    """Pure-Python restatement of F from the scalar definitions (no numpy matmul,
    no shared quantizer internals beyond the per-element grids)."""
    M, K = X.shape
    N = R.shape[0]
    r_t = D_f.shape[1]
    qX = nvfp4.quantize_blockwise(X, 1)
    qR = nvfp4.quantize_blockwise(R, 16)
    gx, gr = float(qX["g_dec"]), float(qR["g_dec"])
    Y = np.zeros((M, N))
    H = np.zeros((M, r_t), np.float32)
    for m in range(M):
        for j in range(r_t):
            s = 0.0
            for k in range(K):
                s += float(X[m, k]) * float(D_f[k, j])
            H[m, j] = nvfp4.bf16_round_from_f64(np.array([s]))[0]
    for m in range(M):
        for n in range(N):
            s = 0.0
            for k in range(K):
                xv = float(nvfp4.e2m1_decode(qX["codes"][m, k])) * float(nvfp4.e4m3_decode(qX["sf"][m, k // 16])) * gx
                rv = float(nvfp4.e2m1_decode(qR["codes"][n, k])) * float(nvfp4.e4m3_decode(qR["sf"][n // 16, k // 16])) * gr
                s += xv * rv
            for j in range(r_t):
                s += float(H[m, j]) * float(U_f[j, n])
            Y[m, n] = s
    return Y, H


def test_forward_bruteforce_tiny():
    X, G, R, D_f, U_f, _ = _tiny_layer(21, 3, 32, 16, 2, 2)
    Yb, Hb = _brute_forward(X, R, D_f, U_f)
    out = layer.forward(X, layer.quantize_weight(R), D_f, U_f, prescale=False, out_bf16=False)
    assert np.array_equal(out["H"], Hb)
    assert np.allclose(out["Y"], Yb, rtol=1e-12, atol=1e-15)


def test_dgrad_wgrad_bruteforce_tiny():
    X, G, R, D_f, U_f, _ = _tiny_layer(22, 3, 32, 16, 2, 2)
    M, K = X.shape
    N = R.shape[0]
    r_s, r_t = 2, 4
    qR = layer.quantize_weight(R)
    qG = nvfp4.quantize_blockwise(G, 1)
    dqG, dqR = nvfp4.dequantize(qG), nvfp4.dequantize(qR)
    out = layer.dgrad(G, qR, D_f, U_f, prescale=False, out_bf16=False)
    P = out["P"]
    for m in range(M):
        for j in range(r_t):
            s = sum(float(G[m, n]) * float(U_f[j, n]) for n in range(N))
            assert P[m, j] == nvfp4.bf16_round_from_f64(np.array([s]))[0]
        for k in range(K):
            s = sum(dqG[m, n] * dqR[n, k] for n in range(N))
            s += sum(float(P[m, j]) * float(D_f[k, j]) for j in range(r_t))
            assert abs(out["dX"][m, k] - s) <= 1e-12 * max(1.0, abs(s))
    fw = layer.forward(X, qR, D_f, U_f)
    w = layer.wgrad(X, G, fw["H"], P, r_s)
    for j in range(r_t - r_s):
        for n in range(N):
            s = sum(float(fw["H"][m, r_s + j]) * float(G[m, n]) for m in range(M))
            assert abs(w["dB"][j, n] - s) <= 1e-6 * max(1e-6, abs(s))
        for k in range(K):
            s = sum(float(X[m, k]) * float(P[m, r_s + j]) for m in range(M))
            assert abs(w["dA"][k, j] - s) <= 1e-6 * max(1e-6, abs(s))
    assert w["dA"].shape == (K, 2) and w["dB"].shape == (2, N)


# ------------------------------------------------------ P-5: degenerate layers
def test_no_lowrank_reduces_to_matmul_of_dequantized():
    X, G, R, D_f, U_f, _ = _tiny_layer(23, 20, 64, 48, 0, 0)
    assert D_f.shape[1] == 0
    qR = layer.quantize_weight(R)
    for prescale in (False, True):
        out = layer.forward(X, qR, D_f, U_f, prescale=prescale, out_bf16=False)
        ref = nvfp4.dequantize(out["qX"]) @ nvfp4.dequantize(qR).T
        rtol = 2e-7 if prescale else 1e-12      # alpha is ONE float32 product in the prescaled variant
        assert np.allclose(out["Y"], ref, rtol=rtol, atol=0)
        outb = layer.dgrad(G, qR, D_f, U_f, prescale=prescale, out_bf16=False)
        refb = nvfp4.dequantize(outb["qG"]) @ nvfp4.dequantize(qR)
        assert np.allclose(outb["dX"], refb, rtol=rtol, atol=0)


def test_zero_adapter_cases():
    X, G, R, D_f, U_f, _ = _tiny_layer(24, 16, 64, 32, 4, 4)
    qR = layer.quantize_weight(R)
    r_s = 4
    base = layer.forward(X, qR, D_f, U_f, out_bf16=False)
    # B = 0: branch 3 contributes exactly 0 to Y and dX; dA = 0, dB != 0
    U0 = U_f.copy(); U0[r_s:] = 0
    f0 = layer.forward(X, qR, D_f, U0, out_bf16=False)
    no_lora = layer.forward(X, qR, D_f[:, :r_s], U_f[:r_s], out_bf16=False)
    assert np.array_equal(f0["Y"], no_lora["Y"])
    assert not np.array_equal(f0["Y"], base["Y"])
    b0 = layer.dgrad(G, qR, D_f, U0, out_bf16=False)
    bn = layer.dgrad(G, qR, D_f[:, :r_s], U_f[:r_s], out_bf16=False)
    assert np.array_equal(b0["dX"], bn["dX"])
    w0 = layer.wgrad(X, G, f0["H"], b0["P"], r_s)
    assert np.count_nonzero(w0["dA"]) == 0 and np.count_nonzero(w0["dB"]) > 0
    # A = 0: dB = 0
    D0 = D_f.copy(); D0[:, r_s:] = 0
    fA = layer.forward(X, qR, D0, U_f)
    bA = layer.dgrad(G, qR, D0, U_f)
    wA = layer.wgrad(X, G, fA["H"], bA["P"], r_s)
    assert np.count_nonzero(wA["dB"]) == 0 and np.count_nonzero(wA["dA"]) > 0
    # L1 = 0: stabilizer vanishes
    D1 = D_f.copy(); D1[:, :r_s] = 0
    f1 = layer.forward(X, qR, D1, U_f, out_bf16=False)
    f1n = layer.forward(X, qR, D_f[:, r_s:], U_f[r_s:], out_bf16=False)
    assert np.allclose(f1["Y"], f1n["Y"], rtol=1e-13, atol=1e-18)


# ------------------------------------------- P-6: exact-linearity special case
def _grid_exact(rng, rows, cols, block_rows, emin, emax):
    """Values from the E2M1 grid times one power of two per block, every block
    holding a +-6, so that Q is the identity given amax_t = 2688 * 2^-J."""
    codes = rng.integers(0, 16, (rows, cols)).astype(np.uint8)
    br = block_rows
    cb = codes.reshape(rows // br, br, cols // 16, 16)
    cb[:, 0, :, 0] = 7
    expo = rng.integers(emin, emax + 1, (rows // br, cols // 16))
    scale = np.repeat(np.repeat(np.exp2(expo), br, 0), 16, 1)
    return (nvfp4.e2m1_decode(codes) * scale).astype(np.float32)


def test_adjoint_identity_exact_linear_case():
    rng = np.random.default_rng(31)
    M, K, N, r_s, r = 8, 64, 48, 2, 3
    R = _grid_exact(rng, N, K, 16, -5, 1)
    amax = 2688.0 / 64.0
    qR = nvfp4.quantize_blockwise(R, 16, amax_t=amax)
    assert np.array_equal(nvfp4.dequantize(qR), R.astype(np.float64))         # Q is the identity here
    # low-rank factors with few significant bits so that bf16(H), bf16(P) are exact
    D_f = (rng.integers(-2, 3, (K, r_s + r)) * 2.0 ** -3).astype(np.float32)
    U_f = (rng.integers(-2, 3, (r_s + r, N)) * 2.0 ** -3).astype(np.float32)
    Xs = (rng.integers(-3, 4, (M, K)) * 0.5).astype(np.float32)               # small-integer X for exact H
    Xs[:, ::16] = 6.0
    qXs = nvfp4.quantize_blockwise(Xs, 1, amax_t=amax)
    assert np.array_equal(nvfp4.dequantize(qXs), Xs.astype(np.float64))
    Gs = (rng.integers(-3, 4, (M, N)) * 0.5).astype(np.float32); Gs[:, ::16] = 6.0
    f = layer.forward(Xs, qR, D_f, U_f, x_amax=amax, out_bf16=False)
    b = layer.dgrad(Gs, qR, D_f, U_f, g_amax=amax, out_bf16=False)
    assert np.array_equal(f["H"].astype(np.float64), Xs.astype(np.float64) @ D_f.astype(np.float64))
    # with Q the identity the layer is Y = X W_eff: <Y, G> == <X, dX> for all three branches
    W_eff = R.astype(np.float64).T + D_f.astype(np.float64) @ U_f.astype(np.float64)      # K x N
    assert np.allclose(f["Y"], Xs.astype(np.float64) @ W_eff, rtol=1e-13)
    assert np.allclose(b["dX"], Gs.astype(np.float64) @ W_eff.T, rtol=1e-13)
    lhs = np.sum(f["Y"] * Gs.astype(np.float64))
    rhs = np.sum(Xs.astype(np.float64) * b["dX"])
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    # Eq. 4: <dA, A'> + <dB, B'> is the directional derivative of <Y, G> along (A', B')
    w = layer.wgrad(Xs, Gs, f["H"], b["P"], r_s)
    Ad = rng.standard_normal((K, r)); Bd = rng.standard_normal((r, N))
    A0, B0 = D_f[:, r_s:].astype(np.float64), U_f[r_s:].astype(np.float64)
    Xd, Gd = Xs.astype(np.float64), Gs.astype(np.float64)
    dirder = np.sum((Xd @ (Ad @ B0 + A0 @ Bd)) * Gd)
    got = np.sum(w["dA"].astype(np.float64) * Ad) + np.sum(w["dB"].astype(np.float64) * Bd)
    assert abs(got - dirder) <= 1e-6 * abs(dirder) + 1e-9
    # guard that the check can fail: a slipped wgrad (H and P exchanged in role) breaks it
    slipped = np.sum((Xd.T @ f["H"][:, r_s:].astype(np.float64)) * Ad)
    assert abs(slipped + np.sum(w["dB"].astype(np.float64) * Bd) - dirder) > 1e-3 * abs(dirder)


# ------------------------------------- O-10': the prescaled variant is the same layer
def test_prescaled_variant_close_to_plain():
    X, G, R, D_f, U_f, _ = _tiny_layer(25, 64, 256, 128, 8, 8)
    qR = layer.quantize_weight(R)
    a = layer.forward(X, qR, D_f, U_f, prescale=False, out_bf16=False)
    p = layer.forward(X, qR, D_f, U_f, prescale=True, out_bf16=False)
    assert np.array_equal(a["H"], p["H"])
    # the two differ only by one bf16 rounding of the rank-r_t intermediate
    lr = a["H"].astype(np.float64) @ U_f.astype(np.float64)
    diff = np.linalg.norm(a["Y"] - p["Y"])
    assert 0 < diff <= 2.0 ** -7 * np.linalg.norm(lr)
    # Hs * alpha reproduces H to bf16 precision
    assert np.allclose(p["Hs"].astype(np.float64) * p["alpha"], a["H"], rtol=2.0 ** -7)
    # staged comparison hook: feeding Hs back in reproduces the same Y
    p2 = layer.forward(X, qR, D_f, U_f, prescale=True, H_given=p["Hs"], out_bf16=False)
    assert np.array_equal(p2["Y"], p["Y"])
    ab = layer.dgrad(G, qR, D_f, U_f, prescale=False, out_bf16=False)
    pb = layer.dgrad(G, qR, D_f, U_f, prescale=True, out_bf16=False)
    lrb = ab["P"].astype(np.float64) @ D_f.astype(np.float64).T
    assert np.linalg.norm(ab["dX"] - pb["dX"]) <= 2.0 ** -7 * np.linalg.norm(lrb)


def test_qrt_is_permuted_qr_in_dgrad():
    """dgrad with Q(R)^T must equal dgrad with a separately quantized R^T (16x16 blocks)."""
    X, G, R, D_f, U_f, _ = _tiny_layer(26, 16, 64, 32, 0, 0)
    qR = layer.quantize_weight(R)
    qRt = layer.quantize_weight(np.ascontiguousarray(R.T))
    out = layer.dgrad(G, qR, D_f, U_f, out_bf16=False)
    ref = nvfp4.dequantize(out["qG"]) @ nvfp4.dequantize(qRt).T
    assert np.allclose(out["dX"], ref, rtol=1e-10, atol=1e-14 * np.abs(ref).max())   # summation order only


# ------------------------------------------- NEXT-2 / O-12': dA from the saved 4-bit activations
def test_wgrad_saved4_bruteforce_and_special_cases():
    X, G, R, D_f, U_f, _ = _tiny_layer(31, 5, 32, 16, 2, 2)
    M, K = X.shape
    r_s = 2
    qR = layer.quantize_weight(R)
    fw = layer.forward(X, qR, D_f, U_f)
    P = layer.dgrad(G, qR, D_f, U_f)["P"]
    qX = fw["qX"]
    w4 = layer.wgrad_saved4(qX, G, fw["H"], P, r_s)
    w = layer.wgrad(X, G, fw["H"], P, r_s)
    # brute force from the codes, the scale bytes and g_dec, decoded by hand (not through dequantize):
    # E2M1 magnitudes by table, E4M3 by its bit fields
    mag = [0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0]
    def e4m3(b):
        e, m = (int(b) >> 3) & 15, int(b) & 7
        return (m / 8.0) * 2.0 ** -6 if e == 0 else (1 + m / 8.0) * 2.0 ** (e - 7)
    g_dec = float(np.float32(qX["g_dec"]))
    for k in range(K):
        for j in range(2):
            s = 0.0
            for m in range(M):
                c = int(qX["codes"][m, k])
                v = (-1.0 if c & 8 else 1.0) * mag[c & 7] * e4m3(qX["sf"][m, k // 16]) * g_dec
                s += v * float(P[m, r_s + j])
            assert abs(w4["dA"][k, j] - s) <= 1e-6 * max(1e-6, abs(s))
    # dB never touches X
    assert np.array_equal(w4["dB"], w["dB"])
    # the two readings of Eq. 4 differ by exactly the quantization error of X against P
    err = (nvfp4.dequantize(qX) - X.astype(np.float64)).T @ P[:, r_s:].astype(np.float64)
    assert np.allclose(w4["dA"] - w["dA"], err, rtol=0, atol=1e-6 * np.abs(w["dA"]).max() + 1e-12)
    assert np.any(w4["dA"] != w["dA"])
    # on data Q(.) represents exactly the two readings coincide: grid values times a power-of-two
    # block scale, tensor amax 42 = 2688 / 64 so that g_enc = 64 exactly, a +-6 in every block
    rng = synth.make_rng(5)
    grid = np.array(mag + [-v for v in mag], np.float32)
    Xe = grid[rng.integers(0, 16, (M, K))].reshape(M, K // 16, 16)
    Xe[:, :, 0] = 6.0 * np.where(rng.integers(0, 2, (M, K // 16)) == 1, 1.0, -1.0)
    sfe = (2.0 ** rng.integers(-3, 4, (M, K // 16))).astype(np.float32)
    sfe[0, 0] = 448.0
    Xe = (Xe * sfe[:, :, None] / 64.0).reshape(M, K).astype(np.float32)
    assert np.abs(Xe).max() == 42.0
    qXe = nvfp4.quantize_blockwise(Xe, 1)
    assert np.array_equal(nvfp4.dequantize(qXe), Xe.astype(np.float64))
    assert np.array_equal(layer.wgrad_saved4(qXe, G, fw["H"], P, r_s)["dA"],
                          layer.wgrad(Xe, G, fw["H"], P, r_s)["dA"])


# ------------------------------------------------------------------ NEXT-1: MLP fusion oracle (reading O-16)
def test_gelu_tanh_closed_forms_and_derivative():
    """gelu_tanh against what the mathematics fixes: gelu(0) = 0; gelu(y) - gelu(-y) = y (the tanh form's 1 + tanh
    and 1 - tanh halves add to 2); gelu(y) -> y and gelu(-y) -> 0 for large y; within 1e-3 of the erf form it
    approximates (Hendrycks & Gimpel); hand value gelu(1) = 0.5 (1 + tanh(0.7978845608 * 1.044715)); and the
    derivative against central differences."""
    import math
    assert layer.gelu_tanh(0.0) == 0.0
    y = np.linspace(-6, 6, 2401)
    g = layer.gelu_tanh(y)
    assert np.allclose(g - layer.gelu_tanh(-y), y, rtol=0, atol=1e-15)
    assert abs(layer.gelu_tanh(12.0) - 12.0) < 1e-12 and abs(layer.gelu_tanh(-12.0)) < 1e-12
    erf_form = np.array([0.5 * v * (1.0 + math.erf(v / math.sqrt(2.0))) for v in y])
    assert np.max(np.abs(g - erf_form)) < 1e-3 and np.max(np.abs(g - erf_form)) > 1e-5      # close, not the same function
    assert abs(layer.gelu_tanh(1.0) - 0.5 * (1.0 + math.tanh(0.7978845608028654 * 1.044715))) < 1e-15
    h = 1e-6
    fd = (layer.gelu_tanh(y + h) - layer.gelu_tanh(y - h)) / (2 * h)
    assert np.max(np.abs(fd - layer.gelu_tanh_grad(y))) < 1e-8
    assert abs(layer.gelu_tanh_grad(0.0) - 0.5) < 1e-15
    # the left tail, where 1 + tanh(t) cancels in float64: against y e^{2t} / (1 + e^{2t}) with e^{2t} tiny and exact
    # to float64 precision, and against the textbook expression wherever that one still has digits (t > -15)
    yl = np.linspace(-12.0, -3.0, 91)
    tl = math.sqrt(2.0 / math.pi) * (yl + 0.044715 * yl ** 3)
    e2 = np.exp(2.0 * tl)
    assert np.allclose(layer.gelu_tanh(yl), yl * e2 / (1.0 + e2), rtol=1e-13, atol=0)
    ok = tl > -15
    assert np.allclose(layer.gelu_tanh(yl[ok]), 0.5 * yl[ok] * (1.0 + np.tanh(tl[ok])), rtol=1e-3, atol=0)
    assert layer.gelu_tanh(-9.0) < 0 and abs(layer.gelu_tanh(-9.0)) > 1e-30      # not flushed to zero


def test_mlp_forward_is_the_two_layers_with_the_quantizer_in_between():
    """mlp_forward against a brute-force restatement on a tiny MLP: FC1 by the layer oracle's own brute-force-pinned
    forward, GeLU element by element in Python floats, Q(Z) with the CALLER's amax (delayed scaling: a stale, larger
    amax must change the scales), FC2 by Python triple loops over the dequantized codes; and the staged inputs
    (Z_given) are honoured."""
    import math
    rng = np.random.default_rng(3)
    M, K, N1, N2, r_t = 8, 64, 32, 16, 16
    bf = nvfp4.bf16_round
    X = bf(rng.standard_normal((M, K)).astype(np.float32))
    R1 = bf((rng.standard_normal((N1, K)) * 0.05).astype(np.float32)); R2 = bf((rng.standard_normal((N2, N1)) * 0.05).astype(np.float32))
    D1 = bf((rng.standard_normal((K, r_t)) * 0.1).astype(np.float32)); U1 = bf((rng.standard_normal((r_t, N1)) * 0.1).astype(np.float32))
    D2 = bf((rng.standard_normal((N1, r_t)) * 0.1).astype(np.float32)); U2 = bf((rng.standard_normal((r_t, N2)) * 0.1).astype(np.float32))
    q1, q2 = layer.quantize_weight(R1), layer.quantize_weight(R2)
    f1 = layer.forward(X, q1, D1, U1, prescale=True)
    Zb = np.zeros((M, N1), np.float32)
    for m in range(M):
        for n in range(N1):
            v = float(f1["Y"][m, n])
            Zb[m, n] = 0.5 * v * (1.0 + math.tanh(math.sqrt(2.0 / math.pi) * (v + 0.044715 * v ** 3)))
    Zb = nvfp4.bf16_round_from_f64(Zb.astype(np.float64))
    z_amax = np.float32(2.0) * nvfp4.tensor_amax(Zb)          # a stale amax from "the previous step"
    out = layer.mlp_forward(X, q1, D1, U1, q2, D2, U2, z_amax=z_amax, y1_amax=nvfp4.tensor_amax(f1["Y"]))
    assert np.array_equal(out["Y1"], f1["Y"]) and np.array_equal(out["Z"], Zb)
    qZ = nvfp4.quantize_blockwise(Zb, 1, amax_t=z_amax)
    assert np.array_equal(out["qZ"]["codes"], qZ["codes"]) and np.array_equal(out["qZ"]["sf"], qZ["sf"])
    assert not np.array_equal(qZ["sf"], nvfp4.quantize_blockwise(Zb, 1)["sf"])     # the caller's amax is what counts
    assert np.array_equal(out["qY1"]["codes"], nvfp4.quantize_blockwise(f1["Y"], 1)["codes"])
    dZ, dR2 = nvfp4.dequantize_unscaled(qZ), nvfp4.dequantize_unscaled(q2)
    alpha2 = float(np.float32(qZ["g_dec"]) * np.float32(q2["g_dec"]))
    H2 = Zb.astype(np.float64) @ D2.astype(np.float64)
    H2s = nvfp4.bf16_round_from_f64(H2 / alpha2).astype(np.float64)
    Y2 = np.zeros((M, N2))
    for m in range(M):
        for n in range(N2):
            acc = 0.0
            for k in range(N1):
                acc += dZ[m, k] * dR2[n, k]
            for j in range(r_t):
                acc += H2s[m, j] * float(U2[j, n])
            Y2[m, n] = alpha2 * acc
    assert np.array_equal(out["Y2"], nvfp4.bf16_round_from_f64(Y2))
    # staged comparison: a given Z replaces the oracle's own
    Z2 = Zb.copy(); Z2[0, 0] += np.float32(0.5)
    out2 = layer.mlp_forward(X, q1, D1, U1, q2, D2, U2, z_amax=z_amax, y1_amax=nvfp4.tensor_amax(f1["Y"]), Z_given=Z2)
    assert np.array_equal(out2["Z"], Z2) and not np.array_equal(out2["Y2"][0], out["Y2"][0])
    # GeLU backward on the saved 4-bit pre-activation, element by element
    G = bf((rng.standard_normal((M, N1)) * 1e-2).astype(np.float32))
    dY1 = layer.gelu_backward_saved4(G, out["qY1"])
    y1q = nvfp4.dequantize(out["qY1"])
    for m in (0, 3, 7):
        for n in (0, 5, 31):
            v = float(y1q[m, n]); c = math.sqrt(2.0 / math.pi)
            t = math.tanh(c * (v + 0.044715 * v ** 3))
            want = float(G[m, n]) * (0.5 * (1 + t) + 0.5 * v * (1 - t * t) * c * (1 + 3 * 0.044715 * v * v))
            assert dY1[m, n] == nvfp4.bf16_round_from_f64(np.float64(want))
