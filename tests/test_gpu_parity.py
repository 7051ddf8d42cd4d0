"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bars (BASELINE.json north_star, O-11): FP4 codes, block scales and the tensor scale
bit-exact; GEMM / branch outputs within relative Frobenius error 1e-3 of the oracle's float64
accumulation of the same dequantized operands (the oracle consumes the GPU's own bf16 low-rank
intermediate, which is itself checked against the oracle's to 2e-3 and >= 99 % identical)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import layer as olayer
from oracle import nvfp4
from paper_2607_05711_b200 import synth

pytestmark = pytest.mark.gpu
TOL = 1e-3


@pytest.fixture(scope="module")
def B():
    from paper_2607_05711_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def t16(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda().to(torch.bfloat16)


def npf(t):
    return t.float().cpu().numpy()


def rel(a, b):
    d = np.linalg.norm(np.asarray(b, np.float64))
    return np.linalg.norm(np.asarray(a, np.float64) - np.asarray(b, np.float64)) / (d if d > 0 else 1.0)


def sf_ntile_layout(sf_rows, ntile):
    """The scales of a weight operand cut to output tiles of `ntile` rows (include/fourtune.h, ft_qtensor::sf_ntile),
    from per-row scales [rows x nblk]: an index function of its own, written from the header's description."""
    rows, nblk = sf_rows.shape
    k64, tiles = nblk // 4, (rows + ntile - 1) // ntile
    out = np.zeros(tiles * k64 * 1024, dtype=np.uint8)
    r, c = np.meshgrid(np.arange(rows), np.arange(nblk), indexing="ij")
    nt, rt = r // ntile, r % ntile
    half, r128 = rt // 128, rt % 128
    off = ((nt * k64 + c // 4) * 2 + half) * 512 + (r128 % 32) * 16 + (r128 // 32) * 4 + c % 4
    out[off] = sf_rows
    return out


def assert_q_equal(qt, q, layout, B):
    rows, cols = q["codes"].shape
    assert np.array_equal(qt.codes.cpu().numpy(), q["packed"])
    sf = qt.sf.cpu().numpy()
    if layout == B.FT_SF_ROWMAJOR:
        assert np.array_equal(sf.reshape(q["sf"].shape), q["sf"])
    else:
        assert np.array_equal(sf, nvfp4.sf_to_tile128x4(nvfp4.sf_expand_rows(q["sf"], q["block_rows"])))
    assert qt.tensor_dec_scale.cpu().numpy().view(np.uint32)[0] == np.float32(q["g_dec"]).view(np.uint32)


# ------------------------------------------------------------------ a0
@pytest.mark.parametrize("n", [8, 24, 1000, 4608 * 3072 + 3])
def test_amax(B, n):
    rng = synth.make_rng(n)
    x = synth.to_bf16_f32(rng.standard_normal(n + 8, dtype=np.float32) * 3)[:n]
    x[n // 2] = -77.5
    xt = t16(np.concatenate([x, np.zeros(8, np.float32)]))[:n]
    got = B.ft_tensor_amax(xt).cpu().numpy()[0]
    assert got == nvfp4.tensor_amax(x) == np.float32(77.5)


# ------------------------------------------------------------------ a1 / a3 / a6: quantizer
QCASES = [  # rows, cols, kind, layout
    (1, 64, "x", 0), (16, 64, "g", 1), (128, 256, "x", 0), (130, 512, "x", 1), (257, 1024, "g", 1),
    (256, 3072, "x", 1), (256, 3072, "g", 1), (384, 15360, "x", 1)]


@pytest.fixture(params=[0, 1], ids=["single_pass", "two_pass"])
def qmode(request, B):
    """Both routes to the tensor amax: inside the quantize kernel (grid barrier, tensor resident
    in shared memory) and the separate k_amax launch followed by the streaming kernel."""
    B.debug_set_quantize_mode(request.param)
    yield request.param
    B.debug_set_quantize_mode(0)


# BASELINE.json configs[3] (C4): the four tensors of the quantizer sweep at full size
C4_CASES = [(rows, cols, "x", 1) for rows, cols in synth.C4_SHAPES]


@pytest.mark.parametrize("rows,cols,kind,layout", QCASES + [(2304, 3072, "x", 1), (4608, 3072, "g", 1)] + C4_CASES)
def test_quantize_1x16_bit_exact(B, qmode, rows, cols, kind, layout):
    rng = synth.make_rng(rows * 131 + cols)
    x = synth.outlier_normal(rng, rows, cols) if kind == "x" else synth.student_t_grad(rng, rows, cols)
    out = B.QTensor(rows, cols, 1, layout)
    B.ft_quantize_blockwise(t16(x), out)
    assert_q_equal(out, nvfp4.quantize_blockwise(x, 1), layout, B)


def test_quantize_with_caller_amax(B):
    """tensor_amax supplied by the caller (delayed / static scaling): streaming kernel only."""
    rng = synth.make_rng(77)
    x = synth.outlier_normal(rng, 300, 1024)
    xt = t16(x)
    out = B.QTensor(300, 1024, 1, B.FT_SF_TILE128x4)
    B.ft_quantize_blockwise(xt, out, tensor_amax=B.ft_tensor_amax(xt))
    assert_q_equal(out, nvfp4.quantize_blockwise(x, 1), B.FT_SF_TILE128x4, B)


@pytest.mark.parametrize("rows,cols,layout", [(1, 64, 0), (130, 512, 1), (300, 1024, 0), (2304, 3072, 1)])
def test_quantize_stochastic_rounding_bit_exact(B, rows, cols, layout):
    """NEXT-4 / O-6': FT_ROUND_STOCHASTIC against the oracle's stochastic quantizer on the same Philox4x32-10 stream
    (64-bit seed, an offset that crosses 2^32): codes, scales and tensor scale bit for bit.  Counter-based: the lower
    part of the tensor quantized alone, with the whole tensor's amax and the offset advanced, gives the same bits."""
    rng = synth.make_rng(rows * 7 + cols)
    x = synth.student_t_grad(rng, rows, cols)
    seed, offset = 0x1234567890ABCDEF, (1 << 32) - 100
    out = B.QTensor(rows, cols, 1, layout)
    B.ft_quantize_blockwise(t16(x), out, round_mode=B.FT_ROUND_STOCHASTIC, seed=seed, offset=offset)
    q = nvfp4.quantize_blockwise(x, 1, round_mode="stochastic", seed=seed, offset=offset)
    assert_q_equal(out, q, layout, B)
    qn = nvfp4.quantize_blockwise(x, 1)
    assert np.array_equal(q["sf"], qn["sf"]) and (q["codes"] != qn["codes"]).mean() > 0.05   # same scales, other codes
    if rows >= 130:
        a = 64
        amax = torch.tensor([float(nvfp4.tensor_amax(x))], dtype=torch.float32, device="cuda")
        part = B.QTensor(rows - a, cols, 1, layout)
        B.ft_quantize_blockwise(t16(x[a:]), part, tensor_amax=amax, round_mode=B.FT_ROUND_STOCHASTIC, seed=seed,
                                offset=offset + a * cols // 4)
        assert np.array_equal(part.codes.cpu().numpy(), q["packed"][a:])
    # the mode is a variant of the plain quantizer: no fused projection, no 16x16 blocks
    with pytest.raises(B.FtError):
        B.ft_quantize_blockwise(t16(x), out, down=t16(np.zeros((cols, 16), np.float32)), round_mode=B.FT_ROUND_STOCHASTIC)


def test_dgrad_with_stochastically_rounded_gradient(B):
    """The use the variant is meant for: Q(G) by stochastic rounding feeding the dgrad GEMM (ft_quantize_blockwise +
    ft_gemm4 with Q(R)^T), against the oracle's float64 product of the same dequantized operands."""
    M, K, N = 300, 512, 768
    rng = synth.make_rng(91)
    G = synth.student_t_grad(rng, M, N)
    W = synth.normal(rng, (N, K), 0.02)
    L = B.Layer(t16(W), None, None, 0, 0)
    qg = B.QTensor(M, N)
    B.ft_quantize_blockwise(t16(G), qg, round_mode=B.FT_ROUND_STOCHASTIC, seed=5, offset=17)
    dx = torch.zeros(M, K, dtype=torch.bfloat16, device="cuda")
    B.ft_gemm4(qg, L.r_nmajor, None, None, dx)
    oG = nvfp4.quantize_blockwise(G, 1, round_mode="stochastic", seed=5, offset=17)
    oR = nvfp4.quantize_blockwise(W, 16)
    assert_q_equal(qg, oG, B.FT_SF_TILE128x4, B)
    alpha = np.float64(np.float32(oG["g_dec"]) * np.float32(oR["g_dec"]))
    uG, uR = nvfp4.dequantize_unscaled(oG), nvfp4.dequantize_unscaled(oR)
    want = nvfp4.bf16_round_from_f64(alpha * (uG @ uR))
    got = npf(dx)
    assert rel(got, want) <= TOL and (got == want).mean() >= 0.95
    elementwise_ok(got, want, alpha * (np.abs(uG) @ np.abs(uR)), "dX")


def test_quantize_16x16_blocks_on_activations_through_the_gemm(B):
    """NEXT-4's third arm (Table 5 at 240-243; reading O-2 keeps 1x16 for activations): an ACTIVATION
    quantized in 16x16 blocks -- ft_quantize_blockwise(block_rows = 16), scales expanded per row by the TILE128x4
    layout -- fed to ft_gemm4 against 16x16 weights, compared with the oracle; and it is the coarser quantizer."""
    M, K, N = 256, 512, 384
    rng = synth.make_rng(92)
    X = synth.outlier_normal(rng, M, K)
    W = synth.normal(rng, (N, K), 0.02)
    qx = B.QTensor(M, K, 16, B.FT_SF_TILE128x4)
    B.ft_quantize_blockwise(t16(X), qx)
    oX = nvfp4.quantize_blockwise(X, 16)
    assert_q_equal(qx, oX, B.FT_SF_TILE128x4, B)
    L = B.Layer(t16(W), None, None, 0, 0)
    y = torch.zeros(M, N, dtype=torch.bfloat16, device="cuda")
    B.ft_gemm4(qx, L.r_kmajor, None, None, y)
    oW = nvfp4.quantize_blockwise(W, 16)
    alpha = np.float64(np.float32(oX["g_dec"]) * np.float32(oW["g_dec"]))
    uX, uW = nvfp4.dequantize_unscaled(oX), nvfp4.dequantize_unscaled(oW)
    want = nvfp4.bf16_round_from_f64(alpha * (uX @ uW.T))
    got = npf(y)
    assert rel(got, want) <= TOL and (got == want).mean() >= 0.95
    elementwise_ok(got, want, alpha * (np.abs(uX) @ np.abs(uW).T), "Y")
    # Table 5's direction on activations too: 16x16 blocks lose more than 1x16 (an outlier channel costs its 15
    # neighbouring ROWS their resolution as well)
    assert rel(nvfp4.dequantize(oX), X) > rel(nvfp4.dequantize(nvfp4.quantize_blockwise(X, 1)), X)


def test_quantize_degenerate_inputs(B):
    # all zeros; -0.0; a block of tiny values next to the tensor maximum; saturating ties
    x = np.zeros((128, 128), np.float32)
    out = B.QTensor(128, 128, 1, 0)
    B.ft_quantize_blockwise(t16(x), out)
    assert_q_equal(out, nvfp4.quantize_blockwise(x, 1), 0, B)
    x[0, :16] = [0.5, -1, 1.5, 2, 3, -6, 0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5, 0, -0.0, 4]
    x[1, 16:32] = 1e-6
    x[2, 32:48] = -0.0
    x[3, :] = synth.to_bf16_f32(np.linspace(-6, 6, 128, dtype=np.float32))
    x[5, 64] = 2688.0
    x = synth.to_bf16_f32(x)
    B.ft_quantize_blockwise(t16(x), out)
    assert_q_equal(out, nvfp4.quantize_blockwise(x, 1), 0, B)
    # caller-supplied tensor amax (static scaling) is honoured
    amax = torch.tensor([6.0 * 448], dtype=torch.float32, device="cuda")
    B.ft_quantize_blockwise(t16(x), out, tensor_amax=amax)
    assert_q_equal(out, nvfp4.quantize_blockwise(x, 1, amax_t=np.float32(2688.0)), 0, B)


@pytest.mark.parametrize("N,K", [(64, 64), (256, 512), (320, 448), (832, 192), (3072, 3072)])
def test_weight_quantize_16x16_and_pack(B, N, K):
    rng = synth.make_rng(N + K)
    W = synth.normal(rng, (N, K), 0.02)
    q = nvfp4.quantize_blockwise(W, 16)
    L = B.Layer(t16(W), None, None, 0, 0)
    assert_q_equal(L.q_rowmajor, q, B.FT_SF_ROWMAJOR, B)
    assert_q_equal(L.r_kmajor, q, B.FT_SF_TILE128x4, B)
    # Q(R)^T is the same codes and scales re-indexed: compare with the
    # transposed oracle object, and with the oracle quantizing R^T afresh (pin P-4)
    qT = dict(q, codes=np.ascontiguousarray(q["codes"].T), sf=np.ascontiguousarray(q["sf"].T))
    qT["packed"] = nvfp4.pack_codes(qT["codes"])
    assert_q_equal(L.r_nmajor, qT, B.FT_SF_TILE128x4, B)
    q2 = nvfp4.quantize_blockwise(np.ascontiguousarray(W.T), 16)
    assert np.array_equal(q2["packed"], qT["packed"]) and np.array_equal(q2["sf"], qT["sf"])
    # the same scales once more, cut to the 224-wide tiles of the GEMM (both orientations)
    for qt, qo in ((L.r_kmajor, q), (L.r_nmajor, qT)):
        assert qt.ntile == 224
        want = sf_ntile_layout(nvfp4.sf_expand_rows(qo["sf"], 16), 224)
        assert np.array_equal(qt.sf_ntile.cpu().numpy(), want)


@pytest.mark.parametrize("rows,cols,r_t,kind", [(128, 512, 16, "x"), (200, 1024, 64, "x"), (256, 3072, 48, "x"),
                                                (384, 2048, 96, "g"), (130, 4096, 128, "g"), (1, 64, 32, "x"),
                                                (2000, 128, 64, "x"), (4608, 3072, 64, "x"), (2304, 3072, 128, "g"),
                                                # 481 row tiles: more than the workspace has per-tile counters for
                                                # (480): k_finalize_h falls back to the grid-wide wait
                                                (61500, 64, 16, "g")] +
                         [(rows, cols, 32, "x") for rows, cols in synth.C4_SHAPES])
def test_fused_projection(B, qmode, rows, cols, r_t, kind):
    rng = synth.make_rng(rows + cols + r_t)
    x = synth.outlier_normal(rng, rows, cols) if kind == "x" else synth.student_t_grad(rng, rows, cols)
    D = synth.normal(rng, (cols, r_t), 0.01)
    other = np.float32(3.7e-5)
    out = B.QTensor(rows, cols, 1, B.FT_SF_TILE128x4)
    h = torch.zeros(rows, r_t, dtype=torch.bfloat16, device="cuda")
    hs = torch.zeros_like(h)
    B.ft_quantize_blockwise(t16(x), out, down=t16(D), h_out=h, hs_out=hs,
                            other_dec_scale=torch.tensor([other], device="cuda"))
    q = nvfp4.quantize_blockwise(x, 1)
    assert_q_equal(out, q, B.FT_SF_TILE128x4, B)   # fusing the projection must not change a bit
    Hex = x.astype(np.float64) @ D.astype(np.float64)
    Ho = nvfp4.bf16_round_from_f64(Hex)
    alpha = np.float64(np.float32(q["g_dec"]) * other)
    Hso = nvfp4.bf16_round_from_f64(Hex / alpha)
    for got, want in ((npf(h), Ho), (npf(hs), Hso)):
        assert rel(got, want) <= 2e-3
        assert (got == want).mean() >= 0.99
        # every element within one bf16 ulp of the oracle's, plus the fp32 accumulation error
        # of a length-`cols` dot product on elements that cancel to nearly zero
        assert np.all(np.abs(got - want) <= np.abs(want) * 2.0 ** -7 + 1e-5 * np.abs(want).max())


def test_fused_projection_random_shapes(B, qmode):
    """Seeded sweep over ragged shapes: every way a CTA's chunk range can cut the row tiles (one chunk per
    row tile, ranges spanning several tiles, more CTAs than chunks, ...) against the oracle."""
    rng = synth.make_rng(2024)
    for case in range(36):
        rows = int(rng.integers(1, 900))
        cols = 64 * int(rng.integers(1, 40))
        r_t = 16 * int(rng.integers(0, 9))
        x = synth.outlier_normal(rng, rows, cols) if case % 2 else synth.student_t_grad(rng, rows, cols)
        out = B.QTensor(rows, cols, 1, B.FT_SF_TILE128x4 if case % 3 else B.FT_SF_ROWMAJOR)
        q = nvfp4.quantize_blockwise(x, 1)
        if r_t == 0:
            B.ft_quantize_blockwise(t16(x), out)
            assert_q_equal(out, q, out.sf_layout, B)
            continue
        D = synth.normal(rng, (cols, r_t), 0.01)
        h = torch.zeros(rows, r_t, dtype=torch.bfloat16, device="cuda")
        hs = torch.zeros_like(h)
        other = np.float32(1.3e-3)
        B.ft_quantize_blockwise(t16(x), out, down=t16(D), h_out=h, hs_out=hs,
                                other_dec_scale=torch.tensor([other], device="cuda"))
        assert_q_equal(out, q, out.sf_layout, B), (rows, cols, r_t)
        Hex = x.astype(np.float64) @ D.astype(np.float64)
        alpha = np.float64(np.float32(q["g_dec"]) * other)
        for got, want in ((npf(h), nvfp4.bf16_round_from_f64(Hex)), (npf(hs), nvfp4.bf16_round_from_f64(Hex / alpha))):
            assert rel(got, want) <= 2e-3, (rows, cols, r_t)
            assert (got == want).mean() >= 0.98, (rows, cols, r_t)


# ------------------------------------------------------------------ a2 / a4 / a5: the layer
def make_layer(B, seed, M, K, N, r_s, r, x_kind="outlier", ntile=224):
    d = synth.layer_inputs(seed, M, K, N, max(r, 1), x_kind)
    R, L1, L2 = olayer.prepare_weight(d["W"], r_s)
    D_f = np.concatenate([L1, d["A"][:, :r]], 1).astype(np.float32)
    U_f = np.concatenate([L2, d["B"][:r, :]], 0).astype(np.float32)
    r_t = r_s + r
    L = B.Layer(t16(R), t16(D_f) if r_t else None, t16(U_f.T) if r_t else None, r_s, r, ntile=ntile)
    return d, R, D_f, U_f, L


def range_finder_split(W, r_s, seed):
    """Eq. 1 with a cheap rank-r_s subspace (one randomized range-finder pass instead of a full SVD): still
    W = R + (L1 L2)^T up to the bf16 rounding of R, and any L1, L2 is a valid stabilizer for parity purposes (the
    oracle and the CUDA path receive the same R, L1, L2).  float64 numpy, input preparation only."""
    N, K = W.shape
    if r_s == 0:
        return W.astype(np.float32), np.zeros((K, 0), np.float32), np.zeros((0, N), np.float32)
    rng = synth.make_rng(seed + 100)
    W64 = W.astype(np.float64)
    Qb, _ = np.linalg.qr(W64 @ rng.standard_normal((K, r_s)))        # N x r_s
    L2 = nvfp4.bf16_round_from_f64(Qb.T)                              # r_s x N
    L1 = nvfp4.bf16_round_from_f64((Qb.T @ W64).T)                    # K x r_s
    R = nvfp4.bf16_round_from_f64(W64 - (L1.astype(np.float64) @ L2.astype(np.float64)).T)
    return R, L1, L2


def make_layer_fast(B, seed, M, K, N, r_s, r, x_kind="outlier", ntile=224):
    """make_layer with the range-finder split: for shapes where the full SVD of W would dominate the test."""
    d = synth.layer_inputs(seed, M, K, N, max(r, 1), x_kind)
    R, L1, L2 = range_finder_split(d["W"], r_s, seed)
    D_f = np.concatenate([L1, d["A"][:, :r]], 1).astype(np.float32)
    U_f = np.concatenate([L2, d["B"][:r, :]], 0).astype(np.float32)
    r_t = r_s + r
    L = B.Layer(t16(R), t16(D_f) if r_t else None, t16(U_f.T) if r_t else None, r_s, r, ntile=ntile)
    return d, R, D_f, U_f, L


def run_layer(B, L, X, G, M, K, N, r_t, r, fused_bwd=False):
    y = torch.zeros(M, N, dtype=torch.bfloat16, device="cuda")
    dx = torch.zeros(M, K, dtype=torch.bfloat16, device="cuda")
    h = torch.zeros(M, max(r_t, 1), dtype=torch.bfloat16, device="cuda")
    p = torch.zeros_like(h)
    ws = torch.zeros(B.ft_workspace_bytes(M, max(K, N), max(K, N), r_t), dtype=torch.uint8, device="cuda")
    qx, qg = B.QTensor(M, K), B.QTensor(M, N)
    xt, gt = t16(X), t16(G)
    scaled = lambda: (npf(B.workspace_hs(ws, M, r_t)) if r_t else None)
    B.ft_linear_fwd(L, xt, y, h, qx, ws)
    torch.cuda.synchronize()
    hs = scaled()
    dA = dBt = None
    if r > 0:
        dA = torch.full((K, r), 7.0, dtype=torch.float32, device="cuda")
        dBt = torch.full((N, r), 7.0, dtype=torch.float32, device="cuda")
    if fused_bwd:
        B.ft_linear_bwd(L, xt, gt, h, dx, p, dA, dBt, qg, ws)
    else:
        B.ft_linear_bwd_dgrad(L, gt, dx, p, qg, ws)
    torch.cuda.synchronize()
    ps = scaled()
    if r > 0 and not fused_bwd:
        B.ft_lora_wgrad(L, xt, gt, h, p, dA, dBt)
    return dict(y=npf(y), dx=npf(dx), h=npf(h), p=npf(p), hs=hs, ps=ps, qx=qx, qg=qg,
                dA=None if dA is None else dA.cpu().numpy(), dBt=None if dBt is None else dBt.cpu().numpy(),
                xt=xt, gt=gt, ht=h, pt=p)


LAYER_CASES = [  # seed, M, K, N, r_s, r, tile_n (fourtune_debug.h: 0 auto, 128/192/256 1-CTA, 1224/1240/1256 pair kernel)
    (11, 1, 64, 64, 0, 0, 0), (12, 128, 256, 128, 0, 0, 256), (13, 130, 320, 192, 16, 16, 0),
    (14, 256, 512, 384, 16, 16, 192), (15, 200, 1024, 768, 32, 64, 256), (16, 300, 576, 448, 32, 32, 128),
    (17, 129, 2048, 640, 0, 16, 192),
    # the CTA-pair kernel with 224-wide tiles: N = 64 (one ragged tile of 64), 192, 448 (two full tiles), 640 (224 + 224
    # + 192), 768 (3 x 224 + 96: a 32-column unit in a ragged tile), K with a partial stage; and the 256-wide one forced
    (18, 1, 64, 64, 0, 0, 1224), (19, 130, 320, 192, 16, 16, 1224), (20, 300, 576, 448, 32, 32, 1224),
    (21, 129, 2048, 640, 0, 16, 1224), (22, 200, 1024, 768, 32, 64, 1224), (23, 260, 448, 1024, 16, 96, 1224),
    (24, 300, 576, 448, 32, 32, 1256), (25, 200, 1024, 768, 32, 64, 1256),
    (26, 1, 64, 64, 0, 0, 1240), (27, 130, 320, 192, 16, 16, 1240), (28, 300, 576, 448, 32, 32, 1240),
    (29, 129, 2048, 640, 0, 16, 1240), (30, 260, 448, 1024, 16, 96, 1240), (31, 200, 1024, 960, 32, 64, 1240),
    (32, 140, 256, 256, 16, 16, 1240)]   # N = 240 + 16: the launcher must not run a 16-column tile (falls back to 256)


@pytest.mark.parametrize("seed,M,K,N,r_s,r,bn", LAYER_CASES)
def test_layer_small(B, seed, M, K, N, r_s, r, bn):
    B.debug_set_gemm_tile_n(bn)
    try:
        d, R, D_f, U_f, L = make_layer(B, seed, M, K, N, r_s, r, ntile=240 if bn == 1240 else 224)
        out = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r)
    finally:
        B.debug_set_gemm_tile_n(0)
    check_layer(B, d, R, D_f, U_f, out, r_s, r)


@pytest.mark.parametrize("seed,M,K,N,r_s,r", [(21, 130, 320, 192, 16, 16), (22, 300, 1024, 768, 32, 32),
                                               (23, 1000, 512, 2048, 0, 16), (24, 64, 2048, 640, 32, 64)])
def test_layer_fused_backward(B, qmode, seed, M, K, N, r_s, r):
    """ft_linear_bwd = ft_linear_bwd_dgrad + ft_lora_wgrad.  Both of its schedules: G small enough for
    the single-pass quantizer (qmode 0 at these sizes) and the dB^T pass that also finds the amax of G
    (forced by qmode 1, which switches the single-pass route off)."""
    d, R, D_f, U_f, L = make_layer(B, seed, M, K, N, r_s, r)
    out = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r, fused_bwd=True)
    check_layer(B, d, R, D_f, U_f, out, r_s, r)
    ref = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r)
    # same amax -> identical codes; P (and through Ps, dX) may differ in the last bf16 bit of a few
    # elements: the two schedules run the quantize kernel with different grids, i.e. a different (each
    # time fixed) association of the fp32 partial sums of P
    assert np.array_equal(out["qg"].codes.cpu().numpy(), ref["qg"].codes.cpu().numpy())
    for k in ("p", "dx"):
        assert (out[k] == ref[k]).mean() >= 0.999 and rel(out[k], ref[k]) < 1e-3
    assert rel(out["dA"], ref["dA"]) < 1e-5 and rel(out["dBt"], ref["dBt"]) < 1e-5


def elementwise_ok(got, want, absdot, what):
    """Every element of a bf16 GEMM output against the oracle's (O-11): both sides are one bf16 rounding
    of nearly the same real number, so they differ by at most one bf16 ulp (<= 2^-7 |want|) -- plus the fp32
    accumulation error of the tensor core, which only shows on elements that cancel: 2^-20 of the sum of the
    absolute products (sixteen fp32 ulps of headroom over the 2^-24 of a single rounding)."""
    bound = np.abs(want) * 2.0 ** -7 + absdot * 2.0 ** -20
    bad = np.abs(got.astype(np.float64) - want.astype(np.float64)) > bound
    assert not bad.any(), "%s: %d of %d elements out of bound, first at %s" % (
        what, int(bad.sum()), bad.size, np.argwhere(bad)[0])


def check_layer(B, d, R, D_f, U_f, out, r_s, r, rows=None):
    """Full comparison, or on a row sample (rows) for sizes the oracle cannot finish whole."""
    X, G = d["X"], d["dY"]
    r_t = r_s + r
    qR = olayer.quantize_weight(R)
    ax, ag = nvfp4.tensor_amax(X), nvfp4.tensor_amax(G)
    sel = slice(None) if rows is None else rows
    # (i) codes / scales bit-exact, on the whole tensors
    assert_q_equal(out["qx"], nvfp4.quantize_blockwise(X, 1), B.FT_SF_TILE128x4, B)
    assert_q_equal(out["qg"], nvfp4.quantize_blockwise(G, 1), B.FT_SF_TILE128x4, B)
    f = olayer.forward(X[sel], qR, D_f, U_f, prescale=True, x_amax=ax,
                       H_given=None if r_t == 0 else out["hs"][sel])
    b = olayer.dgrad(G[sel], qR, D_f, U_f, prescale=True, g_amax=ag,
                     P_given=None if r_t == 0 else out["ps"][sel])
    if r_t:
        # (ii) the low-rank intermediates against the oracle's own
        for got, want in ((out["h"][sel], f["H"]), (out["hs"][sel], f["Hs"]), (out["p"][sel], b["P"]),
                          (out["ps"][sel], b["Ps"])):
            assert rel(got, want) <= 2e-3 and (got == want).mean() >= 0.99
    # (iii) outputs, both cast to bf16: norm, identical fraction, and a bound on EVERY element
    assert rel(out["y"][sel], f["Y"]) <= TOL
    assert rel(out["dx"][sel], b["dX"]) <= TOL
    assert (out["y"][sel] == f["Y"]).mean() >= 0.95 and (out["dx"][sel] == b["dX"]).mean() >= 0.95
    aR = np.abs(nvfp4.dequantize_unscaled(qR))
    absdot_f = np.abs(nvfp4.dequantize_unscaled(f["qX"])) @ aR.T
    absdot_b = np.abs(nvfp4.dequantize_unscaled(b["qG"])) @ aR
    if r_t:
        absdot_f += np.abs(out["hs"][sel].astype(np.float64)) @ np.abs(U_f.astype(np.float64))
        absdot_b += np.abs(out["ps"][sel].astype(np.float64)) @ np.abs(D_f.astype(np.float64)).T
    elementwise_ok(out["y"][sel], f["Y"], f["alpha"] * absdot_f, "Y")
    elementwise_ok(out["dx"][sel], b["dX"], b["alpha"] * absdot_b, "dX")
    if r > 0 and rows is None:
        w = olayer.wgrad(X, G, out["h"], out["p"], r_s)
        assert rel(out["dA"], w["dA"]) <= TOL and rel(out["dBt"].T, w["dB"]) <= TOL


# Shapes whose tile count exceeds 2 x 74 in one GEMM direction, so that every CTA pair of the persistent kernel
# runs three or more tiles there -- both accumulators, the hand-over of the scale columns, the barrier phase wrap
# -- with EVERY output element compared (the full-size cases below only sample rows).  Ragged M.
MULTI_TILE_CASES = [   # seed, M, K, N, r_s, r
    (71, 1100, 512, 7936, 32, 32),     # forward: 5 x 31 = 155 tiles of 256 x 256
    (72, 1100, 7936, 512, 32, 64),     # dgrad:   155 tiles, 31 K stages forward
    (73, 2304, 4352, 4352, 32, 64),    # 9 x 17 = 153 tiles in both directions, r_t = 96
    (74, 1300, 320, 6400, 0, 16),      # 6 x 25 = 150 tiles, a partial K stage, one low-rank group of 16
    (75, 2304, 4352, 4352, 0, 0),      # no low-rank stage at all
]


@pytest.mark.parametrize("bn", [1224, 1240, 1256], ids=["pair224", "pair240", "pair256"])
@pytest.mark.parametrize("seed,M,K,N,r_s,r", MULTI_TILE_CASES)
def test_layer_multi_tile_per_cta_pair(B, seed, M, K, N, r_s, r, bn):
    """Both tile widths of the CTA-pair GEMM: 256 (scale columns overlaid on the draining accumulator, hand-over
    per tile) and 224 (scale columns of their own, ragged last tile of every row of tiles)."""
    B.debug_set_gemm_tile_n(bn)
    try:
        d, R, D_f, U_f, L = make_layer_fast(B, seed, M, K, N, r_s, r, ntile=240 if bn == 1240 else 224)
        out = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r, fused_bwd=r > 0)
    finally:
        B.debug_set_gemm_tile_n(0)
    check_layer(B, d, R, D_f, U_f, out, r_s, r)


def test_gemm4_alone_multi_tile(B):
    """ft_gemm4 by itself (no low-rank term) on 150 tiles, every element against the oracle's float64 product of the
    dequantized operands (pin P-5: r_s = r = 0 reduces the layer to a plain block-scaled GEMM)."""
    M, K, N = 1500, 576, 6400
    rng = synth.make_rng(76)
    X = synth.outlier_normal(rng, M, K)
    W = synth.normal(rng, (N, K), 0.02)
    qx = B.QTensor(M, K)
    B.ft_quantize_blockwise(t16(X), qx)
    L = B.Layer(t16(W), None, None, 0, 0)
    y = torch.zeros(M, N, dtype=torch.bfloat16, device="cuda")
    B.ft_gemm4(qx, L.r_kmajor, None, None, y)
    oX, oW = nvfp4.quantize_blockwise(X, 1), nvfp4.quantize_blockwise(W, 16)
    alpha = np.float64(np.float32(oX["g_dec"]) * np.float32(oW["g_dec"]))
    uX, uW = nvfp4.dequantize_unscaled(oX), nvfp4.dequantize_unscaled(oW)
    want = nvfp4.bf16_round_from_f64(alpha * (uX @ uW.T))
    got = npf(y)
    assert rel(got, want) <= TOL and (got == want).mean() >= 0.95
    elementwise_ok(got, want, alpha * (np.abs(uX) @ np.abs(uW).T), "Y")


def test_layer_degenerate_branches(B):
    """B = 0 -> branch 3 contributes nothing to Y and dX, dA = 0, dB != 0; A = 0 -> dB = 0 (pin P-5)."""
    M, K, N, r_s, r = 128, 256, 128, 16, 16
    d, R, D_f, U_f, _ = make_layer(B, 31, M, K, N, r_s, r)
    U0 = U_f.copy(); U0[r_s:, :] = 0
    L0 = B.Layer(t16(R), t16(D_f), t16(U0.T), r_s, r)
    o0 = run_layer(B, L0, d["X"], d["dY"], M, K, N, r_s + r, r)
    Ls = B.Layer(t16(R), t16(D_f[:, :r_s]), t16(U_f[:r_s].T), r_s, 0)
    os_ = run_layer(B, Ls, d["X"], d["dY"], M, K, N, r_s, 0)
    assert rel(o0["y"], os_["y"]) <= 1e-3 and np.all(o0["dA"] == 0) and np.any(o0["dBt"] != 0)
    D0 = D_f.copy(); D0[:, r_s:] = 0
    L1 = B.Layer(t16(R), t16(D0), t16(U_f.T), r_s, r)
    o1 = run_layer(B, L1, d["X"], d["dY"], M, K, N, r_s + r, r)
    assert np.all(o1["dBt"] == 0) and np.any(o1["dA"] != 0)


def test_wgrad_accumulate(B):
    M, K, N, r_s, r = 192, 128, 192, 16, 16
    d, R, D_f, U_f, L = make_layer(B, 41, M, K, N, r_s, r)
    o = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r)
    dA = torch.from_numpy(o["dA"]).cuda().clone(); dBt = torch.from_numpy(o["dBt"]).cuda().clone()
    B.ft_lora_wgrad(L, o["xt"], o["gt"], o["ht"], o["pt"], dA, dBt, accumulate=True)
    assert rel(dA.cpu().numpy(), 2 * o["dA"]) <= 1e-5 and rel(dBt.cpu().numpy(), 2 * o["dBt"]) <= 1e-5


@pytest.mark.parametrize("seed,M,K,N,r_s,r", [(51, 1, 64, 64, 0, 16), (52, 130, 320, 192, 16, 16),
                                               (53, 300, 576, 448, 32, 32), (54, 1100, 512, 256, 32, 64),
                                               (55, 2049, 1024, 128, 0, 128), (56, 64, 2048, 640, 16, 48)])
def test_wgrad_saved4(B, seed, M, K, N, r_s, r):
    """NEXT-2 / O-12': ft_lora_wgrad_q4 = Eq. 4 with dequant(Q(X)) as the saved activation, against
    oracle.layer.wgrad_saved4 on the ORACLE's own Q(X).  Ragged M, K % 128 == 64 (half feature tile),
    one and several M slices (M >= 1024: fp32 reductions), every r group count; then accumulate."""
    d, R, D_f, U_f, L = make_layer(B, seed, M, K, N, r_s, r)
    o = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r)
    qX = nvfp4.quantize_blockwise(d["X"], 1)
    assert_q_equal(o["qx"], qX, B.FT_SF_TILE128x4, B)
    w = olayer.wgrad_saved4(qX, d["dY"], o["h"], o["p"], r_s)
    dA = torch.full((K, r), 7.0, dtype=torch.float32, device="cuda")
    dBt = torch.full((N, r), 7.0, dtype=torch.float32, device="cuda")
    B.ft_lora_wgrad_q4(L, o["qx"], o["gt"], o["ht"], o["pt"], dA, dBt)
    torch.cuda.synchronize()
    assert rel(dA.cpu().numpy(), w["dA"]) <= 1e-5, "dA from 4-bit saved activations"
    assert rel(dBt.cpu().numpy().T, w["dB"]) <= TOL
    assert rel(dBt.cpu().numpy(), o["dBt"]) <= 1e-5            # the same kernel as ft_lora_wgrad
    # the two readings of Eq. 4 differ by the quantization error of X, far above the kernel's own error
    assert rel(dA.cpu().numpy(), o["dA"]) > 1e-3
    once = dA.cpu().numpy().copy()
    B.ft_lora_wgrad_q4(L, o["qx"], o["gt"], o["ht"], o["pt"], dA, dBt, accumulate=True)
    torch.cuda.synchronize()
    assert rel(dA.cpu().numpy(), 2 * once) <= 1e-5 and rel(dBt.cpu().numpy(), 2 * o["dBt"]) <= 1e-5


@pytest.mark.parametrize("seed,M,K,N,r_s,r", [(58, 300, 576, 448, 32, 32), (59, 1100, 512, 2048, 16, 16)])
def test_fused_backward_saved4(B, qmode, seed, M, K, N, r_s, r):
    """ft_linear_bwd_q4 (both schedules, see test_layer_fused_backward) = ft_linear_bwd with dA from Q(X)."""
    d, R, D_f, U_f, L = make_layer(B, seed, M, K, N, r_s, r)
    o = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r, fused_bwd=True)
    dx = torch.zeros(M, K, dtype=torch.bfloat16, device="cuda")
    p = torch.zeros_like(o["pt"])
    dA = torch.full((K, r), 7.0, dtype=torch.float32, device="cuda")
    dBt = torch.full((N, r), 7.0, dtype=torch.float32, device="cuda")
    ws = torch.zeros(B.ft_workspace_bytes(M, max(K, N), max(K, N), r_s + r), dtype=torch.uint8, device="cuda")
    qg = B.QTensor(M, N)
    B.ft_linear_bwd_q4(L, o["qx"], o["gt"], o["ht"], dx, p, dA, dBt, qg, ws)
    torch.cuda.synchronize()
    assert torch.equal(qg.codes, o["qg"].codes) and np.array_equal(npf(dx), o["dx"]) and np.array_equal(npf(p), o["p"])
    assert rel(dBt.cpu().numpy(), o["dBt"]) <= 1e-5
    w = olayer.wgrad_saved4(nvfp4.quantize_blockwise(d["X"], 1), d["dY"], o["h"], o["p"], r_s)
    assert rel(dA.cpu().numpy(), w["dA"]) <= 1e-5
    B.ft_linear_bwd_q4(L, o["qx"], o["gt"], o["ht"], dx, p, dA, dBt, qg, ws, accumulate=True)
    torch.cuda.synchronize()
    assert rel(dA.cpu().numpy(), 2 * w["dA"]) <= 1e-5 and rel(dBt.cpu().numpy(), 2 * o["dBt"]) <= 1e-5


def test_wgrad_saved4_errors(B):
    M, K, N, r_s, r = 128, 256, 128, 16, 16
    d, R, D_f, U_f, L = make_layer(B, 57, M, K, N, r_s, r)
    o = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r)
    dA = torch.zeros(K, r, dtype=torch.float32, device="cuda"); dBt = torch.zeros(N, r, dtype=torch.float32, device="cuda")
    with pytest.raises(B.FtError):      # Q(G) has the wrong column count for the X operand
        B.ft_lora_wgrad_q4(L, o["qg"] if N != K else B.QTensor(M, K + 64), o["gt"], o["ht"], o["pt"], dA, dBt)


@pytest.mark.parametrize("M,K,N", [(200, 448, 320), (512, 3072, 1024)])
def test_single_copy_weights(B, M, K, N):
    """NEXT-5: one copy of the 4-bit codes per layer.  ft_weight_transpose_codes rebuilds the
    codes of Q(R)^T into a scratch buffer: the bytes ft_pack_weight wrote (themselves compared with the oracle's
    transposed object in test_weight_quantize_16x16_and_pack), and the dgrad through the scratch is bit-identical."""
    r_s, r = 16, 16
    rng = synth.make_rng(M + K + N)
    W = synth.normal(rng, (N, K), 0.02)
    D = synth.normal(rng, (K, r_s + r), 0.01)
    U = synth.normal(rng, (N, r_s + r), 0.01)
    G = synth.student_t_grad(rng, M, N)
    L = B.Layer(t16(W), t16(D), t16(U), r_s, r)
    q = nvfp4.quantize_blockwise(W, 16)
    want = nvfp4.pack_codes(np.ascontiguousarray(q["codes"].T))
    scratch = torch.full_like(L.r_nmajor.codes, 0xAB)
    B.ft_weight_transpose_codes(L, scratch)
    assert np.array_equal(scratch.cpu().numpy().reshape(K, N // 2), want)
    ws = B.new_workspace(M, max(K, N), max(K, N), r_s + r, "cuda")
    outs = []
    for codes in (L.r_nmajor.codes, scratch):
        L.r_nmajor.codes = codes
        dx = torch.zeros(M, K, dtype=torch.bfloat16, device="cuda")
        p = torch.zeros(M, r_s + r, dtype=torch.bfloat16, device="cuda")
        B.ft_linear_bwd_dgrad(L, t16(G), dx, p, B.QTensor(M, N), ws)
        outs.append(dx.view(torch.int16).cpu().numpy())
    assert np.array_equal(outs[0], outs[1])


def test_forward_with_1x16_weight_blocks(B):
    """The other arm of the paper's granularity ablation (Table 5): group-wise 1x16 weight
    scales.  Forward only -- such scales do not transpose (oracle pin P-4), which is why the layer uses 16x16 --
    composed from the two exported calls: ft_quantize_blockwise(block_rows=1) on the weight, then ft_gemm4."""
    M, K, N = 200, 512, 384
    rng = synth.make_rng(77)
    X = synth.outlier_normal(rng, M, K)
    W = synth.normal(rng, (N, K), 0.02)
    qx, qw = B.QTensor(M, K), B.QTensor(N, K, 1, B.FT_SF_TILE128x4)
    B.ft_quantize_blockwise(t16(X), qx)
    B.ft_quantize_blockwise(t16(W), qw)
    y = torch.zeros(M, N, dtype=torch.bfloat16, device="cuda")
    B.ft_gemm4(qx, qw, None, None, y)
    oX, oW = nvfp4.quantize_blockwise(X, 1), nvfp4.quantize_blockwise(W, 1)
    assert_q_equal(qw, oW, B.FT_SF_TILE128x4, B)
    want = nvfp4.bf16_round_from_f64(nvfp4.dequantize(oX) @ nvfp4.dequantize(oW).T)
    got = npf(y)
    assert rel(got, want) <= TOL and (got == want).mean() >= 0.95
    # and it is the finer quantizer of the two (Table 5's direction) on these weights
    e1 = rel(nvfp4.dequantize(oW), W)
    e16 = rel(nvfp4.dequantize(nvfp4.quantize_blockwise(W, 16)), W)
    assert e1 < e16


def test_fused_backward_accumulate_and_errors(B, qmode):
    """ft_linear_bwd with accumulate=1 adds to dA / dB^T (both schedules); a short workspace is refused
    before anything is enqueued."""
    M, K, N, r_s, r = 300, 256, 320, 16, 32
    d, R, D_f, U_f, L = make_layer(B, 43, M, K, N, r_s, r)
    o = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r)
    dA = torch.from_numpy(o["dA"]).cuda().clone(); dBt = torch.from_numpy(o["dBt"]).cuda().clone()
    dx = torch.zeros(M, K, dtype=torch.bfloat16, device="cuda")
    p = torch.zeros(M, r_s + r, dtype=torch.bfloat16, device="cuda")
    ws = torch.zeros(B.ft_workspace_bytes(M, max(K, N), max(K, N), r_s + r), dtype=torch.uint8, device="cuda")
    B.ft_linear_bwd(L, o["xt"], o["gt"], o["ht"], dx, p, dA, dBt, o["qg"], ws, accumulate=True)
    assert rel(dA.cpu().numpy(), 2 * o["dA"]) <= 1e-5 and rel(dBt.cpu().numpy(), 2 * o["dBt"]) <= 1e-5
    assert (npf(dx) == o["dx"]).mean() >= 0.999
    before = dA.clone()
    with pytest.raises(B.FtError, match="workspace too small"):
        B.ft_linear_bwd(L, o["xt"], o["gt"], o["ht"], dx, p, dA, dBt, o["qg"], ws[:1024])
    torch.cuda.synchronize()
    assert torch.equal(before, dA)


def test_layer_c1_full(B):
    """BASELINE.json configs[0] in full: M=256, K=N=3072, r_s=32, r=16, seed 0."""
    seed, M, K, N, r_s, r, kind = synth.CONFIGS["C1"]
    d, R, D_f, U_f, L = make_layer(B, seed, M, K, N, r_s, r, kind)
    out = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r)
    check_layer(B, d, R, D_f, U_f, out, r_s, r)


@pytest.mark.parametrize("name", ["C2", "C3u", "C3d"])
def test_layer_full_size_sampled(B, name):
    """BASELINE.json configs[1..2] at full size in the launch configuration bench.py times:
    codes/scales compared in full, outputs on sampled rows spanning tiles and the ragged ends
    (rows of Y / dX depend only on their own row of X / G and the tensor amax).  The weight
    split uses a cheap randomized range finder instead of a full SVD: any L1, L2 is a valid
    stabilizer for parity purposes (the oracle receives the same R, L1, L2)."""
    _full_size_sampled(B, *synth.CONFIGS[name])


@pytest.mark.parametrize("name", [l[0] for l in synth.C5_LAYERS])
def test_layer_c5_shapes_sampled(B, name):
    """BASELINE.json configs[4]: ALL ten distinct (M, K, N) of the FLUX.1-dev-shaped layer list (the shapes bench.py
    times and sums into the C5 figure), r_s = r = 32, seed 4, same sampled comparison as above."""
    _, _, M, K, N = next(l for l in synth.C5_LAYERS if l[0] == name)
    _full_size_sampled(B, 4, M, K, N, 32, 32, "outlier")


def sample_rows(M):
    """Rows of a full-size output to compare: in EVERY 256-row tile of the CTA-pair GEMM two rows from each 32-lane
    quarter of each of the two CTAs (rows 3, 40, 77, 110 of the first CTA's 128, 131 - 128 = 3, 42, 72, 122 of the
    second's: TMEM lane quarters 0, 1, 2, 3 = epilogue warps q = 0..3), plus the tile edges and the ragged end."""
    rows = set()
    for t in range((M + 255) // 256):
        rows.update(t * 256 + o for o in (3, 40, 77, 110, 131, 170, 200, 250))
    rows.update((0, 1, 127, 128, 129, 255, 256, M - 129, M - 2, M - 1))
    return np.array(sorted(r for r in rows if 0 <= r < M))


def _full_size_sampled(B, seed, M, K, N, r_s, r, kind):
    d = synth.layer_inputs(seed, M, K, N, r, kind)
    R, L1, L2 = range_finder_split(d["W"], r_s, seed)
    D_f = np.concatenate([L1, d["A"]], 1).astype(np.float32)
    U_f = np.concatenate([L2, d["B"]], 0).astype(np.float32)
    L = B.Layer(t16(R), t16(D_f), t16(U_f.T), r_s, r)
    # the schedule bench.py times: ft_linear_fwd + ft_linear_bwd (C2, C3u: G is too large for the
    # single-pass quantizer -> dB^T pass with the amax of G first; C3d: G fits -> quantize, GEMM, one wgrad)
    out = run_layer(B, L, d["X"], d["dY"], M, K, N, r_s + r, r, fused_bwd=True)
    check_layer(B, d, R, D_f, U_f, out, r_s, r, rows=sample_rows(M))
    # wgrad in full (Eq. 4 is two skinny products: the oracle finishes them at any of these sizes)
    w = olayer.wgrad(d["X"], d["dY"], out["h"], out["p"], r_s)
    assert rel(out["dA"], w["dA"]) <= TOL and rel(out["dBt"].T, w["dB"]) <= TOL
    # the same with 4-bit saved activations (NEXT-2): dA = dequant(Q(X))^T P_lora
    dA4 = torch.zeros(K, r, dtype=torch.float32, device="cuda"); dBt4 = torch.zeros(N, r, dtype=torch.float32, device="cuda")
    B.ft_lora_wgrad_q4(L, out["qx"], out["gt"], out["ht"], out["pt"], dA4, dBt4)
    torch.cuda.synchronize()
    w4 = olayer.wgrad_saved4(nvfp4.quantize_blockwise(d["X"], 1), d["dY"], out["h"], out["p"], r_s)
    assert rel(dA4.cpu().numpy(), w4["dA"]) <= 1e-5
    assert rel(dBt4.cpu().numpy().T, w4["dB"]) <= TOL


# ------------------------------------------------------------------ NEXT-1: MLP fusion
MLP_CASES = [   # seed, M, K, N1, N2, r_s, r1, r2 (LoRA rank of FC2; r_t2 = r_s + r2)
    (81, 300, 320, 384, 256, 16, 16, 32),       # ragged M, partial K stage, two column tiles
    (82, 1024, 512, 3072, 512, 32, 64, 64),     # r_t2 = 96 (the C3 ranks), 64 tiles: one per pair
    (83, 2304, 256, 1920, 320, 16, 16, 16),     # 90 tiles on 74 pairs: ranges that cross a row tile
    (84, 1100, 512, 7680, 256, 32, 32, 80),     # 200 tiles: 2-3 per pair, r_t2 = 112 (the widest H2 accumulator)
]


@pytest.mark.parametrize("seed,M,K,N1,N2,r_s,r1,r2", MLP_CASES)
def test_mlp_fused_forward(B, seed, M, K, N1, N2, r_s, r1, r2):
    """ft_mlp_fwd against oracle.layer.mlp_forward (reading O-16), staged as in O-11: every tensor the CUDA path
    hands from one stage to the next is checked against the oracle's, then fed to the oracle's next stage bit for
    bit -- Q(X), H1/Hs1, Y1, Z = bf16(gelu(Y1)), Q(Z) and Q(Y1) with the CALLER's (stale) amax, H2/Hs2, Y2, and this
    step's amax of Z and Y1."""
    rng = synth.make_rng(seed)
    X = synth.outlier_normal(rng, M, K)
    W1, W2 = synth.normal(rng, (N1, K), 0.05), synth.normal(rng, (N2, N1), 0.02)
    rt1, rt2 = r_s + r1, r_s + r2
    R1, L11, L12 = range_finder_split(W1, r_s, seed)
    R2, L21, L22 = range_finder_split(W2, r_s, seed + 1)
    D1 = np.concatenate([L11, synth.normal(rng, (K, r1), 0.02)], 1).astype(np.float32)
    U1 = np.concatenate([L12, synth.normal(rng, (r1, N1), 0.02)], 0).astype(np.float32)
    D2 = np.concatenate([L21, synth.normal(rng, (N1, r2), 0.02)], 1).astype(np.float32)
    U2 = np.concatenate([L22, synth.normal(rng, (r2, N2), 0.02)], 0).astype(np.float32)
    fc1 = B.Layer(t16(R1), t16(D1), t16(U1.T), r_s, r1, ntile=192)
    fc2 = B.Layer(t16(R2), t16(D2), t16(U2.T), r_s, r2)
    q1, q2 = olayer.quantize_weight(R1), olayer.quantize_weight(R2)
    # "the previous step's" amax: 1.5 x and 0.8 x this step's (so the scales differ from a fresh quantization, and
    # some blocks of Y1 saturate)
    pre = olayer.forward(X, q1, D1, U1, prescale=True)
    z_amax = np.float32(1.5) * nvfp4.tensor_amax(nvfp4.bf16_round_from_f64(olayer.gelu_tanh(pre["Y"])))
    y1_amax = np.float32(0.8) * nvfp4.tensor_amax(pre["Y"])
    dev = "cuda"
    y2 = torch.zeros(M, N2, dtype=torch.bfloat16, device=dev)
    h1 = torch.zeros(M, rt1, dtype=torch.bfloat16, device=dev); h2 = torch.zeros(M, rt2, dtype=torch.bfloat16, device=dev)
    qx, qz, qy1 = B.QTensor(M, K), B.QTensor(M, N1), B.QTensor(M, N1)
    zd = torch.zeros(M, N1, dtype=torch.bfloat16, device=dev); yd = torch.zeros_like(zd)
    za = torch.tensor([z_amax], dtype=torch.float32, device=dev); ya = torch.tensor([y1_amax], dtype=torch.float32, device=dev)
    zn = torch.full((1,), 7.0, dtype=torch.float32, device=dev); yn = torch.full((1,), 7.0, dtype=torch.float32, device=dev)
    ws = B.new_mlp_workspace(M, K, N1, rt1, rt2)
    B.ft_mlp_fwd(fc1, fc2, t16(X), za, ya, y2, h1, h2, qx, qz, qy1, ws, z_amax_next=zn, y1_amax_next=yn, z_debug=zd, y1_debug=yd)
    torch.cuda.synchronize()
    hs1, hs2 = npf(B.workspace_hs(ws, M, rt1)), npf(B.mlp_workspace_hs2(ws, M, rt1, rt2))
    Y1g, Zg = npf(yd), npf(zd)
    # FC1
    assert_q_equal(qx, nvfp4.quantize_blockwise(X, 1), B.FT_SF_TILE128x4, B)
    f1 = olayer.forward(X, q1, D1, U1, prescale=True, H_given=hs1)
    for got, want in ((npf(h1), f1["H"]), (hs1, f1["Hs"])):
        assert rel(got, want) <= 2e-3 and (got == want).mean() >= 0.99
    assert rel(Y1g, f1["Y"]) <= TOL and (Y1g == f1["Y"]).mean() >= 0.95
    aR1 = np.abs(nvfp4.dequantize_unscaled(q1))
    ad = np.abs(nvfp4.dequantize_unscaled(f1["qX"])) @ aR1.T + np.abs(hs1.astype(np.float64)) @ np.abs(U1.astype(np.float64))
    elementwise_ok(Y1g, f1["Y"], f1["alpha"] * ad, "Y1")
    # GeLU on the CUDA path's own Y1: within one bf16 ulp of the float64 evaluation, almost always identical
    Zo = nvfp4.bf16_round_from_f64(olayer.gelu_tanh(Y1g))
    assert (Zg == Zo).mean() >= 0.98
    assert np.all(np.abs(Zg.astype(np.float64) - Zo) <= np.abs(Zo) * 2.0 ** -7 + 1e-30)   # (flush-to-zero below 1e-37)
    # the two quantizers, on the CUDA path's own bits and the caller's amax: bit for bit
    assert_q_equal(qz, nvfp4.quantize_blockwise(Zg, 1, amax_t=z_amax), B.FT_SF_TILE128x4, B)
    assert_q_equal(qy1, nvfp4.quantize_blockwise(Y1g, 1, amax_t=y1_amax), B.FT_SF_TILE128x4, B)
    assert zn.cpu().numpy()[0] == nvfp4.tensor_amax(Zg) and yn.cpu().numpy()[0] == nvfp4.tensor_amax(Y1g)
    # FC2 on that Z
    f2 = olayer.forward(Zg, q2, D2, U2, prescale=True, x_amax=z_amax, H_given=hs2)
    for got, want in ((npf(h2), f2["H"]), (hs2, f2["Hs"])):
        assert rel(got, want) <= 2e-3 and (got == want).mean() >= 0.99
    Y2g = npf(y2)
    assert rel(Y2g, f2["Y"]) <= TOL and (Y2g == f2["Y"]).mean() >= 0.95
    aR2 = np.abs(nvfp4.dequantize_unscaled(q2))
    ad2 = np.abs(nvfp4.dequantize_unscaled(f2["qX"])) @ aR2.T + np.abs(hs2.astype(np.float64)) @ np.abs(U2.astype(np.float64))
    elementwise_ok(Y2g, f2["Y"], f2["alpha"] * ad2, "Y2")
    # and the whole thing is the oracle's mlp_forward when it is handed the same staged tensors
    o = olayer.mlp_forward(X, q1, D1, U1, q2, D2, U2, z_amax=z_amax, y1_amax=y1_amax, Y1_given=Y1g, Z_given=Zg,
                           H1s_given=hs1, H2s_given=hs2)
    assert np.array_equal(o["Y2"], f2["Y"]) and np.array_equal(o["qZ"]["codes"], nvfp4.unpack_codes(qz.codes.cpu().numpy()))
    # GeLU backward on the saved 4-bit pre-activation
    dz = synth.student_t_grad(rng, M, N1)
    dy = torch.zeros(M, N1, dtype=torch.bfloat16, device=dev)
    B.ft_gelu_bwd_q4(t16(dz), qy1, dy)
    want = olayer.gelu_backward_saved4(dz, o["qY1"])
    got = npf(dy)
    assert rel(got, want) <= 2e-3 and (got == want).mean() >= 0.95
    assert np.all(np.abs(got.astype(np.float64) - want) <= np.abs(want) * 2.0 ** -6 + 1e-12)


def test_without_programmatic_launch():
    """FT_PDL=0 switches every programmatic edge (and with it the late-wait modes of the dA kernels and of the
    dgrad GEMM) off: the plain stream-ordered schedule must give the same answers.  Re-runs the fused-backward,
    saved-activation and small-layer parity tests in a fresh process, since the switch is read once per process."""
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, FT_PDL="0")
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_gpu_parity.py", "-x", "-q", "-m", "gpu", "-k",
                        "fused_backward or saved4 or layer_small"], cwd=root, env=env, capture_output=True, text=True,
                       timeout=900)
    assert r.returncode == 0 and " passed" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]


def test_step_under_cuda_graph_capture_ragged_m(B):
    """A forward + backward step with ragged M on the streaming route (G too large for the single-pass quantizer),
    captured into a CUDA graph and replayed: the same bits as the eager step (programmatic edges, the cooperative
    single-pass launch for X and the cluster launches all have to survive capture; nothing in a call may touch the
    host after validation)."""
    M, K, N, r_s, r = 4500, 512, 4096, 32, 32      # 35.2 rows of 128: a ragged last row tile; G = 36.9 MB
    r_t = r_s + r
    d, R, D_f, U_f, L = make_layer(B, 63, M, K, N, r_s, r)
    x, g = t16(d["X"]), t16(d["dY"])
    y = torch.zeros(M, N, dtype=torch.bfloat16, device="cuda"); dx = torch.zeros(M, K, dtype=torch.bfloat16, device="cuda")
    h = torch.zeros(M, r_t, dtype=torch.bfloat16, device="cuda"); p = torch.zeros_like(h)
    ws = B.new_workspace(M, max(K, N), max(K, N), r_t, "cuda")
    qx, qg = B.QTensor(M, K), B.QTensor(M, N)
    dA = torch.zeros(K, r, dtype=torch.float32, device="cuda"); dBt = torch.zeros(N, r, dtype=torch.float32, device="cuda")
    outs = (y, dx, h, p, qx.codes, qx.sf, qg.codes, qg.sf, dBt)

    def step():
        B.ft_linear_fwd(L, x, y, h, qx, ws)
        B.ft_linear_bwd(L, x, g, h, dx, p, dA, dBt, qg, ws)

    step()
    torch.cuda.synchronize()
    want = [t.clone() for t in outs]
    want_dA = dA.clone()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        step()                                     # warm the stream (tensor-map memo, function attributes)
        side.synchronize()
        with torch.cuda.graph(graph, stream=side):
            step()
    for rep in range(3):
        for t in outs:
            t.zero_()
        dA.zero_()
        graph.replay()
        torch.cuda.synchronize()
        for j, (t, w) in enumerate(zip(outs, want)):
            assert torch.equal(t, w), (rep, j)
        assert rel(dA.cpu().numpy(), want_dA.cpu().numpy()) <= 1e-5


def test_back_to_back_steps_without_sync(B):
    """The programmatic-launch shortcuts (dgrad GEMM started beside k_finalize_h, dA kernels started beside the
    GEMM with their wait at the end, clear kernels with programmatic edges) must not let a step see a neighbour's
    half-written buffers: 24 forward+backward steps enqueued back to back with no host sync, alternating two
    inputs through the SAME output and scratch buffers, against the same two steps run alone.  G is large enough
    (37 MB) for the streaming route, i.e. the schedule bench.py times."""
    M, K, N, r_s, r = 4608, 512, 4096, 32, 32
    r_t = r_s + r
    d1, R, D_f, U_f, L = make_layer(B, 61, M, K, N, r_s, r)
    d2 = synth.layer_inputs(62, M, K, N, r)
    xs, gs = [t16(d1["X"]), t16(d2["X"])], [t16(d1["dY"]), t16(d2["dY"])]
    y = torch.zeros(M, N, dtype=torch.bfloat16, device="cuda"); dx = torch.zeros(M, K, dtype=torch.bfloat16, device="cuda")
    h = torch.zeros(M, r_t, dtype=torch.bfloat16, device="cuda"); p = torch.zeros_like(h)
    ws = torch.zeros(B.ft_workspace_bytes(M, max(K, N), max(K, N), r_t), dtype=torch.uint8, device="cuda")
    qx, qg = B.QTensor(M, K), B.QTensor(M, N)
    dA = torch.zeros(K, r, dtype=torch.float32, device="cuda"); dBt = torch.zeros(N, r, dtype=torch.float32, device="cuda")

    def step(i, q4):
        B.ft_linear_fwd(L, xs[i], y, h, qx, ws)
        if q4:
            B.ft_linear_bwd_q4(L, qx, gs[i], h, dx, p, dA, dBt, qg, ws)
        else:
            B.ft_linear_bwd(L, xs[i], gs[i], h, dx, p, dA, dBt, qg, ws)
        return [t.clone() for t in (y, dx, h, p, qx.codes, qg.codes, dA, dBt)]   # stream-ordered copies

    for q4 in (False, True):
        ref = []
        for i in (0, 1):
            torch.cuda.synchronize()
            ref.append(step(i, q4))
            torch.cuda.synchronize()
        got = [step(it & 1, q4) for it in range(24)]
        torch.cuda.synchronize()
        for it, out in enumerate(got):
            want = ref[it & 1]
            for j in range(6):      # Y, dX, H, P, codes: the same bits as the step run alone
                assert torch.equal(out[j], want[j]), (q4, it, j)
            for j in (6, 7):        # dA, dB^T: fp32 reductions in no fixed order
                assert rel(out[j].cpu().numpy(), want[j].cpu().numpy()) <= 1e-5, (q4, it, j)
        # the same with NOTHING between the calls (the clones above are kernels of their own): the last kernel of
        # one step (dA, late wait) is directly followed by the first of the next (clear kernel, programmatic edge)
        for n_steps in (2, 3, 8):
            for it in range(n_steps):
                B.ft_linear_fwd(L, xs[it & 1], y, h, qx, ws)
                if q4:
                    B.ft_linear_bwd_q4(L, qx, gs[it & 1], h, dx, p, dA, dBt, qg, ws)
                else:
                    B.ft_linear_bwd(L, xs[it & 1], gs[it & 1], h, dx, p, dA, dBt, qg, ws)
            torch.cuda.synchronize()
            want = ref[(n_steps - 1) & 1]
            for j, t in enumerate((y, dx, h, p, qx.codes, qg.codes)):
                assert torch.equal(t, want[j]), (q4, n_steps, j)
            assert rel(dA.cpu().numpy(), want[6].cpu().numpy()) <= 1e-5 and rel(dBt.cpu().numpy(), want[7].cpu().numpy()) <= 1e-5
    # and the forward of step 0 is right in the first place (sampled rows against the oracle)
    rows = np.array([0, 127, 128, 2047, M - 1])
    qR = olayer.quantize_weight(R)
    torch.cuda.synchronize()
    B.ft_linear_fwd(L, xs[0], y, h, qx, ws)
    torch.cuda.synchronize()
    hs = npf(B.workspace_hs(ws, M, r_t))
    f = olayer.forward(d1["X"][rows], qR, D_f, U_f, prescale=True, x_amax=nvfp4.tensor_amax(d1["X"]), H_given=hs[rows])
    assert rel(npf(y)[rows], f["Y"]) <= TOL
