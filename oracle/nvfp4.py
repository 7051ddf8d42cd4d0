"""Oracle: NVFP4 block quantizer Q(.) -- TEST INFRASTRUCTURE, not product code.

What the paper fixes (PAPER.md = /root/reference/PAPER.md):
  * "W~ = Round(W / s) with scaling factor s" and "group-wise scaling"
    (section 2.3).
  * the 4-bit format is "NVFP4" (section 3.1) -- by name only.
  * weights use "block-wise quantization with a 16x16 granularity", the
    alternative being "group-wise (1x16)" (Table 5 at 240-243);
    blocks make Q(R)^T the same codes and scales as Q(R).
  * Q is "applied offline for the residual weights R and dynamically for
    activations X".

Everything the paper leaves open is pinned by the readings Q1..Q5 / O-1..O-8 of
DESIGN.md (taken from SURVEY.md section 8(c)); each function below names the
reading it follows.  The algorithm is written step by step in that order, with
no blocking or fusion, so it can be checked against DESIGN.md by eye.

Pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
  e2m1_encode / e4m3_encode : exhaustive comparison with the host conversion
      routines of CUDA's cuda_fp4.h / cuda_fp8.h (an independent source), and
      tests/golden/e2m1_ties.txt.
  quantize_blockwise        : hand-worked blocks tests/golden/nvfp4_blocks.txt,
      half-ULP error bound, amax -> largest code, idempotence on exactly
      representable data, transposition identity for 16x16 blocks.
  bf16 helpers              : comparison with torch's bfloat16 cast.
Parity that stays unpinned against the authors' own bits: the paper never
states the tensor-scale rule, the float32 operation order or the rounding mode
(O-3..O-6); this oracle is the definition for this build.
"""
import numpy as np

# ---------------------------------------------------------------- bf16 helpers


def bf16_round(x):
    """Round float64/float32 values to the nearest bfloat16 (ties to even) and
    return them as float32.  bf16 = the top 16 bits of an IEEE binary32."""
    x32 = np.asarray(x, dtype=np.float32)
    bits = x32.view(np.uint32).astype(np.uint64)
    lsb = (bits >> np.uint64(16)) & np.uint64(1)
    rounded = (bits + np.uint64(0x7FFF) + lsb) >> np.uint64(16)
    out = (rounded << np.uint64(16)).astype(np.uint32)
    return out.view(np.float32).reshape(x32.shape)


def bf16_round_from_f64(x):
    """float64 -> bf16 with a single rounding (no double rounding through
    float32): the bf16 neighbours of x are found on the float64 value."""
    x = np.asarray(x, dtype=np.float64)
    # bf16 has 8 significand bits (7 stored).  Scale so that one bf16 ulp == 1.
    mant, exp = np.frexp(x)                      # x = mant * 2**exp, 0.5<=|mant|<1
    exp = np.maximum(exp, -125)                  # float32/bf16 subnormal range
    scaled = np.ldexp(x, 8 - exp)                # |scaled| in [128, 256) for normals
    r = np.rint(scaled)                          # ties to even
    out = np.ldexp(r, exp - 8)
    return out.astype(np.float32)                # exact: result is a bf16 value


def bf16_to_bits(x):
    """float32 array holding bf16-representable values -> uint16 bit patterns."""
    x32 = np.ascontiguousarray(x, dtype=np.float32)
    return (x32.view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def bits_to_bf16(bits):
    """uint16 bf16 bit patterns -> float32 values."""
    b = np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return b.view(np.float32)

# --------------------------------------------------- Q1: element grid (E2M1)

# Magnitudes of codes 0..7; bit 3 of a code is the sign (Q1).
E2M1_VALUES = np.array([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0], dtype=np.float64)
# Midpoints between neighbouring magnitudes and, for each, whether a value that
# lands exactly on it goes UP (the upper neighbour has the even code).
_E2M1_MID = np.array([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0], dtype=np.float64)
_E2M1_TIE_UP = np.array([False, True, False, True, False, True, False])


def e2m1_encode(v):
    """Q1: round-to-nearest, ties to the even code, saturate at 6.
    The sign bit is the sign bit of the input, including -0.0 and negative
    values that round to zero (code 8)."""
    v = np.asarray(v, dtype=np.float32)
    mag = np.abs(v).astype(np.float64)
    code = np.zeros(v.shape, dtype=np.uint8)
    for mid, up in zip(_E2M1_MID, _E2M1_TIE_UP):
        code += (mag >= mid) if up else (mag > mid)
    sign = np.signbit(v).astype(np.uint8)
    return (code | (sign << 3)).astype(np.uint8)


def e2m1_decode(code):
    code = np.asarray(code, dtype=np.uint8)
    mag = E2M1_VALUES[code & 7]
    return np.where((code & 8) != 0, -mag, mag)


# ------------------------------------------- Q2: block-scale grid (E4M3, >= 0)


def e4m3_decode(b):
    """value = (1 + m/8) * 2**(e-7) for e = 1..15, (m/8) * 2**-6 for e = 0."""
    b = np.asarray(b, dtype=np.uint8)
    e = (b >> 3).astype(np.int64) & 15
    m = (b & 7).astype(np.float64)
    normal = (1.0 + m / 8.0) * np.exp2((e - 7).astype(np.float64))
    sub = (m / 8.0) * 2.0 ** -6
    return np.where(e == 0, sub, normal)


def e4m3_encode(t):
    """Q2: non-negative float32 -> E4M3 byte, round to nearest, ties to even
    code, saturate at 448 (0x7E); 0x7F is never produced."""
    t = np.asarray(t, dtype=np.float32).astype(np.float64)
    t = np.minimum(t, 448.0)
    out = np.zeros(t.shape, dtype=np.uint8)
    # subnormal range: multiples of 2**-9 below 2**-6 (m = 8 is code 0x08 = 2**-6)
    sub = t < 2.0 ** -6
    m_sub = np.rint(t * 2.0 ** 9)                      # ties to even
    out = np.where(sub, m_sub.astype(np.uint8), out)
    # normal range
    tn = np.where(sub, 1.0, t)                         # dummy 1.0 where unused
    frac, exp = np.frexp(tn)                           # tn = frac * 2**exp, frac in [0.5,1)
    e_unb = exp - 1                                    # tn = (2*frac) * 2**e_unb
    m = np.rint((2.0 * frac - 1.0) * 8.0)              # 0..8, ties to even
    carry = m == 8
    e_unb = np.where(carry, e_unb + 1, e_unb)
    m = np.where(carry, 0, m)
    code = ((e_unb + 7).astype(np.int64) << 3) | m.astype(np.int64)
    code = np.minimum(code, 0x7E)                      # satfinite
    out = np.where(sub, out, code.astype(np.uint8))
    return out.astype(np.uint8)


# ----------------------------------------------- Q3: tensor-level FP32 scale

F32 = np.float32
FLT_MAX = np.finfo(np.float32).max


def tensor_scales(amax_t):
    """Q3: g_enc = 2688 / amax_t (2688 = 6 * 448; IEEE float32 divide),
    g_enc = 1 if amax_t == 0, clamped to FLT_MAX; g_dec = 1 / g_enc."""
    amax_t = F32(amax_t)
    if amax_t == F32(0.0):
        g_enc = F32(1.0)
    else:
        with np.errstate(over="ignore"):
            g_enc = F32(2688.0) / amax_t
        if not np.isfinite(g_enc):
            g_enc = FLT_MAX
    g_dec = F32(1.0) / g_enc
    return F32(g_enc), F32(g_dec)


def tensor_amax(x):
    """a0: amax_t = max |x| over the whole tensor (exact: inputs are bf16)."""
    x = np.asarray(x, dtype=np.float32)
    return F32(np.max(np.abs(x))) if x.size else F32(0.0)


# ------------------------------ O-6': stochastic rounding of the element codes (NEXT-4 variant)

PHILOX_M0, PHILOX_M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
PHILOX_W0, PHILOX_W1 = np.uint32(0x9E3779B9), np.uint32(0xBB67AE85)


def philox4x32_10(counter, key):
    """Philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3", SC'11), the
    counter-based generator both the oracle and the CUDA kernel implement, each on its own.
    counter: uint32 [..., 4], key: uint32 [2] -> uint32 [..., 4].  Ten rounds of
        hi0:lo0 = M0 * c0,  hi1:lo1 = M1 * c2,   c = (hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0),   k += (W0, W1)."""
    c = np.array(counter, dtype=np.uint32, copy=True)
    k0, k1 = np.uint32(key[0]), np.uint32(key[1])
    m32 = np.uint64(0xFFFFFFFF)
    with np.errstate(over="ignore"):
        for _ in range(10):
            p0 = PHILOX_M0 * c[..., 0].astype(np.uint64)
            p1 = PHILOX_M1 * c[..., 2].astype(np.uint64)
            hi0, lo0 = (p0 >> np.uint64(32)).astype(np.uint32), (p0 & m32).astype(np.uint32)
            hi1, lo1 = (p1 >> np.uint64(32)).astype(np.uint32), (p1 & m32).astype(np.uint32)
            c = np.stack([hi1 ^ c[..., 1] ^ k0, lo1, hi0 ^ c[..., 3] ^ k1, lo0], axis=-1)
            k0, k1 = np.uint32(k0 + PHILOX_W0), np.uint32(k1 + PHILOX_W1)
    return c


def sr_uniforms(n_elements, seed, offset):
    """One uniform u in [0, 1) per element of a tensor, in linear (row-major) element order: element idx takes
    word idx % 4 of philox4x32_10(counter = (lo, hi, 0, 0) of the 64-bit value offset + idx // 4, key = (lo, hi) of
    the 64-bit seed), and u = (word >> 8) * 2**-24 (24 bits: exact in float32).  n_elements % 4 == 0."""
    assert n_elements % 4 == 0
    ctr = np.uint64(offset) + np.arange(n_elements // 4, dtype=np.uint64)
    counter = np.zeros((n_elements // 4, 4), dtype=np.uint32)
    counter[:, 0] = (ctr & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    counter[:, 1] = (ctr >> np.uint64(32)).astype(np.uint32)
    key = (np.uint32(np.uint64(seed) & np.uint64(0xFFFFFFFF)), np.uint32(np.uint64(seed) >> np.uint64(32)))
    words = philox4x32_10(counter, key).reshape(-1)
    return ((words >> np.uint32(8)).astype(np.float32) * np.float32(2.0 ** -24)).astype(np.float32)


def e2m1_encode_stochastic(v, u):
    """Stochastic rounding onto the E2M1 grid (reading O-6' of DESIGN.md): with lo <= |v| < hi the neighbouring
    magnitudes, the result is hi with probability (|v| - lo) / (hi - lo) and lo otherwise -- decided by
    `u * (hi - lo) < |v| - lo` on the element's uniform u -- so that E[dequant] = v (unbiased) inside the grid.
    |v| >= 6 saturates to 6; a value already on the grid is kept (|v| - lo = 0); the sign bit is the input's.
    Every quantity is exact in float32 (|v| - lo by Sterbenz, hi - lo a power of two, u a 24-bit fraction)."""
    v = np.asarray(v, dtype=np.float32)
    u = np.asarray(u, dtype=np.float32)
    mag = np.abs(v).astype(np.float64)
    grid = E2M1_VALUES
    lo_idx = np.clip(np.searchsorted(grid, mag, side="right") - 1, 0, 7)      # largest grid value <= |v|
    lo = grid[lo_idx]
    hi = grid[np.minimum(lo_idx + 1, 7)]
    step = hi - lo                                                            # 0 at the top of the grid
    up = (u.astype(np.float64) * step < mag - lo) & (lo_idx < 7)
    code = (lo_idx + up).astype(np.uint8)
    sign = np.signbit(v).astype(np.uint8)
    return (code | (sign << 3)).astype(np.uint8)


# ------------------------------------------------------ Q4: per-block quantize


def quantize_blockwise(x, block_rows=1, block_cols=16, amax_t=None, round_mode="nearest", seed=0, offset=0):
    """Q(.) of DESIGN.md Q3-Q5 on a [rows, cols] float32 array of bf16 values.

    round_mode "nearest" (reading O-6, the default) or "stochastic" (O-6', the NEXT-4 variant for gradients):
    the scales are computed the same way; only the last line changes to
        code_i = E2M1_stochastic(float(x_i) * enc_b, u_i),  u_i = sr_uniforms(...)[row * cols + col].

    Blocks are block_rows x block_cols (1x16 for X and G along the reduction
    dim, 16x16 for the residual weights R; O-2).  Every float32
    operation below is one IEEE-754 binary32 round-to-nearest operation, in
    this order, with no fused multiply-add (O-5):

        amax_b = max |x_i|
        t      = (amax_b / 6.0f) * g_enc
        sf8    = E4M3_rne_satfinite(min(t, 448.0f))
        sf     = float(sf8)
        enc_b  = (sf8 == 0) ? 0.0f : 1.0f / (sf * g_dec)
        code_i = E2M1_rne_satfinite(float(x_i) * enc_b)

    Returns a dict: codes [rows, cols] uint8 (one code per element, unpacked),
    packed [rows, cols/2] uint8 (Q5), sf [rows/block_rows, cols/block_cols]
    uint8, g_dec float32, g_enc float32, amax_t float32.
    """
    x = np.ascontiguousarray(x, dtype=np.float32)
    rows, cols = x.shape
    assert rows % block_rows == 0 and cols % block_cols == 0 and cols % 2 == 0
    if amax_t is None:
        amax_t = tensor_amax(x)
    g_enc, g_dec = tensor_scales(amax_t)

    nbr, nbc = rows // block_rows, cols // block_cols
    xb = x.reshape(nbr, block_rows, nbc, block_cols)
    amax_b = np.max(np.abs(xb), axis=(1, 3)).astype(np.float32)        # [nbr, nbc]
    t = (amax_b / F32(6.0)).astype(np.float32)                         # divide ...
    with np.errstate(over="ignore"):
        t = (t * g_enc).astype(np.float32)                             # ... then multiply
    sf8 = e4m3_encode(np.minimum(t, F32(448.0)))
    sf = e4m3_decode(sf8).astype(np.float32)                           # exact
    prod = (sf * g_dec).astype(np.float32)
    with np.errstate(divide="ignore", over="ignore"):
        enc_b = np.where(sf8 == 0, F32(0.0), F32(1.0) / prod).astype(np.float32)
    with np.errstate(over="ignore", invalid="ignore"):
        scaled = (xb * enc_b[:, None, :, None]).astype(np.float32)
    if round_mode == "nearest":
        codes = e2m1_encode(scaled).reshape(rows, cols)
    elif round_mode == "stochastic":
        u = sr_uniforms(rows * cols, seed, offset).reshape(nbr, block_rows, nbc, block_cols)
        codes = e2m1_encode_stochastic(scaled, u).reshape(rows, cols)
    else:
        raise ValueError(round_mode)
    return {
        "codes": codes,
        "packed": pack_codes(codes),
        "sf": sf8,
        "g_dec": g_dec,
        "g_enc": g_enc,
        "amax_t": F32(amax_t),
        "block_rows": block_rows,
        "block_cols": block_cols,
        "scaled": scaled.reshape(rows, cols),      # x_i * enc_b, kept for the invariants tests
    }


def dequantize(q):
    """dequant(x_i) = E2M1(code_i) * sf * g_dec, evaluated in float64."""
    codes = q["codes"]
    rows, cols = codes.shape
    br, bc = q["block_rows"], q["block_cols"]
    sf = e4m3_decode(q["sf"])                                           # float64
    sf_full = np.repeat(np.repeat(sf, br, axis=0), bc, axis=1)
    return e2m1_decode(codes) * sf_full * np.float64(q["g_dec"])


def dequantize_unscaled(q):
    """E2M1(code_i) * sf without the tensor scale (what the tensor core sums)."""
    codes = q["codes"]
    br, bc = q["block_rows"], q["block_cols"]
    sf = e4m3_decode(q["sf"])
    sf_full = np.repeat(np.repeat(sf, br, axis=0), bc, axis=1)
    return e2m1_decode(codes) * sf_full


# ------------------------------------------------------------- Q5: packing


def pack_codes(codes):
    """Byte j of a row holds element 2j in bits 0-3 and element 2j+1 in bits 4-7."""
    codes = np.asarray(codes, dtype=np.uint8)
    return (codes[:, 0::2] | (codes[:, 1::2] << 4)).astype(np.uint8)


def unpack_codes(packed):
    packed = np.asarray(packed, dtype=np.uint8)
    rows, half = packed.shape
    out = np.empty((rows, 2 * half), dtype=np.uint8)
    out[:, 0::2] = packed & 0xF
    out[:, 1::2] = packed >> 4
    return out


def sf_expand_rows(sf, block_rows):
    """Row-major per-row scales sf_R[n][kb] = S[n / block_rows][kb] (Q5)."""
    return np.repeat(np.asarray(sf, dtype=np.uint8), block_rows, axis=0)


def sf_tile128x4_offset(r, c, n_col_blocks):
    """Byte offset of scale (row r, 16-wide block c) in the tile-interleaved
    layout the tensor core's scale-factor copy expects (Q5 / H-2):
    512-byte tiles of 128 rows x 4 blocks, tiles ordered with the block index
    fastest.  A pure permutation (plus zero padding) of the row-major layout."""
    tiles_c = (n_col_blocks + 3) // 4
    tile = (r // 128) * tiles_c + (c // 4)
    return tile * 512 + (r % 32) * 16 + ((r % 128) // 32) * 4 + (c % 4)


def sf_to_tile128x4(sf_rows):
    """[rows, nblk] uint8 per-row scales -> flat tile-interleaved byte array,
    zero padded to 128 rows x 4 blocks."""
    sf_rows = np.asarray(sf_rows, dtype=np.uint8)
    rows, nblk = sf_rows.shape
    tiles_r, tiles_c = (rows + 127) // 128, (nblk + 3) // 4
    out = np.zeros(tiles_r * tiles_c * 512, dtype=np.uint8)
    r, c = np.meshgrid(np.arange(rows), np.arange(nblk), indexing="ij")
    out[sf_tile128x4_offset(r, c, nblk)] = sf_rows
    return out
