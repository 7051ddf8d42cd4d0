"""Seeded synthetic inputs for the BASELINE.json configs.

Serves BOTH the CPU oracle's tests and the CUDA path's tests/bench, and so holds
none of the method's arithmetic: it only draws random tensors with the shapes
and value distributions BASELINE.json prescribes and rounds them to bf16
(input preparation).  The SVD weight split (Eq. 1) is NOT here.

Recipe: rng = numpy.random.Generator(numpy.random.Philox(seed)), one generator
per config, tensors drawn in the order listed in DESIGN.md; outlier channel
indices are drawn BEFORE the tensor they scale; float32 -> bf16 by RNE.
These tensors stand in for FLUX.1-dev activations / weights / gradients, which
are not available here (no dataset item or trained weight is reproduced).
"""
import math

import numpy as np


def to_bf16_f32(x):
    """float32 -> nearest bf16 (ties to even), returned as float32."""
    x32 = np.ascontiguousarray(x, dtype=np.float32)
    b = x32.view(np.uint32).astype(np.uint64)
    b = (b + np.uint64(0x7FFF) + ((b >> np.uint64(16)) & np.uint64(1))) >> np.uint64(16)
    return (b << np.uint64(16)).astype(np.uint32).view(np.float32).reshape(x32.shape)


def bf16_bits(x):
    """float32 array of bf16-representable values -> uint16 bit patterns."""
    x32 = np.ascontiguousarray(x, dtype=np.float32)
    return (x32.view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def from_bf16_bits(bits):
    b = np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return b.view(np.float32)


def make_rng(seed):
    return np.random.Generator(np.random.Philox(seed))


def outlier_normal(rng, rows, cols, frac=0.01, factor=50.0):
    """N(0,1) with ceil(frac*cols) channels (columns) scaled by `factor`."""
    n_out = int(math.ceil(frac * cols)) if frac > 0 else 0
    idx = rng.choice(cols, size=n_out, replace=False) if n_out else np.zeros(0, np.int64)
    x = rng.standard_normal((rows, cols), dtype=np.float32)
    if n_out:
        x[:, idx] *= np.float32(factor)
    return to_bf16_f32(x)


def gelu_tanh(z):
    z = z.astype(np.float32)
    return (0.5 * z * (1.0 + np.tanh(0.7978845608028654 * (z + 0.044715 * z ** 3)))).astype(np.float32)


def mlp_down_input(rng, rows, cols, frac=0.005, factor=30.0):
    """C3 down-projection input: bf16(gelu_tanh(N(0,1))) with frac of channels x factor."""
    n_out = int(math.ceil(frac * cols))
    idx = rng.choice(cols, size=n_out, replace=False)
    z = rng.standard_normal((rows, cols), dtype=np.float32)
    x = to_bf16_f32(gelu_tanh(z))
    x[:, idx] *= np.float32(factor)
    return to_bf16_f32(x)


def normal(rng, shape, sigma):
    return to_bf16_f32(rng.standard_normal(shape, dtype=np.float32) * np.float32(sigma))


def student_t_grad(rng, rows, cols, nu=3.0, scale=1e-3):
    g = rng.standard_t(nu, size=(rows, cols)).astype(np.float32) * np.float32(scale)
    return to_bf16_f32(g)


def layer_inputs(seed, M, K, N, r, x_kind="outlier"):
    """One triple-branch layer's raw inputs in draw order X, W, A, B, dY.
    W is the un-split weight [N x K]; the caller applies Eq. 1."""
    rng = make_rng(seed)
    if x_kind == "outlier":
        X = outlier_normal(rng, M, K, 0.01, 50.0)
    elif x_kind == "gelu":
        X = mlp_down_input(rng, M, K, 0.005, 30.0)
    else:
        raise ValueError(x_kind)
    W = normal(rng, (N, K), 0.02)
    A = normal(rng, (K, r), 0.01)
    B = normal(rng, (r, N), 0.01)
    dY = student_t_grad(rng, M, N)
    return {"X": X, "W": W, "A": A, "B": B, "dY": dY}


# BASELINE.json configs (shorthand of DESIGN.md): name -> (seed, M, K, N, r_s, r, x_kind)
CONFIGS = {
    "C1": (0, 256, 3072, 3072, 32, 16, "outlier"),
    "C2": (1, 4608, 3072, 9216, 32, 32, "outlier"),
    "C3u": (2, 4608, 3072, 12288, 32, 64, "outlier"),
    "C3d": (2, 4608, 12288, 3072, 32, 64, "gelu"),
}

# C4: quantizer-only sweep tensors (rows, cols), seed 3
C4_SHAPES = [(4608, 3072), (4608, 12288), (4608, 15360), (9216, 3072)]

# C5: FLUX.1-dev-shaped DiT linear layers: (name, count, M, K, N); r_s = r = 32, seed 4
C5_LAYERS = [
    ("dual.img.qkv", 19, 4096, 3072, 9216), ("dual.img.proj", 19, 4096, 3072, 3072),
    ("dual.img.mlp_up", 19, 4096, 3072, 12288), ("dual.img.mlp_down", 19, 4096, 12288, 3072),
    ("dual.txt.qkv", 19, 512, 3072, 9216), ("dual.txt.proj", 19, 512, 3072, 3072),
    ("dual.txt.mlp_up", 19, 512, 3072, 12288), ("dual.txt.mlp_down", 19, 512, 12288, 3072),
    ("single.lin1", 38, 4608, 3072, 21504), ("single.lin2", 38, 4608, 15360, 3072),
]
