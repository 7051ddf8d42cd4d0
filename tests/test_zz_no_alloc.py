"""ft_quantize_blockwise_static (no caller workspace, no device allocation: the scratch is a static device array
inside the library) against ft_quantize_blockwise with a workspace, on calls in a row that share the array.
Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from paper_2607_05711_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2607_05711_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def t16(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda().to(torch.bfloat16)


def run_both(B, x, D, other, amax):
    """Quantize + project x through both entry points; returns the two sets of outputs as numpy arrays."""
    rows, cols = x.shape
    r_t = D.shape[1]
    outs = []
    for static in (False, True):
        q = B.QTensor(rows, cols)
        h = torch.full((rows, r_t), 7.0, dtype=torch.bfloat16, device="cuda")
        hs = torch.full((rows, r_t), 7.0, dtype=torch.bfloat16, device="cuda")
        if static:
            B.ft_quantize_blockwise_static(x, q, tensor_amax=amax, down=D, h_out=h, hs_out=hs, other_dec_scale=other)
        else:
            ws = B.new_workspace(rows, cols, 0, r_t, "cuda")
            B.ft_quantize_blockwise(x, q, tensor_amax=amax, down=D, h_out=h, hs_out=hs, other_dec_scale=other,
                                    workspace=ws)
        torch.cuda.synchronize()
        outs.append(dict(codes=q.codes.cpu().numpy(), sf=q.sf.cpu().numpy(),
                         g_dec=q.tensor_dec_scale.cpu().numpy().view(np.uint32),
                         h=h.float().cpu().numpy(), hs=hs.float().cpu().numpy()))
    return outs


def compare(ref, got):
    # integer / byte work: bit-exact
    assert np.array_equal(got["codes"], ref["codes"])
    assert np.array_equal(got["sf"], ref["sf"])
    assert np.array_equal(got["g_dec"], ref["g_dec"])
    # H, Hs: the staged bar of the parity tests (O-11): <= 2e-3 relative Frobenius, >= 99 % identical
    for k in ("h", "hs"):
        a, b = got[k].astype(np.float64), ref[k].astype(np.float64)
        assert np.isfinite(a).all()
        assert np.linalg.norm(a - b) <= 2e-3 * np.linalg.norm(b)
        assert (got[k] == ref[k]).mean() >= 0.99


def test_static_scratch_two_calls_in_a_row(B):
    rng = synth.make_rng(4242)
    other = torch.tensor([1.0 / 1024], dtype=torch.float32, device="cuda")
    # call 1: amax unknown (single-pass route: grid barrier + amax words of the control region), ragged rows
    x1 = t16(synth.outlier_normal(rng, 1100, 1024))
    D1 = t16(synth.normal(rng, (1024, 64), 0.01))
    ref, got = run_both(B, x1, D1, other, None)
    compare(ref, got)
    # call 2, straight behind it on the same array: another shape, another rank, amax given (streaming route);
    # the array still holds call 1's slots
    x2 = t16(synth.student_t_grad(rng, 700, 3072))
    D2 = t16(synth.normal(rng, (3072, 32), 0.01))
    amax = B.ft_tensor_amax(x2)
    ref, got = run_both(B, x2, D2, other, amax)
    compare(ref, got)
    # call 3: call 1 again gives call 1's bits again
    ref, got = run_both(B, x1, D1, other, None)
    compare(ref, got)


def test_static_scratch_limit(B):
    L = B.lib()
    cap = L.ft_static_scratch_bytes()
    assert cap == 8 << 20
    assert L.ft_static_scratch_needed(4608, 64) <= cap        # the FLUX-shaped activations fit
    assert L.ft_static_scratch_needed(4608, 128) > cap
    x = torch.zeros(256, 128, dtype=torch.bfloat16, device="cuda")
    D = torch.zeros(128, 128, dtype=torch.bfloat16, device="cuda")
    q = B.QTensor(256, 128)
    h = torch.zeros(256, 128, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(B.FtError, match="workspace"):
        B.ft_quantize_blockwise_static(x, q, down=D, h_out=h)
    # without a projection any size goes through
    B.ft_quantize_blockwise_static(x, q)
    torch.cuda.synchronize()
    assert not bool(q.codes.any())     # zeros quantize to code 0
