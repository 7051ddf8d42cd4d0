"""The product's own Eq. 1 split (paper_2607_05711_b200/prepare.py, reading O-13) against the
oracle's (oracle/layer.py::prepare_weight).  CPU only: both run a float64 SVD (torch / numpy LAPACK)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import layer as olayer
from oracle import nvfp4
from paper_2607_05711_b200 import prepare, synth


def _canon(L1, L2):
    """SVD factors are unique up to one sign per singular pair: make the largest entry of each L1 column positive."""
    s = np.sign(L1[np.abs(L1).argmax(axis=0), np.arange(L1.shape[1])])
    s[s == 0] = 1
    return L1 * s[None, :], L2 * s[:, None]


@pytest.mark.parametrize("N,K,r_s", [(96, 64, 8), (128, 192, 32), (64, 64, 0)])
def test_split_weight_matches_oracle_prepare_weight(N, K, r_s):
    rng = synth.make_rng(N + K + r_s)
    W = synth.normal(rng, (N, K), 0.02)
    W[:, 3] *= 40.0                                        # an outlier channel for the stabilizer to pick up
    W = synth.to_bf16_f32(W)
    Ro, L1o, L2o = olayer.prepare_weight(W, r_s)
    R, L1, L2t = prepare.split_weight(torch.from_numpy(W).to(torch.bfloat16), r_s)
    R, L1, L2 = R.float().numpy(), L1.float().numpy(), L2t.float().numpy().T
    assert R.shape == (N, K) and L1.shape == (K, r_s) and L2.shape == (r_s, N)
    if r_s == 0:
        assert np.array_equal(R, Ro)
        return
    # the identity that defines R: it absorbs the bf16 rounding of the factors (bit for bit, from the product's OWN factors)
    want_R = nvfp4.bf16_round_from_f64(W.astype(np.float64) - (L1.astype(np.float64) @ L2.astype(np.float64)).T)
    assert np.array_equal(R, want_R)
    # and the factors are the oracle's (two LAPACK builds agree to the last float64 bits, so after the bf16
    # rounding all but a stray near-tie are identical)
    a1, a2 = _canon(L1, L2)
    b1, b2 = _canon(L1o, L2o)
    assert (a1 == b1).mean() >= 0.999 and (a2 == b2).mean() >= 0.999
    assert (R == Ro).mean() >= 0.999
    # Eckart-Young direction: the residual is no larger than W and the outlier column is mostly gone
    assert np.linalg.norm(R) < np.linalg.norm(W)
    assert np.abs(R[:, 3]).max() < 0.25 * np.abs(W[:, 3]).max()
