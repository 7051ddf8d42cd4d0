"""Offline weight preparation (harness utility, not a kernel): the SVDQuant-style split of
PAPER.md:77-80 (Eq. 1), W ~= R + L1 L2, under reading O-13 of DESIGN.md.  Runs once per layer in
torch float64; the hot path only ever sees its outputs (R, L1, L2 in bf16)."""
import torch


def split_weight(W_bf16, r_s):
    """W [N x K] bf16 -> (R [N x K], L1 [K x r_s], L2t [N x r_s]) in bf16, with
    W ~= R + (L1 @ L2t^T)^T.  L1 = V_r sqrt(S_r), L2 = sqrt(S_r) U_r^T from the float64 SVD;
    R absorbs the bf16 rounding of L1, L2.  r_s = 0 returns W itself."""
    N, K = W_bf16.shape
    if r_s == 0:
        z = W_bf16.new_zeros
        return W_bf16.clone(), z((K, 0)), z((N, 0))
    W = W_bf16.double()
    # top-r_s subspace by the Gram matrix of the smaller side (exact, cheaper than a full SVD)
    U, S, Vh = torch.linalg.svd(W, full_matrices=False)
    rs = S[:r_s].sqrt()
    L1 = (Vh[:r_s].T * rs).to(torch.bfloat16)            # K x r_s
    L2t = (U[:, :r_s] * rs).to(torch.bfloat16)           # N x r_s  (= L2^T)
    R = (W - L2t.double() @ L1.double().T).to(torch.bfloat16)
    return R, L1, L2t


def random_range_split(W_bf16, r_s, seed=0):
    """Cheap stand-in for split_weight on large layers (randomized range finder, one pass):
    still an exact identity W = R + (L1 L2)^T up to the bf16 rounding of R.  Used by bench.py,
    where throughput does not depend on which rank-r_s subspace the stabilizer spans."""
    N, K = W_bf16.shape
    if r_s == 0:
        return split_weight(W_bf16, 0)
    g = torch.Generator(device=W_bf16.device)
    g.manual_seed(seed)
    W = W_bf16.float()
    Q, _ = torch.linalg.qr(W @ torch.randn(K, r_s, device=W.device, generator=g))   # N x r_s
    L2t = Q.to(torch.bfloat16)
    L1 = (W.T @ Q).to(torch.bfloat16)
    R = (W - L2t.float() @ L1.float().T).to(torch.bfloat16)
    return R, L1, L2t
