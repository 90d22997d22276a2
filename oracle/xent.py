"""TEST INFRASTRUCTURE ONLY: oracle of `bs_softmax_xent`, the fused softmax cross-entropy of
PAPER.md:334 ("takes BF16 inputs, and still performs online computations in FP32 precision"):
per token i with logits x_i (bf16 values, read exactly) and label y_i,

    loss_i    = log(sum_j exp(x_ij)) - x_i[y_i]
    dlogits_i = g * (softmax(x_i) - onehot(y_i))        g = the caller's gradient scale

and loss_i = 0, dlogits_i = 0 for a label < 0 (ignored token).  Written as that definition in
fp64 numpy (a row maximum is subtracted inside log-sum-exp, which changes nothing
mathematically).  Pinned in tests/test_xent.py by closed forms (constant logits: loss = ln V,
dlogits = g (1/V - onehot); two-level logits), shift invariance, rows of dlogits summing to 0,
and central differences of the loss.
"""
import numpy as np


def softmax_xent(logits, labels, grad_scale=1.0):
    """logits [T, V] float64 (the exact values of the bf16 inputs), labels [T] int.
    Returns (loss [T] float64, dlogits [T, V] float64)."""
    x = np.asarray(logits, dtype=np.float64)
    y = np.asarray(labels, dtype=np.int64)
    T, V = x.shape
    m = x.max(axis=1, keepdims=True)
    e = np.exp(x - m)
    s = e.sum(axis=1, keepdims=True)
    lse = (m + np.log(s))[:, 0]
    p = e / s
    keep = y >= 0
    yy = np.where(keep, y, 0)
    loss = np.where(keep, lse - x[np.arange(T), yy], 0.0)
    d = p.copy()
    d[np.arange(T), yy] -= 1.0
    d *= grad_scale
    d[~keep] = 0.0
    return loss, d
