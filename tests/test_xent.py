"""not gpu: the oracle of the fused softmax cross-entropy (oracle/xent.py) against closed forms,
invariants and central differences."""
import numpy as np

from oracle.xent import softmax_xent


def test_constant_logits_closed_form():
    T, V = 5, 1000
    x = np.full((T, V), 3.25)
    y = np.array([0, 7, 999, 500, 1])
    loss, d = softmax_xent(x, y, grad_scale=0.5)
    assert np.allclose(loss, np.log(V), rtol=0, atol=1e-13)
    want = np.full((T, V), 0.5 / V)
    want[np.arange(T), y] -= 0.5
    assert np.allclose(d, want, rtol=0, atol=1e-15)


def test_two_level_logits_closed_form():
    # k logits equal to a, the other V - k equal to 0: Z = k e^a + V - k
    V, k, a = 64, 3, 2.0
    x = np.zeros((2, V))
    x[:, :k] = a
    Z = k * np.exp(a) + V - k
    loss, d = softmax_xent(x, np.array([1, 10]))
    assert np.allclose(loss, [np.log(Z) - a, np.log(Z)], atol=1e-13)
    assert np.isclose(d[0, 1], np.exp(a) / Z - 1.0) and np.isclose(d[0, 0], np.exp(a) / Z)
    assert np.isclose(d[1, 10], 1.0 / Z - 1.0) and np.isclose(d[1, 20], 1.0 / Z)


def test_invariants_and_ignored_tokens():
    g = np.random.default_rng(1)
    x = g.normal(0, 4, (7, 333))
    y = g.integers(0, 333, 7)
    y[3] = -100
    loss, d = softmax_xent(x, y, grad_scale=0.125)
    loss2, d2 = softmax_xent(x + 11.0, y, grad_scale=0.125)   # shift invariance
    assert np.allclose(loss, loss2, atol=1e-11) and np.allclose(d, d2, atol=1e-13)
    assert np.allclose(d.sum(axis=1), 0.0, atol=1e-15)        # softmax sums to 1
    assert loss[3] == 0.0 and np.all(d[3] == 0.0)
    assert np.all(loss[[0, 1, 2, 4, 5, 6]] > 0)
    # a very large logit on the label: loss -> 0, gradient -> 0
    x[0, y[0]] = 200.0
    loss3, d3 = softmax_xent(x, y)
    assert loss3[0] < 1e-30 and np.abs(d3[0]).max() < 1e-30


def test_gradient_by_central_differences():
    g = np.random.default_rng(2)
    x = g.normal(0, 2, (3, 17))
    y = np.array([4, 0, 16])
    w = np.array([0.3, -1.2, 2.0])              # dL/dloss_i
    _, d = softmax_xent(x, y)
    h = 1e-6
    for i in range(3):
        for j in range(17):
            xp, xm = x.copy(), x.copy()
            xp[i, j] += h
            xm[i, j] -= h
            num = (softmax_xent(xp, y)[0] @ w - softmax_xent(xm, y)[0] @ w) / (2 * h)
            assert abs(num - w[i] * d[i, j]) < 1e-8
