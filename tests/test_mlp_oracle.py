"""Pins for the MLP oracle (oracle/mlp_oracle.py) against things other than itself (
Eqs. (18)-(19)): a network worked out by hand, closed forms, invariances, a pure-Python loop."""
import numpy as np
import pytest

from oracle import mlp_oracle as mo


def test_two_layer_network_by_hand():
    # x = (1, -2); W0 = [[1, 2], [-1, 0.5], [0, 1]], b0 = (0.5, 0, -1); W1 = [[1, -1, 2]], b1 = (0.25)
    # pre0 = (1 - 4 + 0.5, -1 - 1, -2 - 1) = (-2.5, -2, -3)
    x = np.array([[1.0, -2.0]])
    W0 = np.array([[1.0, 2.0], [-1.0, 0.5], [0.0, 1.0]]); b0 = np.array([0.5, 0.0, -1.0])
    W1 = np.array([[1.0, -1.0, 2.0]]); b1 = np.array([0.25])
    # leaky ReLU (slope 0.01): h = (-0.025, -0.02, -0.03); pre1 = -0.025 + 0.02 - 0.06 + 0.25 = 0.185
    y = mo.mlp_forward(x, [W0, W1], [b0, b1], "leaky_relu")
    np.testing.assert_allclose(y, [[0.185]], rtol=0, atol=1e-15)
    # ReLU: h = 0; pre1 = 0.25
    np.testing.assert_allclose(mo.mlp_forward(x, [W0, W1], [b0, b1], "relu"), [[0.25]], atol=1e-15)
    # sigmoid everywhere: h = 1/(1+e^{2.5}), 1/(1+e^{2}), 1/(1+e^{3})
    h = 1.0 / (1.0 + np.exp([2.5, 2.0, 3.0]))
    pre1 = h[0] - h[1] + 2 * h[2] + 0.25
    np.testing.assert_allclose(mo.mlp_forward(x, [W0, W1], [b0, b1], "sigmoid"), [[1.0 / (1.0 + np.exp(-pre1))]], rtol=1e-15)
    # linear output layer (reading N1 off): leaky hidden, identity last; a second point with positive pre-activations
    x2 = np.array([[1.0, -2.0], [3.0, 1.0]])      # pre0 of point 2 = (5.5, -2.5, 0) -> h = (5.5, -0.025, 0)
    y2 = mo.mlp_forward(x2, [W0, W1], [b0, b1], "leaky_relu", activate_last=False)
    np.testing.assert_allclose(y2, [[0.185], [5.5 + 0.025 + 0.25]], atol=1e-14)
    # last-layer activation bites when the output is negative
    yneg = mo.mlp_forward(x, [W0, -W1], [b0, -b1], "leaky_relu")
    np.testing.assert_allclose(yneg, [[-0.185 * 0.01]], atol=1e-16)


def test_identity_network_is_the_affine_closed_form_and_is_linear():
    rng = np.random.default_rng(1)
    sizes = [7, 5, 9, 4]
    Ws = [rng.normal(size=(sizes[i + 1], sizes[i])) for i in range(3)]
    bs = [rng.normal(size=sizes[i + 1]) for i in range(3)]
    x1, x2 = rng.normal(size=(6, 7)), rng.normal(size=(6, 7))
    A = Ws[2] @ Ws[1] @ Ws[0]
    c = Ws[2] @ (Ws[1] @ bs[0] + bs[1]) + bs[2]
    y1 = mo.mlp_forward(x1, Ws, bs, "identity")
    np.testing.assert_allclose(y1, x1 @ A.T + c, rtol=1e-12, atol=1e-12)
    y12 = mo.mlp_forward(0.3 * x1 - 1.7 * x2, Ws, bs, "identity")
    y2 = mo.mlp_forward(x2, Ws, bs, "identity")
    np.testing.assert_allclose(y12 - c, 0.3 * (y1 - c) - 1.7 * (y2 - c), rtol=1e-11, atol=1e-11)


@pytest.mark.parametrize("act", mo.ACTIVATIONS)
def test_hidden_permutation_invariance_and_pure_python_loop(act):
    rng = np.random.default_rng(2)
    sizes = [5, 8, 6, 3]
    Ws = [rng.normal(size=(sizes[i + 1], sizes[i])) for i in range(3)]
    bs = [rng.normal(size=sizes[i + 1]) for i in range(3)]
    x = rng.normal(size=(4, 5))
    shift, scale = rng.normal(size=5), rng.uniform(0.5, 2.0, size=5)
    y = mo.mlp_forward(x, Ws, bs, act, in_shift=shift, in_scale=scale)
    # relabel the neurons of both hidden layers
    p1, p2 = rng.permutation(8), rng.permutation(6)
    Wp = [Ws[0][p1], Ws[1][p2][:, p1], Ws[2][:, p2]]
    bp = [bs[0][p1], bs[1][p2], bs[2]]
    np.testing.assert_allclose(mo.mlp_forward(x, Wp, bp, act, in_shift=shift, in_scale=scale), y, rtol=1e-13, atol=1e-13)
    # Eq. (18)/(19) neuron by neuron in pure Python
    import math
    sig = {"identity": lambda v: v, "relu": lambda v: v if v > 0 else 0.0, "leaky_relu": lambda v: v if v > 0 else 0.01 * v,
           "sigmoid": lambda v: 1.0 / (1.0 + math.exp(-v))}[act]
    for n in range(x.shape[0]):
        h = [(x[n, i] - shift[i]) * scale[i] for i in range(5)]
        for W, b in zip(Ws, bs):
            h = [sig(sum(W[o, i] * h[i] for i in range(len(h))) + b[o]) for o in range(W.shape[0])]
        np.testing.assert_allclose(y[n], h, rtol=1e-13, atol=1e-13)


def test_single_neuron_is_eq18_and_shape_errors():
    w, b, x = np.array([[0.5, -1.5, 2.0]]), np.array([0.1]), np.array([[2.0, 1.0, 0.25]])
    pre = 1.0 - 1.5 + 0.5 + 0.1
    np.testing.assert_allclose(mo.mlp_forward(x, [w], [b], "sigmoid"), [[1 / (1 + np.exp(-pre))]], rtol=1e-15)
    with pytest.raises(ValueError):
        mo.mlp_forward(x, [w, w], [b, b])
    with pytest.raises(ValueError):
        mo.mlp_forward(x, [w], [b], "tanh")
