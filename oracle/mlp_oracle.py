"""CPU oracle of the feed-forward network that maps descriptors to the LDOS -- TEST INFRASTRUCTURE ONLY.

SURVEY.md 8(f) row f1.  What it follows (PAPER.md = /root/reference/PAPER.md):
  * a neuron is p(x) = sigma(w . x + b), Eq. (18); a network is the layer map
        x_{l+1} = sigma(W_l x_l + b_l),                                       Eq. (19)
    characterised by its number of layers, the widths w_0 .. w_L and the activation sigma;
  * the network is applied point by point: bispectrum vector B(r, j) in, LDOS vector d(r, epsilon) out;
    the output width is the number of energy levels (e.g. 241);
  * inputs "may need to be scaled (min-max scaling or standardization)": one affine map per feature.

Plain definition in fp64 with numpy: one matrix product per layer, written out layer by layer; nothing is fused,
blocked or reordered.  Readings: N1 the activation follows EVERY layer, the last one included,
as Eq. (19) is written (activate_last=False gives the variant with a linear output layer); N2 the paper does not name
sigma: leaky ReLU with slope 0.01, ReLU, the logistic sigmoid and the identity are offered; N3 the input scaling is
x_0 = (B - shift) * scale per feature.  Weights are W_l[w_{l+1}][w_l] (row = output neuron), as in Eq. (19).

Pins (tests/test_mlp_oracle.py, run with -m "not gpu"): a two-layer network worked out by hand, the affine closed
form of the identity network, invariance under a permutation of the hidden neurons, the rank-one / single-neuron
case of Eq. (18), and agreement with an independently written pure-Python triple loop.
Nothing in the product path may import this module; it shares no code with paper_2411_19617_b200/.
"""
import numpy as np

ACTIVATIONS = ("identity", "relu", "leaky_relu", "sigmoid")


def activation(name, v):
    """sigma of Eq. (18)/(19), elementwise, fp64"""
    v = np.asarray(v, dtype=np.float64)
    if name == "identity":
        return v
    if name == "relu":
        return np.where(v > 0.0, v, 0.0)
    if name == "leaky_relu":
        return np.where(v > 0.0, v, 0.01 * v)
    if name == "sigmoid":
        return 1.0 / (1.0 + np.exp(-v))
    raise ValueError(f"unknown activation {name!r}")


def mlp_forward(x, weights, biases, act="leaky_relu", activate_last=True, in_shift=None, in_scale=None):
    """Eq. (19) applied layer after layer to every row of x [npoints, w_0]; returns [npoints, w_L] in fp64."""
    h = np.asarray(x, dtype=np.float64)
    if h.ndim != 2:
        raise ValueError("x must be [npoints, w_0]")
    if in_shift is not None:
        h = h - np.asarray(in_shift, dtype=np.float64)[None, :]
    if in_scale is not None:
        h = h * np.asarray(in_scale, dtype=np.float64)[None, :]
    nl = len(weights)
    if len(biases) != nl:
        raise ValueError("weights and biases disagree on the number of layers")
    for l in range(nl):
        W = np.asarray(weights[l], dtype=np.float64)
        b = np.asarray(biases[l], dtype=np.float64)
        if W.ndim != 2 or W.shape[1] != h.shape[1] or b.shape != (W.shape[0],):
            raise ValueError(f"layer {l}: shapes do not chain")
        h = h @ W.T + b[None, :]            # W_l x_l + b_l for every point
        if l < nl - 1 or activate_last:
            h = activation(act, h)          # sigma(...)
    return h
