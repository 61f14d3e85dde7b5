"""Pins for oracle O6 (WhiFlash-Neural routing policy), CPU only.

Each test fixes the oracle to something other than itself: closed forms and identities of GELU,
special weights that reduce the MLP to a textbook expression, a pure-Python loop written from the
definition, the library routine (torch fp64) on random inputs, and the decision rule's strictness.
"""

import math

import numpy as np

from oracle import bf16, neural_route
from paper_2606_07710_b200 import synth


def _bits(x):
    return synth.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def _mlp(seed, d, B, w_std=0.05):
    g = synth.rng(seed, 7)
    m = d // 8
    h = synth.normal_bf16(g, (B, d), 1.0)
    w1 = synth.normal_bf16(g, (m, d), w_std)
    b1 = synth.normal_f32(g, (m,), 0.1)
    w2 = synth.normal_bf16(g, (m,), 0.2)
    b2 = np.float32(0.3)
    return h, w1, b1, w2, b2


def test_gelu_closed_forms():
    """GELU(0) = 0; GELU(x) - GELU(-x) = x (x Phi(x) + x Phi(-x) = x); GELU(x) -> x and GELU(-x) -> 0 for large x;
    the minimum of x Phi(x) is about -0.16997 near x = -0.7518."""
    assert neural_route.gelu(0.0) == 0.0
    x = np.linspace(-6, 6, 241)
    np.testing.assert_allclose(neural_route.gelu(x) - neural_route.gelu(-x), x, atol=1e-14)
    assert abs(float(neural_route.gelu(12.0)) - 12.0) < 1e-12 and abs(float(neural_route.gelu(-12.0))) < 1e-12
    grid = np.linspace(-2, 0, 200001)
    y = neural_route.gelu(grid)
    assert abs(y.min() - (-0.169971)) < 1e-5 and abs(grid[y.argmin()] - (-0.75179)) < 1e-3
    # x Phi(x) with Phi from the complementary error function (an independent route to the same number)
    for v in (-3.0, -0.5, 0.25, 1.0, 2.5):
        assert abs(float(neural_route.gelu(v)) - v * 0.5 * math.erfc(-v / math.sqrt(2.0))) < 1e-15


def test_zero_first_layer_reduces_to_bias_terms():
    """W1 = 0: dAL = b2 + sum_j w2_j GELU(b1_j), whatever h is."""
    h, w1, b1, w2, b2 = _mlp(1, 256, 3)
    w1[:] = 0
    want = float(b2) + sum(float(bf16.to_f64(w2[j])) * float(neural_route.gelu(float(b1[j]))) for j in range(len(b1)))
    got = neural_route.delta_al(h, w1, b1, w2, b2)
    np.testing.assert_allclose(got, np.full(3, want), atol=1e-13)


def test_one_hot_hidden_reads_a_column():
    """h = e_k: z_j = W1[j, k] + b1_j (pins the operand orientation W1 in R^{m x d}: a transposed read fails)."""
    d, m, k = 64, 8, 37
    g = synth.rng(2, 7)
    w1 = synth.normal_bf16(g, (m, d), 1.0)
    b1 = synth.normal_f32(g, (m,), 0.5)
    w2 = _bits(np.ones(m))
    h = _bits(np.eye(d)[k][None, :])
    z = bf16.to_f64(w1)[:, k] + b1.astype(np.float64)
    want = neural_route.gelu(z).sum() + 0.0
    got = neural_route.delta_al(h, w1, b1, w2, np.float32(0.0))[0]
    assert abs(got - want) < 1e-13


def test_pure_python_loop():
    """The definition written out as scalar loops with math.erf."""
    h, w1, b1, w2, b2 = _mlp(3, 64, 2)
    hf, w1f, w2f = bf16.to_f64(h), bf16.to_f64(w1), bf16.to_f64(w2)
    got = neural_route.delta_al(h, w1, b1, w2, b2)
    for b in range(2):
        acc = float(np.float32(b2))
        for j in range(w1f.shape[0]):
            z = float(b1[j])
            for k in range(w1f.shape[1]):
                z += w1f[j, k] * hf[b, k]
            acc += w2f[j] * (0.5 * z * (1.0 + math.erf(z / math.sqrt(2.0))))
        assert abs(got[b] - acc) < 1e-12


def test_matches_library_routine():
    """torch fp64: linear -> gelu(approximate='none') -> linear on the same widened inputs."""
    import torch
    h, w1, b1, w2, b2 = _mlp(4, 4096, 5, w_std=0.02)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))
    z = torch.nn.functional.linear(t(bf16.to_f64(h)), t(bf16.to_f64(w1)), t(b1.astype(np.float64)))
    want = torch.nn.functional.gelu(z, approximate="none") @ t(bf16.to_f64(w2)) + float(b2)
    got = neural_route.delta_al(h, w1, b1, w2, b2)
    np.testing.assert_allclose(got, want.numpy(), rtol=0, atol=1e-11)


def test_linear_in_second_layer_and_bias():
    """dAL is affine in (w2, b2): doubling w2 doubles dAL - b2; b2 shifts it."""
    h, w1, b1, w2, b2 = _mlp(5, 256, 4)
    base = neural_route.delta_al(h, w1, b1, w2, np.float32(0.0))
    w2x2 = _bits(2.0 * bf16.to_f64(w2))                 # exact: a power-of-two scale keeps bf16 values representable
    np.testing.assert_allclose(neural_route.delta_al(h, w1, b1, w2x2, np.float32(0.0)), 2.0 * base, atol=1e-13)
    np.testing.assert_allclose(neural_route.delta_al(h, w1, b1, w2, np.float32(1.5)), base + 1.5, atol=1e-13)


def test_route_rule_row_choice_and_ties():
    """Strict '>': dAL == tau -> diffusion; the router reads row a of each block (N4);
    an empty block yields (0, diffusion)."""
    d = 64
    h, w1, b1, w2, b2 = _mlp(6, d, 7)
    q_indptr = np.array([0, 3, 3, 7], dtype=np.int32)         # blocks of 3, 0 and 4 rows
    a = np.array([2, 0, 1], dtype=np.int32)
    per_row = neural_route.delta_al(h, w1, b1, w2, b2)
    dal, route = neural_route.neural_route(h, q_indptr, a, w1, b1, w2, b2, tau=-1e9)
    assert abs(dal[0] - per_row[2]) < 1e-13 and abs(dal[2] - per_row[4]) < 1e-13 and dal[1] == 0.0   # BLAS order differs
    assert abs(dal[0] - per_row[0]) > 1e-6 and abs(dal[2] - per_row[3]) > 1e-6                        # not another row
    assert list(route) == [1, 0, 1]
    tau = np.array([dal[0], 0.0, np.nextafter(dal[2], -np.inf)])
    _, route = neural_route.neural_route(h, q_indptr, a, w1, b1, w2, b2, tau=tau)
    assert list(route) == [0, 0, 1]                       # tie -> diffusion; just above tau -> AR


def test_parameter_count_matches_table5():
    """m = d/8 with biases: d*m + m + m + 1 parameters must round to the numbers the paper prints in Table 5
    (tests/golden/paper_table5_router_params.txt)."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_table5_router_params.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for _, d, millions in rows:
        d = int(d)
        m = d // 8
        assert round((d * m + m + m + 1) / 1e6, 2) == float(millions)
