"""Pins of the oracle's update/apply arithmetic to things OTHER than the oracle itself.

The oracle's gradient formulas (hand-derived chain rule, oracle/ttt_oracle.c:head_grad) are
checked against (i) central finite differences of the loss, (ii) torch.autograd in float64 over
a literal statement of Eq. 9 + Eq. 12 built from library routines (F.silu, matmul), (iii) brute
force one-token-at-a-time accumulation. The forward (apply) is checked against the library
SwiGLU statement. A dropped term, a wrong sign, a transposed operand or a swapped W1/W3 fails
at least one of these.
"""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle.ttt_oracle import OracleTTT, rel_err


def _rand(shape, seed, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    return (torch.randn(*shape, generator=g, dtype=torch.float64) * scale)


def _problem(nh=2, hd=4, H=6, M=5, seed=0):
    W1 = _rand((nh, hd, H), seed + 1, 0.5)
    W2 = _rand((nh, H, hd), seed + 2, 0.5)
    W3 = _rand((nh, hd, H), seed + 3, 0.5)
    Q = _rand((M, nh * hd), seed + 4)
    K = _rand((M, nh * hd), seed + 5)
    V = _rand((M, nh * hd), seed + 6)
    lr = torch.rand(nh, M, generator=torch.Generator().manual_seed(seed + 7), dtype=torch.float64)
    return W1, W2, W3, Q, K, V, lr


def f_W_library(x, W1, W2, W3):
    """Eq. 12 from library routines, row-vector convention (reading P3)."""
    return (F.silu(x @ W1) * (x @ W3)) @ W2


def loss_library(W1, W2, W3, K, V, lr, nh, hd):
    """sum over heads of sum_i eta_i * (-f_W(k_i)^T v_i)  (Eq. 8 with Eq. 9). Returns [nh]."""
    out = []
    for h in range(nh):
        k, v = K[:, h * hd:(h + 1) * hd], V[:, h * hd:(h + 1) * hd]
        f = f_W_library(k, W1[h], W2[h], W3[h])
        out.append(-(lr[h][:, None] * f * v).sum())
    return torch.stack(out)


def test_apply_matches_library_swiglu():
    W1, W2, W3, Q, K, V, lr = _problem(nh=3, hd=8, H=12, M=17)
    o = OracleTTT(W1, W2, W3)
    O = o.apply(Q)
    for h in range(3):
        ref = f_W_library(Q[:, h * 8:(h + 1) * 8], W1[h], W2[h], W3[h]).numpy()
        np.testing.assert_allclose(O[:, h * 8:(h + 1) * 8], ref, rtol=1e-12, atol=1e-13)


def test_gradient_matches_autograd_float64():
    nh, hd, H, M = 2, 4, 6, 5
    W1, W2, W3, Q, K, V, lr = _problem(nh, hd, H, M)
    o = OracleTTT(W1, W2, W3)
    G1, G2, G3, loss = o.grad(K, V, lr)
    w1, w2, w3 = (t.clone().requires_grad_(True) for t in (W1, W2, W3))
    l = loss_library(w1, w2, w3, K, V, lr, nh, hd)
    l.sum().backward()
    np.testing.assert_allclose(loss, l.detach().numpy(), rtol=1e-12)
    np.testing.assert_allclose(G1, w1.grad.numpy(), rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(G2, w2.grad.numpy(), rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(G3, w3.grad.numpy(), rtol=1e-11, atol=1e-13)


def test_gradient_matches_central_finite_differences():
    nh, hd, H, M = 1, 4, 6, 5
    W1, W2, W3, Q, K, V, lr = _problem(nh, hd, H, M, seed=11)
    o = OracleTTT(W1, W2, W3)
    G = dict(zip(("W1", "W2", "W3"), o.grad(K, V, lr)[:3]))
    Ws = {"W1": W1, "W2": W2, "W3": W3}
    h = 1e-6
    for name in ("W1", "W2", "W3"):
        fd = torch.zeros_like(Ws[name])
        flat = Ws[name].view(-1)
        for i in range(flat.numel()):
            old = flat[i].item()
            flat[i] = old + h
            lp = loss_library(Ws["W1"], Ws["W2"], Ws["W3"], K, V, lr, nh, hd).sum().item()
            flat[i] = old - h
            lm = loss_library(Ws["W1"], Ws["W2"], Ws["W3"], K, V, lr, nh, hd).sum().item()
            flat[i] = old
            fd.view(-1)[i] = (lp - lm) / (2 * h)
        assert rel_err(G[name], fd) <= 1e-7, name


def test_whole_chunk_is_one_update_unit_at_pre_update_weights():
    """Eq. 8: the gradient of the SUM at fixed W == sum of per-token gradients at that W."""
    nh, hd, H, M = 2, 4, 6, 7
    W1, W2, W3, Q, K, V, lr = _problem(nh, hd, H, M, seed=3)
    o = OracleTTT(W1, W2, W3)
    G1, G2, G3, loss = o.grad(K, V, lr)
    a1, a2, a3, al = np.zeros_like(G1), np.zeros_like(G2), np.zeros_like(G3), np.zeros_like(loss)
    for i in range(M):
        g1, g2, g3, l = o.grad(K[i:i + 1], V[i:i + 1], lr[:, i:i + 1])
        a1 += g1; a2 += g2; a3 += g3; al += l
    np.testing.assert_allclose(G1, a1, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(G2, a2, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(G3, a3, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(loss, al, rtol=1e-12)


def test_update_is_w_minus_gradient_and_sign():
    """Eq. 8: W <- W - grad. With L = -f^T v a small step must DECREASE the summed loss."""
    nh, hd, H, M = 1, 8, 16, 32
    W1, W2, W3, Q, K, V, lr = _problem(nh, hd, H, M, seed=5)
    lr = torch.full_like(lr, 1e-4)
    o = OracleTTT(W1, W2, W3)
    G1, G2, G3, l0 = o.grad(K, V, lr)
    o.update(K, V, lr)
    np.testing.assert_array_equal(o.W1, W1.numpy() - G1)
    np.testing.assert_array_equal(o.W2, W2.numpy() - G2)
    np.testing.assert_array_equal(o.W3, W3.numpy() - G3)
    l1 = o.grad(K, V, lr)[3]
    assert (l1 < l0).all()


def test_structure_of_swiglu_gradient():
    nh, hd, H, M = 2, 4, 6, 9
    W1, W2, W3, Q, K, V, lr = _problem(nh, hd, H, M, seed=7)
    G1, G2, G3, loss = OracleTTT(W1, W2, W3).grad(K, V, lr)
    # G2 does not depend on W2; G1, G3 are linear in W2
    g1, g2, g3, _ = OracleTTT(W1, 3.0 * W2, W3).grad(K, V, lr)
    np.testing.assert_allclose(g2, G2, rtol=1e-13)
    np.testing.assert_allclose(g1, 3.0 * G1, rtol=1e-13)
    np.testing.assert_allclose(g3, 3.0 * G3, rtol=1e-13)
    # everything is linear in V and in eta; power-of-two scaling is exact in floating point
    a = OracleTTT(W1, W2, W3).grad(K, 2.0 * V, lr)
    b = OracleTTT(W1, W2, W3).grad(K, V, 2.0 * lr)
    for x, y in zip(a, b):
        np.testing.assert_array_equal(x, y)
    # the loss output is the quantity being differentiated, computed the long way
    np.testing.assert_allclose(loss, loss_library(W1, W2, W3, K, V, lr, nh, hd).numpy(), rtol=1e-12)


def test_swapping_w1_w3_changes_the_result():
    """Guards against SiLU being applied to the wrong branch."""
    W1, W2, W3, Q, K, V, lr = _problem(1, 4, 6, 5, seed=9)
    a = OracleTTT(W1, W2, W3).apply(Q)
    b = OracleTTT(W3, W2, W1).apply(Q)
    assert rel_err(a, b) > 1e-2
