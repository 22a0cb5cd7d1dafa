"""Pins of the two BASELINE-required elements the paper does not define (DESIGN.md readings
R-NS and R-RENORM): Newton-Schulz orthonormalisation and fan-in re-normalisation.

NS is pinned to its SVD closed form computed with numpy.linalg.svd (a library routine the
oracle does not call): if G = U diag(s) V^T then NS_n(G) = U diag(p^n(s/||G||_F)) V^T with
p(x) = a x + b x^3 + c x^5.
"""
import os

import numpy as np
import torch

from oracle.ttt_oracle import OracleTTT, newton_schulz, rel_err

A, B, C = 3.4445, -4.7750, 2.0315
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def p(x):
    return A * x + B * x ** 3 + C * x ** 5


def pn(x, n):
    for _ in range(n):
        x = p(x)
    return x


def _mat(r, c, seed):
    return np.random.default_rng(seed).standard_normal((r, c))


def test_ns_svd_closed_form_wide_and_tall():
    for (r, c) in ((8, 20), (20, 8), (16, 16), (64, 128), (128, 64)):
        G = _mat(r, c, r * 100 + c)
        U, s, Vt = np.linalg.svd(G, full_matrices=False)
        fro = np.linalg.norm(G) + 1e-7
        expect = (U * pn(s / fro, 5)) @ Vt
        got = newton_schulz(G, 5)
        assert rel_err(got, expect) <= 1e-10, (r, c)


def test_ns_polynomial_constants_from_golden():
    """tests/golden/ns_polynomial.txt holds values derived in SURVEY.md 8(c.3): p(1) = a+b+c and
    the slope of p^5 at 0 (= a^5)."""
    vals = {}
    for line in open(os.path.join(GOLDEN, "ns_polynomial.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split("=")
            vals[k.strip()] = float(v.split("#")[0])
    assert abs(p(1.0) - vals["p(1)"]) < 5e-4
    assert abs(A ** 5 - vals["slope_p5_at_0"]) < 0.05
    # one NS step on a matrix with a single singular value 1 (rank 1, unit Frobenius norm)
    u = np.zeros((4, 1)); u[1] = 1.0
    v = np.zeros((1, 6)); v[0, 2] = 1.0
    got = newton_schulz(u @ v, 1)
    assert abs(got[1, 2] - vals["p(1)"]) < 5e-4
    # the tiny-input slope: NS_5(eps * rank-1) ~ a^5 * eps / ... is not used (scale-invariant)


def test_ns_symmetries():
    G = _mat(12, 30, 3)
    X = newton_schulz(G, 5)
    np.testing.assert_allclose(newton_schulz(-G, 5), -X, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(newton_schulz(G.T.copy(), 5), X.T, rtol=1e-12, atol=1e-15)
    assert rel_err(newton_schulz(7.5 * G, 5), X) <= 1e-6          # scale invariance up to eps
    # orthogonal equivariance
    P, _ = np.linalg.qr(_mat(12, 12, 4))
    R, _ = np.linalg.qr(_mat(30, 30, 5))
    assert rel_err(newton_schulz(P @ G @ R, 5), P @ X @ R) <= 1e-10


def test_ns_on_orthonormal_rows_and_singular_value_band():
    Qm, _ = np.linalg.qr(_mat(40, 10, 6))
    G = Qm.T.copy()                                               # 10 orthonormal rows
    X = newton_schulz(G, 5)
    assert rel_err(X, pn(1.0 / np.sqrt(10.0), 5) * G) <= 1e-7
    G = _mat(64, 256, 7)
    s = np.linalg.svd(newton_schulz(G, 5), compute_uv=False)
    assert s.min() >= 0.68 and s.max() <= 1.21


def test_ns_batch_equals_singles_and_update_uses_it():
    Gs = np.stack([_mat(6, 10, 10 + i) for i in range(3)])
    batch = newton_schulz(Gs, 5)
    for i in range(3):
        np.testing.assert_array_equal(batch[i], newton_schulz(Gs[i], 5))
    # update with ns_iters: W' = W - NS(G) for each of the three matrices
    g = torch.Generator().manual_seed(0)
    r = lambda *s: torch.randn(*s, generator=g, dtype=torch.float64)
    nh, hd, H, M = 2, 6, 10, 15
    W1, W2, W3 = r(nh, hd, H), r(nh, H, hd), r(nh, hd, H)
    K, V = r(M, nh * hd), r(M, nh * hd)
    lr = torch.full((nh, M), 0.01, dtype=torch.float64)
    o = OracleTTT(W1, W2, W3, ns_iters=5)
    G1, G2, G3, _ = o.grad(K, V, lr)
    o.update(K, V, lr)
    np.testing.assert_array_equal(o.W1, W1.numpy() - newton_schulz(G1, 5))
    np.testing.assert_array_equal(o.W2, W2.numpy() - newton_schulz(G2, 5))
    np.testing.assert_array_equal(o.W3, W3.numpy() - newton_schulz(G3, 5))
    # lr only acts as relative token weights once NS is on (NS is scale invariant)
    o2 = OracleTTT(W1, W2, W3, ns_iters=5)
    o2.update(K, V, 4.0 * lr)
    assert rel_err(o2.W1, o.W1) <= 1e-6


def test_renorm_restores_initial_fan_in_norms():
    g = torch.Generator().manual_seed(1)
    r = lambda *s: torch.randn(*s, generator=g, dtype=torch.float64)
    nh, hd, H, M = 2, 8, 12, 20
    W1, W2, W3 = r(nh, hd, H), r(nh, H, hd), r(nh, hd, H)
    K, V = r(M, nh * hd), r(M, nh * hd)
    lr = torch.full((nh, M), 0.05, dtype=torch.float64)
    o = OracleTTT(W1, W2, W3, renorm=1)
    o.update(K, V, lr)
    # fan-in vectors: columns of W1[h] / W3[h] (length hd) and of W2[h] (length H)
    for W0, Wn, ax in ((W1.numpy(), o.W1, 1), (W3.numpy(), o.W3, 1), (W2.numpy(), o.W2, 1)):
        n0 = np.linalg.norm(W0, axis=ax)
        n1 = np.linalg.norm(Wn, axis=ax)
        np.testing.assert_allclose(n1, n0, rtol=1e-5)
    # direction equals the un-normalised update's direction
    p_ = OracleTTT(W1, W2, W3, renorm=0)
    p_.update(K, V, lr)
    cos = (p_.W1 * o.W1).sum(1) / (np.linalg.norm(p_.W1, axis=1) * np.linalg.norm(o.W1, axis=1))
    np.testing.assert_allclose(cos, 1.0, rtol=1e-12)
    # idempotent: lr = 0 update with renorm changes nothing beyond the 1e-5 epsilon
    before = o.W1.copy()
    o.update(K, V, torch.zeros_like(lr))
    assert rel_err(o.W1, before) <= 2e-5
