"""Closed forms and invariants that pin the oracle's recurrence (BASELINE.json:north_star lists
the first three): linear fast weight => W += K^T diag(lr) V independent of chunking; lr = 0
leaves the output equal to the initial weights applied to Q; the chunk recurrence is
deterministic. Plus: token permutation (Eq. 8 is a sum), Eq. 10's gradient linearity, head
independence, update-before-apply, checkpoint round trip.
"""
import hashlib
import os
import subprocess
import sys

import numpy as np
import torch

from oracle.ttt_oracle import OracleTTT, rel_err, to_f64

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _rand(shape, seed, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    return torch.randn(*shape, generator=g, dtype=torch.float64) * scale


def _problem(nh=2, hd=8, H=16, M=24, seed=0):
    W1 = _rand((nh, hd, H), seed + 1, hd ** -0.5)
    W2 = _rand((nh, H, hd), seed + 2, hd ** -0.5)
    W3 = _rand((nh, hd, H), seed + 3, hd ** -0.5)
    Q = _rand((M, nh * hd), seed + 4)
    K = _rand((M, nh * hd), seed + 5)
    V = _rand((M, nh * hd), seed + 6)
    lr = torch.rand(nh, M, generator=torch.Generator().manual_seed(seed + 7), dtype=torch.float64) * 0.02
    return W1, W2, W3, Q, K, V, lr


def test_linear_fast_weight_closed_form_any_chunking():
    """north_star: a linear fast weight with dot-product loss reduces to W += lr * V^T K
    (column-vector form) == W1 += K^T diag(lr) V (row-vector form, reading P2/P3), and the
    result does not depend on how the tokens are partitioned into chunks."""
    nh, hd, M = 2, 8, 30
    W1, W2, W3, Q, K, V, lr = _problem(nh, hd, hd, M, seed=21)
    expect = to_f64(W1).copy()
    for h in range(nh):
        k, v = K[:, h * hd:(h + 1) * hd].numpy(), V[:, h * hd:(h + 1) * hd].numpy()
        expect[h] += k.T @ (lr[h].numpy()[:, None] * v)
    for cuts in ([0, 30], [0, 7, 30], [0, 1, 2, 15, 29, 30]):
        o = OracleTTT(W1, W2, W3, linear=True)
        for a, b in zip(cuts[:-1], cuts[1:]):
            o.update(K[a:b], V[a:b], lr[:, a:b])
        np.testing.assert_allclose(o.W1, expect, rtol=1e-13, atol=1e-13)
        O = o.apply(Q)
        for h in range(nh):
            np.testing.assert_allclose(O[:, h * hd:(h + 1) * hd],
                                       Q[:, h * hd:(h + 1) * hd].numpy() @ expect[h],
                                       rtol=1e-12, atol=1e-13)


def test_lr_zero_leaves_weights_bit_identical_and_output_is_initial_apply():
    W1, W2, W3, Q, K, V, lr = _problem(seed=31)
    o = OracleTTT(W1, W2, W3)
    O0 = o.apply(Q)
    O, loss = o.chunk_step(Q, K, V, torch.zeros_like(lr))
    np.testing.assert_array_equal(o.W1, to_f64(W1))
    np.testing.assert_array_equal(o.W2, to_f64(W2))
    np.testing.assert_array_equal(o.W3, to_f64(W3))
    np.testing.assert_array_equal(O, O0)
    assert (loss == 0).all()


def test_token_permutation_invariance():
    """Eq. 8 is a sum over tokens: permuting (K,V,eta) rows together leaves W' unchanged;
    permuting Q rows permutes O rows."""
    W1, W2, W3, Q, K, V, lr = _problem(M=40, seed=41)
    perm = torch.randperm(40, generator=torch.Generator().manual_seed(1))
    a = OracleTTT(W1, W2, W3); Oa, _ = a.chunk_step(Q, K, V, lr)
    b = OracleTTT(W1, W2, W3); Ob, _ = b.chunk_step(Q[perm], K[perm], V[perm], lr[:, perm])
    for x, y in zip(a.weights(), b.weights()):
        assert rel_err(x, y) <= 1e-12
    assert rel_err(Ob, Oa[perm.numpy()]) <= 1e-12


def test_gradient_linearity_across_chunks_eq10():
    """Eq. 10: gradient of the sum over chunks at the same W == sum of the
    chunks' gradients."""
    W1, W2, W3, Q, K, V, lr = _problem(M=36, seed=51)
    o = OracleTTT(W1, W2, W3)
    full = o.grad(K, V, lr)
    a = o.grad(K[:10], V[:10], lr[:, :10])
    b = o.grad(K[10:], V[10:], lr[:, 10:])
    for f, x, y in zip(full, a, b):
        np.testing.assert_allclose(f, x + y, rtol=1e-12, atol=1e-14)


def test_head_independence():
    nh, hd, H, M = 3, 8, 16, 20
    W1, W2, W3, Q, K, V, lr = _problem(nh, hd, H, M, seed=61)
    o = OracleTTT(W1, W2, W3, ns_iters=5, renorm=1)
    O, loss = o.chunk_step(Q, K, V, lr)
    for h in range(nh):
        s = slice(h * hd, (h + 1) * hd)
        oh = OracleTTT(W1[h:h + 1], W2[h:h + 1], W3[h:h + 1], ns_iters=5, renorm=1)
        Oh, lh = oh.chunk_step(Q[:, s].contiguous(), K[:, s].contiguous(), V[:, s].contiguous(),
                               lr[h:h + 1])
        np.testing.assert_array_equal(O[:, s], Oh)
        np.testing.assert_array_equal(o.W1[h], oh.W1[0])
        np.testing.assert_array_equal(o.W2[h], oh.W2[0])
        np.testing.assert_array_equal(loss[h], lh[0])
    # head 0 unchanged when other heads' data change
    K2 = K.clone(); K2[:, hd:] += 1.0
    o2 = OracleTTT(W1, W2, W3, ns_iters=5, renorm=1)
    O2, _ = o2.chunk_step(Q, K2, V, lr)
    np.testing.assert_array_equal(O2[:, :hd], O[:, :hd])
    assert rel_err(O2[:, hd:], O[:, hd:]) > 1e-6


def test_update_precedes_apply():
    """'After the update, the AMUs ... subsequently used to transform the query'."""
    W1, W2, W3, Q, K, V, lr = _problem(seed=71)
    a = OracleTTT(W1, W2, W3); Oa, _ = a.chunk_step(Q, K, V, lr)
    b = OracleTTT(W1, W2, W3); b.update(K, V, lr); Ob = b.apply(Q)
    np.testing.assert_array_equal(Oa, Ob)
    c = OracleTTT(W1, W2, W3); Oc = c.apply(Q)          # causal-LM ordering would give this
    assert rel_err(Oc, Oa) > 1e-4


def test_chunk_recurrence_and_checkpoint_roundtrip():
    W1, W2, W3, Q, K, V, lr = _problem(M=48, seed=81)
    cuts = [0, 16, 32, 48]
    a = OracleTTT(W1, W2, W3, ns_iters=5)
    outs = [a.chunk_step(Q[i:j], K[i:j], V[i:j], lr[:, i:j])[0] for i, j in zip(cuts[:-1], cuts[1:])]
    # stop after chunk 1, re-create from the weights, continue
    b = OracleTTT(W1, W2, W3, ns_iters=5)
    b.chunk_step(Q[0:16], K[0:16], V[0:16], lr[:, 0:16])
    c = OracleTTT(*b.weights(), ns_iters=5)
    O1 = c.chunk_step(Q[16:32], K[16:32], V[16:32], lr[:, 16:32])[0]
    O2 = c.chunk_step(Q[32:48], K[32:48], V[32:48], lr[:, 32:48])[0]
    np.testing.assert_array_equal(O1, outs[1])
    np.testing.assert_array_equal(O2, outs[2])
    # a different chunk order gives a different state: it IS a recurrence (reading P12)
    d = OracleTTT(W1, W2, W3, ns_iters=5)
    d.chunk_step(Q[16:32], K[16:32], V[16:32], lr[:, 16:32])
    d.chunk_step(Q[0:16], K[0:16], V[0:16], lr[:, 0:16])
    assert rel_err(d.W1, b.W1) > 1e-6


def test_empty_chunk_is_a_noop():
    W1, W2, W3, Q, K, V, lr = _problem(seed=91)
    o = OracleTTT(W1, W2, W3)
    O, loss = o.chunk_step(Q[:0], K[:0], V[:0], lr[:, :0])
    assert O.shape == (0, Q.shape[1]) and (loss == 0).all()
    np.testing.assert_array_equal(o.W1, to_f64(W1))


_DET_SNIPPET = r"""
import sys, hashlib, torch
sys.path.insert(0, %r)
from oracle.ttt_oracle import OracleTTT
g = torch.Generator().manual_seed(5)
r = lambda *s: torch.randn(*s, generator=g, dtype=torch.float64)
nh, hd, H, M = 4, 16, 32, 64
o = OracleTTT(r(nh,hd,H)/4, r(nh,H,hd)/4, r(nh,hd,H)/4, ns_iters=5, renorm=1)
O, _ = o.chunk_step(r(M,nh*hd), r(M,nh*hd), r(M,nh*hd), torch.full((nh,M), 0.01, dtype=torch.float64))
print(hashlib.sha256(O.tobytes() + o.W1.tobytes() + o.W2.tobytes() + o.W3.tobytes()).hexdigest())
"""


def test_bitwise_determinism_across_runs_and_thread_counts():
    digests = set()
    for nt in ("1", "3", "8", "8"):
        env = dict(os.environ, OMP_NUM_THREADS=nt)
        out = subprocess.run([sys.executable, "-c", _DET_SNIPPET % ROOT], env=env, check=True,
                             capture_output=True, text=True).stdout.strip()
        digests.add(out)
    assert len(digests) == 1, digests
