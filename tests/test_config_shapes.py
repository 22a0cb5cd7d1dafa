"""Shape facts the paper states (Eq. 13, Table 3) and the workload table of BASELINE.json."""
import os

import torch

import ttt_inputs as ti

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_state_size_formula_matches_paper_table3():
    for line in open(os.path.join(GOLDEN, "state_size.txt")):
        if line.startswith("#") or not line.strip():
            continue
        nh, hd, k, size, label = line.split()
        w = ti.TTTWorkload("paper", nh=int(nh), hd=int(hd), hidden=int(hd) * int(k),
                           tokens_per_frame=1374, frames_per_chunk=60, n_frames=60,
                           act_dtype="bf16", lr=0.01)
        assert w.state_size() == int(size)
        assert round(w.state_size() / 2 ** 20) == int(label[:-1])


def test_baseline_config_table():
    c = ti.CONFIGS
    assert c["cfg1"].chunk_tokens == 256 and c["cfg1"].n_chunks == 4
    assert c["cfg2"].chunk_tokens == 8 * 1374 == 10992 and c["cfg2"].n_chunks == 1
    assert 37 * 37 + 1 + 4 == 1374   # configs[4]'s 2741 is taken as given (37*74+5 is 2743)
    assert c["cfg3"].n_chunks == 8 and c["cfg3"].d == 1024
    assert c["cfg4"].n_chunks == 63 and c["cfg4"].chunk_frames(62) == 16
    assert c["cfg5"].chunk_tokens == 16 * 2741 and c["cfg5"].n_chunks == 32 and c["cfg5"].d == 1024


def test_streams_are_seeded_and_shaped():
    w = ti.scaled(ti.CONFIGS["cfg3"], nh=2, tokens_per_frame=10, frames_per_chunk=3, n_frames=7)
    a = list(ti.TokenStream(w))
    b = list(ti.TokenStream(w))
    assert [x[0].shape[0] for x in a] == [30, 30, 10]
    for ca, cb in zip(a, b):
        for x, y in zip(ca, cb):
            assert (x == y).all()
    # AR(1) over frames: consecutive frames correlate ~rho, also across the chunk boundary
    w = ti.scaled(ti.CONFIGS["cfg3"], nh=2, tokens_per_frame=400, frames_per_chunk=2, n_frames=4)
    ch = list(ti.TokenStream(w))
    q0 = ch[0][0].float().reshape(2, 400, -1)
    q1 = ch[1][0].float().reshape(2, 400, -1)
    corr = lambda x, y: float((x * y).mean() / (x.std() * y.std()))
    assert abs(corr(q0[0], q0[1]) - 0.9) < 0.02
    assert abs(corr(q0[1], q1[0]) - 0.9) < 0.02
    assert abs(float(q1.std()) - 1.0) < 0.02
    # L2-normalised K (cfg2): unit norm per head slice up to bf16 rounding
    w = ti.scaled(ti.CONFIGS["cfg2"], tokens_per_frame=16, frames_per_chunk=2, n_frames=2)
    q, k, v, lr = ti.TokenStream(w).next_chunk()
    n = k.float().reshape(32, w.nh, w.hd).norm(dim=-1)
    assert float((n - 1).abs().max()) < 2 ** -7
    assert lr.shape == (w.nh, 32) and abs(float(lr[0, 0]) - w.lr) < 1e-9


def test_structured_stream_is_three_projections_of_common_tokens():
    """Secondary workload: Q, K, V = X P_q, X P_k, X P_v of common AR(1)
    tokens X: unit marginals, the same frame-to-frame correlation, and K a linear map of Q's
    source (rank check: [Q K V] of d+8 tokens has rank d, iid streams would have rank d+8)."""
    w = ti.scaled(ti.CONFIGS["cfg3"], nh=2, hd=16, hidden=32, act_dtype="f32", tokens_per_frame=40,
                  frames_per_chunk=1, n_frames=3, structured=True)
    ch = list(ti.TokenStream(w))
    q, k, v, lr = ch[0]
    assert q.shape == (40, 32) and lr.shape == (2, 40)
    stacked = torch.cat([q, k, v], dim=1).double()              # [40, 96] = X [40, 32] @ [P_q P_k P_v]
    assert torch.linalg.matrix_rank(stacked, tol=1e-4) == 32
    iid = ti.scaled(w, structured=False)
    q2, k2, v2, _ = ti.TokenStream(iid).next_chunk()
    assert torch.linalg.matrix_rank(torch.cat([q2, k2, v2], dim=1).double(), tol=1e-4) == 40
    big = ti.scaled(w, tokens_per_frame=600, frames_per_chunk=2, n_frames=2)
    qq, kk, vv, _ = ti.TokenStream(big).next_chunk()
    for x in (qq, kk, vv):
        assert abs(float(x.std()) - 1.0) < 0.05
        f = x.reshape(2, 600, -1)
        assert abs(float((f[0] * f[1]).mean() / (f[0].std() * f[1].std())) - 0.9) < 0.05


def test_sharding_helpers_cover_everything_once():
    for n, ws in ((16, 2), (16, 3), (8, 8), (5, 2)):
        got = []
        for r in range(ws):
            lo, hi = ti.shard_heads(n, ws, r)
            got += list(range(lo, hi))
        assert got == list(range(n))
