"""Seeded synthetic inputs for the TTT global-context-memory hot path.

This module is shared by the oracle-side tests and the CUDA-side tests/bench. It holds
NONE of the method's arithmetic (no SwiGLU, no gradient, no Newton-Schulz, no update):
it only draws the random tensors both sides consume, with the shapes and value
distributions that BASELINE.json:configs prescribes (recipe: DESIGN.md "Input recipe",
SURVEY.md section 8(d)). It imports neither `oracle/` nor the CUDA package.

Streams: base seed s -> independent torch CPU generators seeded s*16 + {0:W1, 1:W2, 2:W3,
3:Q, 4:K, 5:V}. Fast weights: every entry N(0, 1/hd) in fp32. Tokens: N(0,1) marginals,
AR(1) over frames with coefficient rho per (position, channel), state carried across
chunk boundaries; optional per-head L2 normalisation of K rows done in fp32 BEFORE the
rounding to the activation dtype. lr: the config's constant, as a [nh, M] fp32 array.

Secondary "structured" workload (parity only): Q, K, V are three fixed seeded
projections X P_q, X P_k, X P_v (P ~ N(0, 1/d), streams 6, 7, 8) of COMMON tokens X (the Q stream's
AR(1) process) - the relation the paper's module has between its q, k, v;
marginals stay N(0,1).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Iterator, Optional, Tuple

import torch

_STREAM = {"W1": 0, "W2": 1, "W3": 2, "Q": 3, "K": 4, "V": 5, "PQ": 6, "PK": 7, "PV": 8}


@dataclasses.dataclass(frozen=True)
class TTTWorkload:
    """One row of BASELINE.json:configs (or a cut-down test variant of it)."""

    name: str
    nh: int                   # heads
    hd: int                   # head dim
    hidden: int               # H = hd * k
    tokens_per_frame: int
    frames_per_chunk: int
    n_frames: int             # total frames streamed (last chunk may be short)
    act_dtype: str            # "f32" | "bf16"
    lr: float
    rho: float = 0.0          # AR(1) coefficient over frames
    l2_k: bool = False        # L2-normalise K rows per head slice
    ns_iters: int = 0         # Newton-Schulz iterations (0 = plain Eq. 8)
    renorm: int = 0           # restore per-unit fan-in norms after the update
    seed: int = 0
    structured: bool = False  # Q, K, V = projections of common tokens (secondary workload)

    @property
    def d(self) -> int:
        return self.nh * self.hd

    @property
    def chunk_tokens(self) -> int:
        return self.tokens_per_frame * self.frames_per_chunk

    @property
    def n_chunks(self) -> int:
        return -(-self.n_frames // self.frames_per_chunk)

    def chunk_frames(self, c: int) -> int:
        lo = c * self.frames_per_chunk
        return min(self.frames_per_chunk, self.n_frames - lo)

    @property
    def torch_dtype(self) -> torch.dtype:
        return {"f32": torch.float32, "bf16": torch.bfloat16}[self.act_dtype]

    def state_size(self) -> int:
        """Eq. 13: nh * hd * hd * k — counts ONE matrix."""
        return self.nh * self.hd * self.hidden


# BASELINE.json:configs[0..4] (1-based "cfg1".."cfg5" as in SURVEY.md section 8(d)).
CONFIGS = {
    "cfg1": TTTWorkload("cfg1", nh=1, hd=64, hidden=128, tokens_per_frame=256,
                        frames_per_chunk=1, n_frames=4, act_dtype="f32", lr=0.01),
    "cfg2": TTTWorkload("cfg2", nh=16, hd=64, hidden=128, tokens_per_frame=1374,
                        frames_per_chunk=8, n_frames=8, act_dtype="bf16", lr=0.01, l2_k=True),
    "cfg3": TTTWorkload("cfg3", nh=16, hd=64, hidden=256, tokens_per_frame=1374,
                        frames_per_chunk=8, n_frames=64, act_dtype="bf16", lr=0.01, rho=0.9,
                        ns_iters=5),
    "cfg4": TTTWorkload("cfg4", nh=16, hd=64, hidden=256, tokens_per_frame=1374,
                        frames_per_chunk=32, n_frames=2000, act_dtype="bf16", lr=0.005,
                        rho=0.95, l2_k=True, renorm=1),
    "cfg5": TTTWorkload("cfg5", nh=8, hd=128, hidden=512, tokens_per_frame=2741,
                        frames_per_chunk=16, n_frames=512, act_dtype="bf16", lr=0.01,
                        ns_iters=5),
    # The shape the paper itself ships (not a BASELINE.json config): ONE head of
    # hd = d = 1024, hidden = k hd with k = 4 ("state size 4M", Table 3),
    # chunks of 60 frames x 1374 tokens, plain Eq. 8 update. lr and L2-normalised K are
    # this build's choice (the paper gives neither; the literal recurrence needs small steps to stay finite).
    "paper_k4": TTTWorkload("paper_k4", nh=1, hd=1024, hidden=4096, tokens_per_frame=1374,
                            frames_per_chunk=60, n_frames=60, act_dtype="bf16", lr=1e-4, l2_k=True),
    "paper_k1": TTTWorkload("paper_k1", nh=1, hd=1024, hidden=1024, tokens_per_frame=1374,
                            frames_per_chunk=60, n_frames=60, act_dtype="bf16", lr=1e-4, l2_k=True),
}


def _gen(seed: int, stream: str) -> torch.Generator:
    g = torch.Generator(device="cpu")
    g.manual_seed(seed * 16 + _STREAM[stream])
    return g


def fast_weights(w: TTTWorkload) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """W1,W3 [nh,hd,H], W2 [nh,H,hd], fp32, every entry N(0, 1/hd) (configs[0]: "init N(0,1/d)")."""
    std = 1.0 / math.sqrt(w.hd)
    W1 = torch.randn(w.nh, w.hd, w.hidden, generator=_gen(w.seed, "W1"), dtype=torch.float32) * std
    W2 = torch.randn(w.nh, w.hidden, w.hd, generator=_gen(w.seed, "W2"), dtype=torch.float32) * std
    W3 = torch.randn(w.nh, w.hd, w.hidden, generator=_gen(w.seed, "W3"), dtype=torch.float32) * std
    return W1, W2, W3


class TokenStream:
    """Streams (Q, K, V, lr) chunk by chunk; AR(1) state is carried across chunks."""

    def __init__(self, w: TTTWorkload):
        self.w = w
        self._g = {s: _gen(w.seed, s) for s in ("Q", "K", "V")}
        self._prev = {s: None for s in ("Q", "K", "V")}
        self._chunk = 0
        self._proj = None
        if w.structured:
            std = 1.0 / math.sqrt(w.d)
            self._proj = {s: torch.randn(w.d, w.d, generator=_gen(w.seed, "P" + s), dtype=torch.float32) * std
                          for s in ("Q", "K", "V")}

    def _frames(self, s: str, nf: int) -> torch.Tensor:
        w = self.w
        E = torch.randn(nf, w.tokens_per_frame, w.d, generator=self._g[s], dtype=torch.float32)
        if w.rho == 0.0:
            return E
        a, b = w.rho, math.sqrt(1.0 - w.rho * w.rho)
        X = torch.empty_like(E)
        prev = self._prev[s]
        for f in range(nf):
            prev = E[f] if prev is None else a * prev + b * E[f]
            X[f] = prev
        self._prev[s] = prev.clone()
        return X

    def next_chunk(self) -> Optional[Tuple[torch.Tensor, torch.Tensor, torch.Tensor, torch.Tensor]]:
        w = self.w
        if self._chunk >= w.n_chunks:
            return None
        nf = w.chunk_frames(self._chunk)
        self._chunk += 1
        M = nf * w.tokens_per_frame
        out = []
        common = self._frames("Q", nf).reshape(M, w.d) if w.structured else None
        for s in ("Q", "K", "V"):
            X = (common @ self._proj[s] if w.structured else self._frames(s, nf)).reshape(M, w.nh, w.hd)
            if s == "K" and w.l2_k:
                X = X / X.norm(dim=-1, keepdim=True)
            out.append(X.reshape(M, w.d).to(w.torch_dtype).contiguous())
        lr = torch.full((w.nh, M), w.lr, dtype=torch.float32)
        return out[0], out[1], out[2], lr

    def __iter__(self) -> Iterator[Tuple[torch.Tensor, torch.Tensor, torch.Tensor, torch.Tensor]]:
        while True:
            c = self.next_chunk()
            if c is None:
                return
            yield c


def scaled(w: TTTWorkload, **kw) -> TTTWorkload:
    """A cut-down variant (fewer heads/frames/tokens) of a config for parity tests."""
    return dataclasses.replace(w, **kw)


def shard_heads(nh: int, world_size: int, rank: int) -> Tuple[int, int]:
    """Head range [lo, hi) owned by `rank` when heads are sharded with no collective
    (heads are independent units: Eq. 13)."""
    base, rem = divmod(nh, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_chunks(n_items: int, world_size: int, rank: int) -> Tuple[int, int]:
    """Contiguous range of independent sequences owned by `rank` (weak scaling)."""
    return shard_heads(n_items, world_size, rank)
