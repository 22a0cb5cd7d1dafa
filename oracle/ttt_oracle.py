"""ctypes front-end of the float64 CPU oracle (oracle/ttt_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs. It shares no code with the CUDA path and imports nothing
from `paper_2604_08542_b200`. All arithmetic lives in ttt_oracle.c; this file only converts the
caller's tensors (bf16 / fp32 / fp64 torch or numpy) EXACTLY to float64 and marshals pointers.

Passages: update Eq. 8, loss Eq. 9, f_W Eq. 12,
apply Eq. 4, update-before-apply, sequential chunks.
Parity against numbers printed by the paper: UNPINNED (the paper prints none for this layer);
the pins are the closed forms / invariants / finite differences in tests/test_oracle_*.py.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ttt_oracle.c")
_LIB = os.path.join(_HERE, "libttt_oracle.so")
_lib = None

_D = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, OpenMP over heads). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.ttt_oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().ttt_oracle_num_threads())


def to_f64(x) -> np.ndarray:
    """Exact conversion of a torch (bf16/fp32/fp64) or numpy array to a C-contiguous float64 array."""
    if hasattr(x, "detach"):  # torch tensor, without importing torch here
        x = x.detach().cpu().double().numpy()
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def _p(a: np.ndarray):
    return a.ctypes.data_as(_D)


class OracleTTT:
    """State (fast weights, float64) + the paper's two operations, all heads.

    W1, W3: [nh, hd, H]; W2: [nh, H, hd]. Q/K/V/O: [M, nh*hd]; lr: [nh, M].
    """

    def __init__(self, W1, W2, W3, ns_iters: int = 0, renorm: int = 0, linear: bool = False):
        self.W1, self.W2, self.W3 = to_f64(W1).copy(), to_f64(W2).copy(), to_f64(W3).copy()
        self.nh, self.hd, self.H = self.W1.shape
        assert self.W3.shape == (self.nh, self.hd, self.H)
        assert self.W2.shape == (self.nh, self.H, self.hd)
        if linear:
            assert self.H == self.hd, "linear fast weight f_W(x) = x W1 needs H == hd"
        self.ns_iters, self.renorm, self.linear = int(ns_iters), int(renorm), int(bool(linear))
        self.n0_1 = np.zeros((self.nh, self.H))
        self.n0_2 = np.zeros((self.nh, self.hd))
        self.n0_3 = np.zeros((self.nh, self.H))
        _load().ttt_oracle_col_norms(_p(self.W1), _p(self.W2), _p(self.W3), self.nh, self.hd,
                                     self.H, _p(self.n0_1), _p(self.n0_2), _p(self.n0_3))

    # -- helpers ---------------------------------------------------------------------------
    def _tok(self, X) -> np.ndarray:
        X = to_f64(X)
        assert X.ndim == 2 and X.shape[1] == self.nh * self.hd, X.shape
        return X

    def _lr(self, lr, M) -> np.ndarray:
        lr = to_f64(lr)
        assert lr.shape == (self.nh, M), (lr.shape, (self.nh, M))
        return lr

    # -- the paper's operations ------------------------------------------------------------
    def grad(self, K, V, lr) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]:
        """(G1, G2, G3, loss[nh]) of Eq. 8's summed, lr-weighted loss at the current W."""
        K, V = self._tok(K), self._tok(V)
        M = K.shape[0]
        lr = self._lr(lr, M)
        G1, G2, G3 = np.zeros_like(self.W1), np.zeros_like(self.W2), np.zeros_like(self.W3)
        loss = np.zeros(self.nh)
        _load().ttt_oracle_grad(_p(K), _p(V), _p(lr), ctypes.c_long(M),
                                ctypes.c_long(K.shape[1]), self.nh, self.hd, self.H, self.linear,
                                _p(self.W1), _p(self.W2), _p(self.W3),
                                _p(G1), _p(G2), _p(G3), _p(loss))
        return G1, G2, G3, loss

    def update(self, K, V, lr) -> np.ndarray:
        """Eq. 8 (+ optional Newton-Schulz / re-normalisation). Returns loss[nh]."""
        K, V = self._tok(K), self._tok(V)
        M = K.shape[0]
        lr = self._lr(lr, M)
        loss = np.zeros(self.nh)
        if M == 0:
            return loss
        _load().ttt_oracle_update(_p(K), _p(V), _p(lr), ctypes.c_long(M),
                                  ctypes.c_long(K.shape[1]), self.nh, self.hd, self.H,
                                  self.linear, self.ns_iters, self.renorm,
                                  _p(self.W1), _p(self.W2), _p(self.W3),
                                  _p(self.n0_1), _p(self.n0_2), _p(self.n0_3), _p(loss))
        return loss

    def apply(self, Q) -> np.ndarray:
        """Eq. 4: O = f_W(Q) with the current weights. Returns float64 [M, nh*hd]."""
        Q = self._tok(Q)
        M = Q.shape[0]
        O = np.zeros((M, self.nh * self.hd))
        if M == 0:
            return O
        _load().ttt_oracle_apply(_p(Q), ctypes.c_long(M), ctypes.c_long(Q.shape[1]), self.nh,
                                 self.hd, self.H, self.linear,
                                 _p(self.W1), _p(self.W2), _p(self.W3), _p(O),
                                 ctypes.c_long(O.shape[1]))
        return O

    def chunk_step(self, Q, K, V, lr) -> Tuple[np.ndarray, np.ndarray]:
        """update then apply. Returns (O, loss)."""
        loss = self.update(K, V, lr)
        return self.apply(Q), loss

    def weights(self) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
        return self.W1.copy(), self.W2.copy(), self.W3.copy()


def newton_schulz(G, iters: int = 5) -> np.ndarray:
    """NS on one matrix [r, c] or a batch [n, r, c] (reading R-NS)."""
    G = to_f64(G).copy()
    shp = G.shape
    G3 = G.reshape((-1,) + shp[-2:])
    _load().ttt_oracle_newton_schulz(_p(G3), G3.shape[0], G3.shape[1], G3.shape[2], int(iters))
    return G3.reshape(shp)


def rel_err(x, ref) -> float:
    """SURVEY.md P17 / DESIGN.md: max_i |x_i - ref_i| / max_i |ref_i| (per tensor)."""
    x, ref = to_f64(x), to_f64(ref)
    den = float(np.max(np.abs(ref)))
    num = float(np.max(np.abs(x - ref))) if x.size else 0.0
    if not np.isfinite(num):
        return float("inf")
    return num / den if den > 0 else num
