"""Error metric of the parity tests (reading P17 of DESIGN.md / SURVEY.md section 8(c.2)):

    err(X) = max_i |X_gpu,i - X_ora,i| / max_i |X_ora,i|     per tensor, PER HEAD, worst head reported

(each chunk's O; W1, W2, W3 after the final chunk). Pooling all heads into one max would let a head
whose weights have grown little hide behind one that has grown a lot. Not a test module."""
import numpy as np

from oracle.ttt_oracle import rel_err, to_f64


def per_head_err_tokens(X, X_ref, nh: int):
    """X, X_ref: [M, nh*hd] token tensors (O). Returns the list of per-head errors."""
    X, X_ref = to_f64(X), to_f64(X_ref)
    hd = X_ref.shape[1] // nh
    return [rel_err(X[:, h * hd:(h + 1) * hd], X_ref[:, h * hd:(h + 1) * hd]) for h in range(nh)]


def per_head_err_weights(W, W_ref):
    """W, W_ref: [nh, r, c] fast-weight tensors. Returns the list of per-head errors."""
    W, W_ref = to_f64(W), to_f64(W_ref)
    return [rel_err(W[h], W_ref[h]) for h in range(W_ref.shape[0])]


def worst_head_tokens(X, X_ref, nh: int) -> float:
    return max(per_head_err_tokens(X, X_ref, nh))


def worst_head_weights(Ws, W_refs) -> float:
    """Worst error over the three matrices and all heads."""
    return max(max(per_head_err_weights(a, b)) for a, b in zip(Ws, W_refs))


def per_head_err_vector(x, x_ref):
    """x, x_ref: [nh] (the per-head loss): relative error of each entry."""
    x, x_ref = to_f64(x), to_f64(x_ref)
    return [abs(a - b) / abs(b) if b != 0 else abs(a - b) for a, b in zip(x, x_ref)]
