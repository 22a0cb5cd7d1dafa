"""ctypes binding of include/ttt.h. Same names, argument marshalling only.

Each method of `TTT` maps 1:1 onto one C entry point (ttt_init, ttt_update, ttt_apply,
ttt_chunk_step, ttt_accumulate, ttt_commit, ttt_pending_gradient, ttt_get_weights); tensors are
torch CUDA tensors whose data pointers are passed through, and work is enqueued on torch's
current stream. Passages: update Eq. 8, loss Eq. 9, f_W
Eq. 12, apply Eq. 4, update before apply.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import torch

TTT_F32, TTT_BF16 = 0, 1
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libttt_b200.so")
_lib = None

EXPORTS = ("ttt_create", "ttt_destroy", "ttt_init", "ttt_update", "ttt_apply", "ttt_chunk_step",
           "ttt_accumulate", "ttt_commit", "ttt_pending_gradient", "ttt_get_weights",
           "ttt_launch_count", "ttt_strerror", "ttt_last_error", "ttt_version", "ttt_create_error",
           "ttt_kernel_path")


class TTTError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str = ""):
        super().__init__(f"{what}: status {status} ({detail})" if detail else f"{what}: status {status}")
        self.status = status


class _Config(ctypes.Structure):
    _fields_ = [("nh", ctypes.c_int32), ("hd", ctypes.c_int32), ("hidden", ctypes.c_int32),
                ("act_dtype", ctypes.c_int32), ("ns_iters", ctypes.c_int32),
                ("renorm", ctypes.c_int32), ("linear_fast_weight", ctypes.c_int32),
                ("device", ctypes.c_int32), ("max_tokens", ctypes.c_int64),
                ("cuda_core_fallback", ctypes.c_int32), ("reserved", ctypes.c_int32)]


def lib_path() -> str:
    return _LIB_PATH


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree C-ABI library. Raises (never falls back) if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2604_08542_b200._build` "
            "(there is no CPU or PyTorch fallback for the TTT hot path)")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, i64, f32p = ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p
    lib.ttt_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(_Config)]
    lib.ttt_destroy.argtypes = [vp]
    lib.ttt_destroy.restype = None
    lib.ttt_init.argtypes = [vp, f32p, f32p, f32p, vp]
    lib.ttt_update.argtypes = [vp, vp, vp, f32p, i64, i64, f32p, vp]
    lib.ttt_accumulate.argtypes = [vp, vp, vp, f32p, i64, i64, f32p, vp]
    lib.ttt_commit.argtypes = [vp, vp]
    lib.ttt_pending_gradient.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(i64), vp]
    lib.ttt_apply.argtypes = [vp, vp, vp, i64, i64, vp]
    lib.ttt_chunk_step.argtypes = [vp, vp, vp, vp, f32p, vp, i64, i64, f32p, vp]
    lib.ttt_get_weights.argtypes = [vp, f32p, f32p, f32p, vp]
    lib.ttt_launch_count.argtypes = [vp]
    lib.ttt_launch_count.restype = ctypes.c_int64
    lib.ttt_strerror.argtypes = [ctypes.c_int]
    lib.ttt_strerror.restype = ctypes.c_char_p
    lib.ttt_last_error.argtypes = [vp]
    lib.ttt_last_error.restype = ctypes.c_char_p
    lib.ttt_version.restype = ctypes.c_char_p
    lib.ttt_create_error.restype = ctypes.c_char_p
    lib.ttt_kernel_path.argtypes = [vp, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
    _lib = lib
    return lib


def version() -> str:
    return load_library().ttt_version().decode()


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


class TTT:
    """One context = the fast weights of `nh` heads (include/ttt.h: ttt_create / ttt_destroy)."""

    def __init__(self, nh: int, hd: int, hidden: int, act_dtype: int = TTT_BF16, ns_iters: int = 0,
                 renorm: int = 0, linear_fast_weight: int = 0, max_tokens: int = 65536,
                 device: int = 0, cuda_core_fallback: int = 0):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        self.cfg = _Config(nh, hd, hidden, act_dtype, ns_iters, renorm, linear_fast_weight, device,
                           max_tokens, cuda_core_fallback, 0)
        self.device = torch.device("cuda", device)
        self.dtype = torch.bfloat16 if act_dtype == TTT_BF16 else torch.float32
        st = self._lib.ttt_create(ctypes.byref(self._ctx), ctypes.byref(self.cfg))
        if st != 0:
            self._ctx = ctypes.c_void_p()
            raise TTTError(st, "ttt_create", self._lib.ttt_strerror(st).decode() + "; " +
                           self._lib.ttt_create_error().decode())

    # -- plumbing --------------------------------------------------------------------------
    def _check(self, st: int, what: str):
        if st != 0:
            raise TTTError(st, what, self._lib.ttt_strerror(st).decode() + "; " +
                           self._lib.ttt_last_error(self._ctx).decode())

    def _stream(self):
        return ctypes.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)

    def _tok(self, X: torch.Tensor, name: str) -> Tuple[int, int]:
        assert X.is_cuda and X.dtype == self.dtype and X.dim() == 2 and X.stride(1) == 1, name
        return X.shape[0], X.stride(0) if X.shape[0] > 1 else max(X.stride(0), X.shape[1])

    def kernel_path(self) -> Tuple[bool, bool]:
        """(update on tensor cores, apply on tensor cores) — include/ttt.h: ttt_kernel_path."""
        u, a = ctypes.c_int(), ctypes.c_int()
        self._check(self._lib.ttt_kernel_path(self._ctx, ctypes.byref(u), ctypes.byref(a)), "ttt_kernel_path")
        return bool(u.value), bool(a.value)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._lib.ttt_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C entry points ----------------------------------------------------------------
    def ttt_init(self, W1: torch.Tensor, W2: torch.Tensor, W3: torch.Tensor):
        for W in (W1, W2, W3):
            assert W.is_cuda and W.dtype == torch.float32 and W.is_contiguous()
        self._check(self._lib.ttt_init(self._ctx, _ptr(W1), _ptr(W2), _ptr(W3), self._stream()),
                    "ttt_init")

    def ttt_update(self, K, V, lr, loss: Optional[torch.Tensor] = None):
        M, ld = self._tok(K, "K")
        assert V.shape == K.shape and V.stride() == K.stride() and lr.dtype == torch.float32
        assert lr.is_contiguous() and tuple(lr.shape) == (self.cfg.nh, M)
        self._check(self._lib.ttt_update(self._ctx, _ptr(K), _ptr(V), _ptr(lr), M, ld, _ptr(loss),
                                         self._stream()), "ttt_update")

    def ttt_accumulate(self, K, V, lr, loss: Optional[torch.Tensor] = None):
        M, ld = self._tok(K, "K")
        assert V.shape == K.shape and V.stride() == K.stride() and lr.dtype == torch.float32
        assert lr.is_contiguous() and tuple(lr.shape) == (self.cfg.nh, M)
        self._check(self._lib.ttt_accumulate(self._ctx, _ptr(K), _ptr(V), _ptr(lr), M, ld,
                                             _ptr(loss), self._stream()), "ttt_accumulate")

    def ttt_commit(self):
        self._check(self._lib.ttt_commit(self._ctx, self._stream()), "ttt_commit")

    def ttt_pending_gradient(self) -> torch.Tensor:
        """Borrowed view [3, nh, H', hd] fp32 of the context-owned dense pending gradient (H' = H, or H
        rounded up to a multiple of 128 where the tensor path pads the hidden units; the pad rows are 0)."""
        p, n = ctypes.c_void_p(), ctypes.c_int64()
        self._check(self._lib.ttt_pending_gradient(self._ctx, ctypes.byref(p), ctypes.byref(n),
                                                   self._stream()), "ttt_pending_gradient")
        c = self.cfg
        shape = (3, c.nh, n.value // (3 * c.nh * c.hd), c.hd)

        class _Arr:  # __cuda_array_interface__ carrier: zero-copy view of library-owned memory
            __cuda_array_interface__ = {"shape": shape, "typestr": "<f4", "data": (p.value, False),
                                        "version": 3, "strides": None}
        return torch.as_tensor(_Arr(), device=self.device)

    def allreduce_pending_gradient(self, group=None) -> torch.Tensor:
        """Eq. 10, the method's one exchange step: sum the pending fast-weight
        gradient over the ranks of `group` IN PLACE (one NCCL all-reduce over the dense buffer that
        ttt_pending_gradient returns, over NVLink / NVSwitch), so that the ttt_commit that follows applies the
        same update on every rank. Plumbing only: torch.distributed carries the library's own buffer."""
        import torch.distributed as dist
        G = self.ttt_pending_gradient()
        dist.all_reduce(G.view(-1), op=dist.ReduceOp.SUM, group=group)
        return G

    def ttt_apply(self, Q, O: Optional[torch.Tensor] = None) -> torch.Tensor:
        M, ld = self._tok(Q, "Q")
        if O is None:
            O = torch.empty_strided(Q.shape, Q.stride(), dtype=Q.dtype, device=Q.device)
        assert O.shape == Q.shape and O.stride() == Q.stride() and O.dtype == Q.dtype
        self._check(self._lib.ttt_apply(self._ctx, _ptr(Q), _ptr(O), M, ld, self._stream()),
                    "ttt_apply")
        return O

    def ttt_chunk_step(self, Q, K, V, lr, O: Optional[torch.Tensor] = None,
                       loss: Optional[torch.Tensor] = None) -> torch.Tensor:
        M, ld = self._tok(Q, "Q")
        if O is None:
            O = torch.empty_strided(Q.shape, Q.stride(), dtype=Q.dtype, device=Q.device)
        for X in (K, V, O):
            assert X.shape == Q.shape and X.stride() == Q.stride() and X.dtype == Q.dtype
        assert lr.dtype == torch.float32 and lr.is_contiguous() and tuple(lr.shape) == (self.cfg.nh, M)
        self._check(self._lib.ttt_chunk_step(self._ctx, _ptr(Q), _ptr(K), _ptr(V), _ptr(lr), _ptr(O),
                                             M, ld, _ptr(loss), self._stream()), "ttt_chunk_step")
        return O

    def ttt_get_weights(self) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
        c = self.cfg
        W1 = torch.empty(c.nh, c.hd, c.hidden, dtype=torch.float32, device=self.device)
        W2 = torch.empty(c.nh, c.hidden, c.hd, dtype=torch.float32, device=self.device)
        W3 = torch.empty(c.nh, c.hd, c.hidden, dtype=torch.float32, device=self.device)
        self._check(self._lib.ttt_get_weights(self._ctx, _ptr(W1), _ptr(W2), _ptr(W3),
                                              self._stream()), "ttt_get_weights")
        return W1, W2, W3

    def launch_count(self) -> int:
        return int(self._lib.ttt_launch_count(self._ctx))
