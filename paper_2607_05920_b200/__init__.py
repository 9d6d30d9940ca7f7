"""paper_2607_05920_b200 -- thin Python binding over the C-ABI library `libfhe_b200.so` (include/fhe.h).

Argument marshalling only: every step of the hot path (limb -> RNS decompose, negacyclic NTT, pointwise / tensor
product, inverse NTT, CRT + reduction mod Q, divide-by-P, rescale) runs in the
hand-written sm_100a kernels behind the C functions of the same names.  PyTorch is used for device memory and streams.
There is no CPU fallback: if the library is missing or fails to load, import of the binding raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_int, c_size_t, c_uint32, c_uint64, c_void_p

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfhe_b200.so")

FHE_OK, FHE_ERR_ARG, FHE_ERR_UNSUPPORTED, FHE_ERR_STATE, FHE_ERR_CUDA, FHE_ERR_NOMEM = range(6)
OP_POLYMUL, OP_HE_MULT, OP_RELINEARIZE, OP_RESCALE, OP_MULT_RELIN_RESCALE, OP_SET_EVK, OP_ROTATE, OP_MULT_PLAIN = range(8)
_STATUS_NAMES = ["FHE_OK", "FHE_ERR_ARG", "FHE_ERR_UNSUPPORTED", "FHE_ERR_STATE", "FHE_ERR_CUDA", "FHE_ERR_NOMEM"]

# every symbol include/fhe.h declares (tests/test_abi.py checks the header against this and the .so)
EXPORTS = [
    "fhe_ctx_create", "fhe_ctx_destroy", "fhe_ctx_info", "fhe_last_error", "fhe_get_modulus", "fhe_workspace_bytes",
    "fhe_set_evk", "fhe_polymul", "fhe_he_mult", "fhe_relinearize", "fhe_rescale", "fhe_mult_relin_rescale",
    "fhe_mult_relin_rescale_host", "fhe_debug_primes", "fhe_debug_decompose", "fhe_debug_ntt",
    "fhe_debug_launch_count", "fhe_debug_timing", "fhe_debug_timing_read", "fhe_debug_int_peak", "fhe_debug_crt_ambiguity",
    "fhe_add", "fhe_sub", "fhe_negate", "fhe_moddown", "fhe_mul_monomial", "fhe_set_rotation_key", "fhe_rotate", "fhe_mult_plain",
    "fhe_add_plain", "fhe_mult_scalar", "fhe_modswitch", "fhe_debug_force_pipeline",
    "fhe_static_scratch_bytes", "fhe_polymul_static_init", "fhe_polymul_static",
]


class FheInfo(ctypes.Structure):
    _fields_ = [("N", c_uint32), ("logQ", c_uint32), ("logP", c_uint32), ("t", c_uint64), ("bitsQ", c_uint32),
                ("bitsPQ", c_uint32), ("L", c_uint32), ("L_PQ", c_uint32), ("K_pm", c_uint32), ("K1", c_uint32),
                ("K2", c_uint32), ("n_sm", c_uint32)]


class FheError(RuntimeError):
    def __init__(self, status: int, msg: str):
        self.status = status
        name = _STATUS_NAMES[status] if 0 <= status < len(_STATUS_NAMES) else str(status)
        super().__init__(f"{name}: {msg}")


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree library and declare the prototypes.  Raises if it is not built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is not built: run `python -m paper_2607_05920_b200.build`")
    lib = ctypes.CDLL(LIB_PATH)
    u32p, vp = POINTER(c_uint32), c_void_p
    lib.fhe_ctx_create.argtypes = [POINTER(vp), c_uint32, c_uint32, c_uint32, c_uint64]
    lib.fhe_ctx_create.restype = c_int
    lib.fhe_ctx_destroy.argtypes = [vp]
    lib.fhe_ctx_destroy.restype = None
    lib.fhe_ctx_info.argtypes = [vp, POINTER(FheInfo)]
    lib.fhe_ctx_info.restype = c_int
    lib.fhe_last_error.argtypes = [vp]
    lib.fhe_last_error.restype = c_char_p
    lib.fhe_get_modulus.argtypes = [vp, c_int, u32p, c_uint32]
    lib.fhe_get_modulus.restype = c_int
    lib.fhe_workspace_bytes.argtypes = [vp, c_int, c_uint32]
    lib.fhe_workspace_bytes.restype = c_size_t
    lib.fhe_set_evk.argtypes = [vp, vp, vp, c_size_t, vp]
    lib.fhe_set_evk.restype = c_int
    lib.fhe_polymul.argtypes = [vp, vp, vp, vp, c_uint32, vp, c_size_t, vp]
    lib.fhe_polymul.restype = c_int
    lib.fhe_static_scratch_bytes.argtypes = []
    lib.fhe_static_scratch_bytes.restype = c_size_t
    lib.fhe_polymul_static_init.argtypes = [vp]
    lib.fhe_polymul_static_init.restype = c_int
    lib.fhe_polymul_static.argtypes = [vp, vp, vp, vp, c_uint32, vp]
    lib.fhe_polymul_static.restype = c_int
    lib.fhe_he_mult.argtypes = [vp, vp, vp, vp, c_uint32, vp, c_size_t, vp]
    lib.fhe_he_mult.restype = c_int
    lib.fhe_relinearize.argtypes = [vp, vp, vp, c_uint32, vp, c_size_t, vp]
    lib.fhe_relinearize.restype = c_int
    lib.fhe_rescale.argtypes = [vp, vp, vp, c_uint32, c_uint32, vp]
    lib.fhe_rescale.restype = c_int
    lib.fhe_mult_relin_rescale.argtypes = [vp, vp, vp, vp, c_uint32, c_uint32, vp, c_size_t, vp]
    lib.fhe_mult_relin_rescale.restype = c_int
    lib.fhe_mult_relin_rescale_host.argtypes = [vp, vp, vp, vp, c_uint32, c_uint32, vp, c_size_t, vp]
    lib.fhe_mult_relin_rescale_host.restype = c_int
    lib.fhe_debug_primes.argtypes = [vp, u32p, u32p, c_uint32]
    lib.fhe_debug_primes.restype = c_int
    lib.fhe_debug_decompose.argtypes = [vp, vp, vp, c_uint32, c_uint32, c_uint32, c_uint32, vp]
    lib.fhe_debug_decompose.restype = c_int
    lib.fhe_debug_ntt.argtypes = [vp, vp, c_uint32, c_uint32, c_int, vp]
    lib.fhe_debug_ntt.restype = c_int
    lib.fhe_debug_launch_count.argtypes = [vp]
    lib.fhe_debug_launch_count.restype = c_uint64
    lib.fhe_mult_plain.argtypes = [vp, vp, vp, vp, c_uint32, c_uint32, vp, c_size_t, vp]
    lib.fhe_mult_plain.restype = c_int
    lib.fhe_set_rotation_key.argtypes = [vp, c_uint32, c_uint32, vp, vp]
    lib.fhe_set_rotation_key.restype = c_int
    lib.fhe_rotate.argtypes = [vp, vp, vp, c_uint32, c_uint32, vp, c_size_t, vp]
    lib.fhe_rotate.restype = c_int
    lib.fhe_add.argtypes = lib.fhe_sub.argtypes = [vp, vp, vp, vp, c_uint32, vp]
    lib.fhe_negate.argtypes = [vp, vp, vp, c_uint32, vp]
    lib.fhe_moddown.argtypes = [vp, vp, vp, c_uint32, c_uint32, vp]
    lib.fhe_mul_monomial.argtypes = [vp, vp, vp, c_uint32, c_uint32, vp]
    lib.fhe_mul_monomial.restype = c_int
    lib.fhe_add.restype = lib.fhe_sub.restype = lib.fhe_negate.restype = lib.fhe_moddown.restype = c_int
    lib.fhe_add_plain.argtypes = [vp, vp, vp, vp, c_uint32, c_uint32, vp]
    lib.fhe_add_plain.restype = c_int
    lib.fhe_mult_scalar.argtypes = [vp, vp, vp, ctypes.c_int32, c_uint32, vp]
    lib.fhe_mult_scalar.restype = c_int
    lib.fhe_modswitch.argtypes = [vp, vp, vp, c_uint32, c_uint32, vp]
    lib.fhe_modswitch.restype = c_int
    lib.fhe_debug_force_pipeline.argtypes = [vp, c_int]
    lib.fhe_debug_force_pipeline.restype = c_int
    lib.fhe_debug_crt_ambiguity.argtypes = [vp, c_uint32]
    lib.fhe_debug_crt_ambiguity.restype = c_int
    lib.fhe_debug_int_peak.argtypes = [vp, c_int, POINTER(ctypes.c_double), vp]
    lib.fhe_debug_int_peak.restype = c_int
    lib.fhe_debug_timing.argtypes = [vp, c_int]
    lib.fhe_debug_timing.restype = c_int
    lib.fhe_debug_timing_read.argtypes = [vp, c_int, POINTER(ctypes.c_double), POINTER(c_uint64)]
    lib.fhe_debug_timing_read.restype = c_int
    _lib = lib
    return lib


def _torch():
    import torch
    return torch


def _dev_ptr(x, n_words: int, what: str) -> int:
    """Pointer of a contiguous CUDA tensor of 4-byte integers holding at least n_words elements."""
    torch = _torch()
    if not isinstance(x, torch.Tensor) or not x.is_cuda:
        raise TypeError(f"{what}: expected a CUDA tensor")
    if x.element_size() != 4 or x.is_floating_point():
        raise TypeError(f"{what}: expected a 4-byte integer dtype (int32/uint32 bit patterns)")
    if not x.is_contiguous():
        raise ValueError(f"{what}: tensor must be contiguous")
    if x.numel() < n_words:
        raise ValueError(f"{what}: {x.numel()} words, need {n_words}")
    return x.data_ptr()


class Context:
    """fhe_ctx handle.  Methods carry the names of the C entry points and only marshal arguments."""

    def __init__(self, N: int, logQ: int, logP: int, t: int = 0, device=None):
        torch = _torch()
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2607_05920_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self._h = c_void_p()
        with torch.cuda.device(self.device):
            st = self._lib.fhe_ctx_create(byref(self._h), N, logQ, logP, t)
        if st != FHE_OK:
            raise FheError(st, (self._lib.fhe_last_error(None) or b"").decode())
        info = FheInfo()
        self._check(self._lib.fhe_ctx_info(self._h, byref(info)))
        self.info = info
        for f, _ in FheInfo._fields_:
            setattr(self, f, int(getattr(info, f)))
        self._ws = None

    # ---- plumbing ----------------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.fhe_ctx_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != FHE_OK:
            raise FheError(st, (self._lib.fhe_last_error(self._h) or b"").decode())

    def _stream(self, stream) -> int:
        torch = _torch()
        s = torch.cuda.current_stream(self.device) if stream is None else stream
        return s.cuda_stream

    def workspace_bytes(self, op: int, batch: int) -> int:
        return int(self._lib.fhe_workspace_bytes(self._h, op, batch))

    def _workspace(self, nbytes: int):
        """Cached torch allocation used as the caller-supplied workspace."""
        torch = _torch()
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = None
            self._ws = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=self.device)
        return self._ws

    def modulus(self, which: int = 0) -> int:
        """Q (0), P (1) or P*Q (2) as a Python int."""
        n = self.L_PQ + 2
        buf = (c_uint32 * n)()
        self._check(self._lib.fhe_get_modulus(self._h, which, buf, n))
        return sum(int(buf[i]) << (32 * i) for i in range(n))

    def primes(self, count: int | None = None):
        count = max(self.K_pm, self.K1, self.K2) if count is None else count
        q = (c_uint32 * count)()
        psi = (c_uint32 * count)()
        self._check(self._lib.fhe_debug_primes(self._h, q, psi, count))
        return list(q), list(psi)

    def launch_count(self) -> int:
        return int(self._lib.fhe_debug_launch_count(self._h))

    KERNEL_CLASSES = ("decompose", "ntt_fwd", "ntt_inv", "pointwise", "crt", "rescale")

    def fhe_debug_force_pipeline(self, mode: int):
        """0 auto, 1 large-shape paths everywhere, 2 small-shape paths wherever they exist (include/fhe.h)."""
        self._check(self._lib.fhe_debug_force_pipeline(self._h, int(mode)))

    def fhe_debug_crt_ambiguity(self, bits: int):
        self._check(self._lib.fhe_debug_crt_ambiguity(self._h, bits))

    def fhe_debug_int_peak(self, mode: int, stream=None) -> float:
        """Register-only throughput per second of 0: the NTT butterfly, 1: mad.lo.u32, 2: mul.hi.u32 (whole device)."""
        v = ctypes.c_double()
        self._check(self._lib.fhe_debug_int_peak(self._h, mode, byref(v), self._stream(stream)))
        return v.value

    def fhe_debug_timing(self, enable: bool):
        self._check(self._lib.fhe_debug_timing(self._h, 1 if enable else 0))

    def fhe_debug_timing_read(self):
        """{class name: (total ms, launches)} for the launches recorded since timing was enabled."""
        out = {}
        for i, name in enumerate(self.KERNEL_CLASSES):
            ms, n = ctypes.c_double(), c_uint64()
            self._check(self._lib.fhe_debug_timing_read(self._h, i, byref(ms), byref(n)))
            out[name] = (ms.value, int(n.value))
        return out

    def _empty(self, *shape):
        torch = _torch()
        return torch.empty(shape, dtype=torch.int32, device=self.device)

    # ---- the C entry points ------------------------------------------------------------------------------------
    def fhe_set_evk(self, evk, stream=None):
        n = 2 * self.L_PQ * self.N
        self._check(self._lib.fhe_set_evk(self._h, _dev_ptr(evk, n, "evk"), None, 0, self._stream(stream)))

    def fhe_polymul(self, a, b, out=None, stream=None):
        batch = a.shape[0]
        n = batch * self.L * self.N
        out = self._empty(batch, self.L, self.N) if out is None else out
        nb = self.workspace_bytes(OP_POLYMUL, batch)
        ws = self._workspace(nb)
        self._check(self._lib.fhe_polymul(self._h, _dev_ptr(out, n, "out"), _dev_ptr(a, n, "a"), _dev_ptr(b, n, "b"),
                                          batch, ws.data_ptr(), nb, self._stream(stream)))
        return out

    def fhe_static_scratch_bytes(self) -> int:
        return int(self._lib.fhe_static_scratch_bytes())

    def fhe_polymul_static_init(self):
        self._check(self._lib.fhe_polymul_static_init(self._h))

    def fhe_polymul_static(self, a, b, out, stream=None):
        """fhe_polymul with the library's static scratch instead of a workspace: `out` is required (the caller owns every
        buffer; nothing is allocated here or in the library)."""
        batch = a.shape[0]
        n = batch * self.L * self.N
        self._check(self._lib.fhe_polymul_static(self._h, _dev_ptr(out, n, "out"), _dev_ptr(a, n, "a"), _dev_ptr(b, n, "b"),
                                                 batch, self._stream(stream)))
        return out

    def fhe_he_mult(self, ct1, ct2, out=None, stream=None):
        batch = ct1.shape[0]
        n = batch * 2 * self.L * self.N
        out = self._empty(batch, 3, self.L, self.N) if out is None else out
        nb = self.workspace_bytes(OP_HE_MULT, batch)
        ws = self._workspace(nb)
        self._check(self._lib.fhe_he_mult(self._h, _dev_ptr(out, n // 2 * 3, "out3"), _dev_ptr(ct1, n, "ct1"),
                                          _dev_ptr(ct2, n, "ct2"), batch, ws.data_ptr(), nb, self._stream(stream)))
        return out

    def fhe_relinearize(self, d3, out=None, stream=None):
        batch = d3.shape[0]
        n = batch * self.L * self.N
        out = self._empty(batch, 2, self.L, self.N) if out is None else out
        nb = self.workspace_bytes(OP_RELINEARIZE, batch)
        ws = self._workspace(nb)
        self._check(self._lib.fhe_relinearize(self._h, _dev_ptr(out, 2 * n, "out2"), _dev_ptr(d3, 3 * n, "in3"), batch,
                                              ws.data_ptr(), nb, self._stream(stream)))
        return out

    def fhe_rescale(self, ct, p_bits: int, out=None, stream=None):
        batch = ct.shape[0]
        n = batch * 2 * self.L * self.N
        out = self._empty(batch, 2, self.L, self.N) if out is None else out
        self._check(self._lib.fhe_rescale(self._h, _dev_ptr(out, n, "out2"), _dev_ptr(ct, n, "in2"), p_bits, batch,
                                          self._stream(stream)))
        return out

    def fhe_mult_relin_rescale(self, ct1, ct2, p_bits: int, out=None, stream=None):
        batch = ct1.shape[0]
        n = batch * 2 * self.L * self.N
        out = self._empty(batch, 2, self.L, self.N) if out is None else out
        nb = self.workspace_bytes(OP_MULT_RELIN_RESCALE, batch)
        ws = self._workspace(nb)
        self._check(self._lib.fhe_mult_relin_rescale(self._h, _dev_ptr(out, n, "out2"), _dev_ptr(ct1, n, "ct1"),
                                                     _dev_ptr(ct2, n, "ct2"), p_bits, batch, ws.data_ptr(), nb,
                                                     self._stream(stream)))
        return out

    def fhe_mult_relin_rescale_host(self, h_ct1, h_ct2, p_bits: int, h_out=None, stream=None):
        """HOST tensors in, HOST tensor out (pinned or pageable); copies are inside the call."""
        torch = _torch()
        batch = h_ct1.shape[0]
        n = batch * 2 * self.L * self.N
        for x, what in ((h_ct1, "h_ct1"), (h_ct2, "h_ct2")):
            if x.is_cuda or x.element_size() != 4 or not x.is_contiguous() or x.numel() < n:
                raise ValueError(f"{what}: expected a contiguous host tensor of 4-byte integers")
        h_out = torch.empty((batch, 2, self.L, self.N), dtype=torch.int32, pin_memory=True) if h_out is None else h_out
        nb = self.workspace_bytes(OP_MULT_RELIN_RESCALE, batch) + 3 * ((n * 4 + 255) // 256 * 256)
        ws = self._workspace(nb)
        self._check(self._lib.fhe_mult_relin_rescale_host(self._h, h_out.data_ptr(), h_ct1.data_ptr(), h_ct2.data_ptr(),
                                                          p_bits, batch, ws.data_ptr(), nb, self._stream(stream)))
        return h_out

    # ---- NEXT-3: ciphertext x plaintext, pairwise (group = 1) or broadcast (group = batch) ----
    def fhe_mult_plain(self, ct, pt, group: int = 1, out=None, stream=None):
        batch = ct.shape[0]
        n = batch * 2 * self.L * self.N
        npt = (batch + group - 1) // group
        out = self._empty(batch, 2, self.L, self.N) if out is None else out
        nb = self.workspace_bytes(OP_MULT_PLAIN, batch)
        ws = self._workspace(nb)
        self._check(self._lib.fhe_mult_plain(self._h, _dev_ptr(out, n, "out"), _dev_ptr(ct, n, "ct"),
                                             _dev_ptr(pt, npt * self.L * self.N, "pt"), batch, group, ws.data_ptr(), nb,
                                             self._stream(stream)))
        return out

    # ---- NEXT-2: rotation / conjugation ----
    def fhe_set_rotation_key(self, slot: int, k: int, key, stream=None):
        n = 2 * self.L_PQ * self.N
        self._check(self._lib.fhe_set_rotation_key(self._h, slot, k, _dev_ptr(key, n, "key"), self._stream(stream)))

    def fhe_rotate(self, ct, slot: int, out=None, stream=None):
        batch = ct.shape[0]
        n = batch * 2 * self.L * self.N
        out = self._empty(batch, 2, self.L, self.N) if out is None else out
        nb = self.workspace_bytes(OP_ROTATE, batch)
        ws = self._workspace(nb)
        self._check(self._lib.fhe_rotate(self._h, _dev_ptr(out, n, "out"), _dev_ptr(ct, n, "ct"), slot, batch, ws.data_ptr(), nb,
                                         self._stream(stream)))
        return out

    # ---- NEXT-1: coefficient-wise operations on [..., L, N] tensors (any leading shape) ----
    def _elem(self, fn, a, b, out, extra=()):
        npoly = a.numel() // (self.L * self.N)
        n = npoly * self.L * self.N
        out = self._torch_empty_like(a) if out is None else out
        args = [self._h, _dev_ptr(out, n, "out"), _dev_ptr(a, n, "a")]
        if b is not None:
            args.append(_dev_ptr(b, n, "b"))
        self._check(fn(*args, *extra, npoly, self._stream(None)))
        return out

    @staticmethod
    def _torch_empty_like(a):
        return _torch().empty_like(a)

    def fhe_add(self, a, b, out=None):
        return self._elem(self._lib.fhe_add, a, b, out)

    def fhe_sub(self, a, b, out=None):
        return self._elem(self._lib.fhe_sub, a, b, out)

    def fhe_negate(self, a, out=None):
        return self._elem(self._lib.fhe_negate, a, None, out)

    def fhe_mul_monomial(self, a, k: int, out=None):
        return self._elem(self._lib.fhe_mul_monomial, a, None, out, extra=(k,))

    def fhe_moddown(self, a, new_logq: int, out=None):
        return self._elem(self._lib.fhe_moddown, a, None, out, extra=(new_logq,))

    # ---- NEXT-4: BGV modulus switch ----
    def fhe_modswitch(self, a, new_logQ: int, out=None):
        return self._elem(self._lib.fhe_modswitch, a, None, out, extra=(new_logQ,))

    # ---- NEXT-3, constants ----
    def fhe_add_plain(self, ct, pt, group: int = 1, out=None):
        B = ct.shape[0]
        npt = (B + group - 1) // group if group else 0
        out = self._torch_empty_like(ct) if out is None else out
        n = B * 2 * self.L * self.N
        self._check(self._lib.fhe_add_plain(self._h, _dev_ptr(out, n, "out"), _dev_ptr(ct, n, "ct"),
                                            _dev_ptr(pt, npt * self.L * self.N, "pt"), B, group, self._stream(None)))
        return out

    def fhe_mult_scalar(self, a, k: int, out=None):
        if not -2 ** 31 <= k < 2 ** 31:
            raise ValueError("k must fit a signed 32-bit integer")
        return self._elem(self._lib.fhe_mult_scalar, a, None, out, extra=(k,))

    # ---- debug entry points --------------------------------------------------------------------------------------
    def fhe_debug_decompose(self, limbs, K: int, mask_bits: int = 0, stream=None):
        npoly, Lin = limbs.shape[0], limbs.shape[1]
        out = self._empty(npoly, K, self.N)
        self._check(self._lib.fhe_debug_decompose(self._h, out.data_ptr(), _dev_ptr(limbs, npoly * Lin * self.N, "limbs"),
                                                  npoly, Lin, K, mask_bits, self._stream(stream)))
        return out

    def fhe_debug_ntt(self, res, inverse: bool, stream=None):
        npoly, K = res.shape[0], res.shape[1]
        self._check(self._lib.fhe_debug_ntt(self._h, _dev_ptr(res, npoly * K * self.N, "res"), npoly, K,
                                            1 if inverse else 0, self._stream(stream)))
        return res
