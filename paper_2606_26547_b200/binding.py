"""ctypes binding of libhdc.so (include/hdc.h).  Argument marshalling only: every step of the HDC
hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory
(`torch.empty`, `data_ptr()`) and streams, nothing else.  There is no CPU fallback: a missing
library or a failing call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "lib", "libhdc.so")

# enums of include/hdc.h
HDC_OK = 0
HDC_ERR_INVALID_ARG, HDC_ERR_UNSUPPORTED, HDC_ERR_ALIGNMENT = -1, -2, -3
HDC_ERR_WORKSPACE, HDC_ERR_CUDA, HDC_ERR_ARCH = -4, -5, -6
HDC_F32, HDC_BF16, HDC_I8, HDC_B1, HDC_U8, HDC_I32, HDC_F16, HDC_I64 = 0, 1, 2, 3, 4, 5, 6, 7
HDC_SIM_DOT, HDC_SIM_COS, HDC_SIM_HAMMING = 0, 1, 2
HDC_TRAIN_BUNDLE, HDC_TRAIN_PERCEPTRON, HDC_TRAIN_KMEANS = 0, 1, 2
HDC_OUT_BITS, HDC_OUT_RAW = 1, 4
HDC_OP_ENCODE_RP, HDC_OP_ENCODE_LEVELID, HDC_OP_SIMILARITY = 0, 1, 2
HDC_OP_CLASSIFY, HDC_OP_TRAIN_EPOCH, HDC_OP_INFER_RP_HOST, HDC_OP_INFER_RP = 3, 4, 5, 6
HDC_FLAG_NONE, HDC_FLAG_SIMT, HDC_FLAG_TC_1CTA, HDC_FLAG_TC_2CTA, HDC_FLAG_F32_FAST = 0, 1, 2, 4, 8
HDC_FLAG_FUSED_INFER = 16
HDC_HV_F16 = 17
HDC_HV_I16 = 18
HDC_HV_I32, HDC_HV_I64 = 19, 20
HDC_K_ENCODE_GEMM, HDC_K_SIM, HDC_K_LEVELID, HDC_K_CLASS_UPDATE = 0, 1, 2, 3
HDC_STAT_TC_LAUNCHES, HDC_STAT_SIMT_FALLBACKS, HDC_STAT_INFER_FUSED, HDC_STAT_INFER_UNFUSED = 0, 1, 2, 3

EXPORTS = ("hdc_create", "hdc_destroy", "hdc_last_error", "hdc_version", "hdc_launch_count",
           "hdc_workspace_bytes", "hdc_encode_rp", "hdc_encode_levelid", "hdc_encode_levelid_u16",
           "hdc_similarity", "hdc_similarity_adc",
           "hdc_classify", "hdc_train_epoch", "hdc_train_delta", "hdc_train_apply", "hdc_infer_rp_host",
           "hdc_kernel_timing", "hdc_kernel_time", "hdc_infer_rp", "hdc_stat", "hdc_model_bytes", "hdc_model_prepare",
           "hdc_encode_rp_m", "hdc_classify_m", "hdc_infer_rp_m", "hdc_classify_hamming_static")


class hdc_knobs_t(C.Structure):
    _fields_ = [("D_eff", C.c_int32), ("precision", C.c_int32), ("hv_bits", C.c_int32),
                ("sim", C.c_int32), ("flags", C.c_int32), ("perf_begin", C.c_int32),
                ("perf_stride", C.c_int32), ("enc_perf_begin", C.c_int32), ("enc_perf_stride", C.c_int32)]


class hdc_adc_t(C.Structure):
    _fields_ = [("res", C.c_int32), ("step", C.c_int32), ("floor", C.c_int32), ("ceil", C.c_int32)]


class hdc_model_t(C.Structure):
    _fields_ = [("magic", C.c_uint32), ("F", C.c_int32), ("D", C.c_int32), ("K", C.c_int32), ("p_dtype", C.c_int32),
                ("ldp", C.c_int64), ("ldc", C.c_int64), ("P", C.c_void_p), ("C_acc", C.c_void_p), ("blob", C.c_void_p),
                ("blob_bytes", C.c_size_t), ("knobs", hdc_knobs_t)]


class HdcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libhdc error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Loads libhdc.so (built in-tree by paper_2606_26547_b200.build); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2606_26547_b200.build` "
                           "(there is no fallback path)")
    L = C.CDLL(_LIB_PATH)
    vp, i32, i64, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t
    kp = C.POINTER(hdc_knobs_t)
    L.hdc_create.argtypes = [C.POINTER(vp), i32]
    L.hdc_create.restype = i32
    L.hdc_destroy.argtypes = [vp]
    L.hdc_destroy.restype = i32
    L.hdc_last_error.argtypes = [vp]
    L.hdc_last_error.restype = C.c_char_p
    L.hdc_version.argtypes = []
    L.hdc_version.restype = i32
    L.hdc_launch_count.argtypes = [vp]
    L.hdc_launch_count.restype = i64
    L.hdc_workspace_bytes.argtypes = [vp, i32, i64, i32, i32, i32, kp]
    L.hdc_workspace_bytes.restype = sz
    L.hdc_encode_rp.argtypes = [vp, vp, i32, i64, i32, i64, vp, i32, i32, i64, kp, i32, vp, i64, vp, i64,
                                vp, sz, vp]
    L.hdc_encode_rp.restype = i32
    L.hdc_encode_levelid.argtypes = [vp, vp, i64, i32, i64, vp, i64, vp, i32, i64, i32, kp, vp, i64, vp, sz,
                                     vp]
    L.hdc_encode_levelid.restype = i32
    L.hdc_encode_levelid_u16.argtypes = L.hdc_encode_levelid.argtypes
    L.hdc_encode_levelid_u16.restype = i32
    L.hdc_similarity.argtypes = [vp, vp, i64, i64, vp, i32, i64, i32, kp, vp, i32, i64, vp, sz, vp]
    L.hdc_similarity.restype = i32
    L.hdc_similarity_adc.argtypes = [vp, vp, i64, i64, vp, i32, i64, i32, kp, C.POINTER(hdc_adc_t), vp, i64, vp, vp,
                                     sz, vp]
    L.hdc_similarity_adc.restype = i32
    L.hdc_classify.argtypes = [vp, vp, i64, i64, vp, i32, i64, i32, kp, vp, vp, vp, vp, sz, vp]
    L.hdc_classify.restype = i32
    L.hdc_classify_hamming_static.argtypes = [vp, vp, i64, i64, vp, i32, i64, i32, kp, vp, vp, vp, vp]
    L.hdc_classify_hamming_static.restype = i32
    L.hdc_train_epoch.argtypes = [vp, i32, vp, i64, i64, vp, vp, i32, i64, i32, kp, C.c_float, i64, vp, vp,
                                  vp, sz, vp]
    L.hdc_train_epoch.restype = i32
    L.hdc_train_delta.argtypes = [vp, vp, i64, i64, vp, vp, i32, i64, i32, kp, vp, vp, vp, vp, sz, vp]
    L.hdc_train_delta.restype = i32
    L.hdc_train_apply.argtypes = [vp, vp, i32, i64, i32, kp, vp, C.c_float, vp]
    L.hdc_train_apply.restype = i32
    L.hdc_infer_rp_host.argtypes = [vp, vp, i32, i64, i32, i64, vp, i32, i32, i64, vp, i32, i64, kp, vp, vp,
                                    sz, vp]
    L.hdc_infer_rp_host.restype = i32
    L.hdc_infer_rp.argtypes = [vp, vp, i32, i64, i32, i64, vp, i32, i32, i64, vp, i32, i64, kp, vp, vp, vp, vp, i64,
                               vp, sz, vp]
    L.hdc_infer_rp.restype = i32
    L.hdc_stat.argtypes = [vp, i32]
    L.hdc_stat.restype = i64
    mp = C.POINTER(hdc_model_t)
    L.hdc_model_bytes.argtypes = [vp, i32, i32, i32, kp]
    L.hdc_model_bytes.restype = sz
    L.hdc_model_prepare.argtypes = [vp, vp, i32, i32, i32, i64, vp, i32, i64, kp, vp, sz, mp, vp]
    L.hdc_model_prepare.restype = i32
    L.hdc_encode_rp_m.argtypes = [vp, vp, i32, i64, i64, mp, vp, i64, vp, sz, vp]
    L.hdc_encode_rp_m.restype = i32
    L.hdc_classify_m.argtypes = [vp, vp, i64, i64, mp, vp, vp, vp, vp, sz, vp]
    L.hdc_classify_m.restype = i32
    L.hdc_infer_rp_m.argtypes = [vp, vp, i32, i64, i64, mp, vp, vp, vp, vp, i64, vp, sz, vp]
    L.hdc_infer_rp_m.restype = i32
    L.hdc_kernel_timing.argtypes = [vp, i32]
    L.hdc_kernel_timing.restype = i32
    L.hdc_kernel_time.argtypes = [vp, i32, C.POINTER(C.c_float), C.POINTER(i64)]
    L.hdc_kernel_time.restype = i32
    _lib = L
    return L


def knobs(D_eff: int, precision: int = HDC_F32, hv_bits: int = 32, sim: int = HDC_SIM_COS,
          flags: int = 0, perf_begin: int = 0, perf_stride: int = 1, enc_perf_begin: int = 0,
          enc_perf_stride: int = 1) -> hdc_knobs_t:
    return hdc_knobs_t(int(D_eff), int(precision), int(hv_bits), int(sim), int(flags), int(perf_begin),
                       int(perf_stride), int(enc_perf_begin), int(enc_perf_stride))


_DT = {torch.float32: HDC_F32, torch.bfloat16: HDC_BF16, torch.int8: HDC_I8, torch.uint8: HDC_U8,
       torch.int32: HDC_I32, torch.int64: HDC_I64}


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _rowmajor(t: torch.Tensor, name: str):
    if t.dim() != 2 or t.stride(1) != 1:
        raise ValueError(f"{name} must be 2-D with a contiguous last axis")
    return t.stride(0) if t.shape[0] > 1 else max(t.stride(0), t.shape[1])


class Handle:
    """hdc_handle_t with a grow-only device workspace.  Methods mirror the C entry points."""

    def __init__(self, device: int = 0):
        self._L = lib()
        self._h = C.c_void_p()
        rc = self._L.hdc_create(C.byref(self._h), int(device))
        if rc != HDC_OK:
            raise HdcError(rc, "hdc_create failed (needs a compute-capability 10.x device)")
        self.device = torch.device("cuda", device)
        self._ws = None

    def close(self):
        if self._h:
            self._L.hdc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    # -------------------------------------------------------------------------------- helpers
    def _check(self, rc: int):
        if rc != HDC_OK:
            raise HdcError(rc, self._L.hdc_last_error(self._h).decode())

    def last_error(self) -> str:
        return self._L.hdc_last_error(self._h).decode()

    def launch_count(self) -> int:
        return int(self._L.hdc_launch_count(self._h))

    def kernel_timing(self, enable: bool):
        self._check(self._L.hdc_kernel_timing(self._h, 1 if enable else 0))

    def kernel_time(self, kernel_id: int):
        """(summed ms, launches) of one kernel id since the last read; synchronises its events."""
        ms, n = C.c_float(0.0), C.c_int64(0)
        self._check(self._L.hdc_kernel_time(self._h, kernel_id, C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    def workspace_bytes(self, op: int, N: int, F_or_Q: int, D: int, K: int, kn: hdc_knobs_t) -> int:
        return int(self._L.hdc_workspace_bytes(self._h, op, N, F_or_Q, D, K, C.byref(kn)))

    def _workspace(self, nbytes: int):
        if nbytes <= 0:
            return None, 0
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        return C.c_void_p(self._ws.data_ptr()), self._ws.numel()

    def alloc_hbits(self, N: int, D_eff: int) -> torch.Tensor:
        """[N][W] int32 view of packed-hypervector rows whose stride is W rounded up to 4 words: 16-byte
        aligned rows let the encode epilogue write one 16-byte store per thread (include/hdc.h: ldh_words)."""
        W = (int(D_eff) + 31) // 32
        ld = (W + 3) // 4 * 4
        return torch.empty((int(N), ld), dtype=torch.int32, device=self.device)[:, :W]

    @staticmethod
    def _stream():
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)

    # -------------------------------------------------------------------------------- (1a)
    def hdc_encode_rp(self, X, P, kn: hdc_knobs_t, Hbits=None, want_raw: bool = False):
        N, F = X.shape
        D = P.shape[0]
        W = (kn.D_eff + 31) // 32
        if Hbits is None:
            Hbits = self.alloc_hbits(N, kn.D_eff)
        Hraw = None
        if want_raw:
            Hraw = torch.empty((N, kn.D_eff), device=self.device,
                               dtype=torch.int32 if kn.precision == HDC_I8 and kn.enc_perf_begin == 0
                               and kn.enc_perf_stride <= 1 else torch.float32)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_ENCODE_RP, N, F, D, 0, kn))
        rc = self._L.hdc_encode_rp(self._h, _ptr(X), _DT[X.dtype], N, F, _rowmajor(X, "X"), _ptr(P),
                                   _DT[P.dtype], D, _rowmajor(P, "P"), C.byref(kn),
                                   HDC_OUT_BITS | (HDC_OUT_RAW if want_raw else 0), _ptr(Hbits),
                                   _rowmajor(Hbits, "Hbits"), _ptr(Hraw),
                                   0 if Hraw is None else Hraw.stride(0), ws, wsb, self._stream())
        self._check(rc)
        return (Hbits, Hraw) if want_raw else Hbits

    # -------------------------------------------------------------------------------- (1b)
    def hdc_encode_levelid(self, levels, IDbits, LVbits, D: int, kn: hdc_knobs_t, Hbits=None):
        N, F = levels.shape
        Q = LVbits.shape[0]
        W = (kn.D_eff + 31) // 32
        if Hbits is None:
            Hbits = self.alloc_hbits(N, kn.D_eff)
        if levels.dtype not in (torch.uint8, torch.int16, torch.uint16):
            raise TypeError("levels must be uint8, or int16 / uint16 (16-bit indices)")
        fn = self._L.hdc_encode_levelid if levels.dtype == torch.uint8 else self._L.hdc_encode_levelid_u16
        rc = fn(self._h, _ptr(levels), N, F, _rowmajor(levels, "levels"),
                                        _ptr(IDbits), _rowmajor(IDbits, "IDbits"), _ptr(LVbits), Q,
                                        _rowmajor(LVbits, "LVbits"), D, C.byref(kn), _ptr(Hbits),
                                        _rowmajor(Hbits, "Hbits"), None, 0, self._stream())
        self._check(rc)
        return Hbits

    # -------------------------------------------------------------------------------- (2)
    def hdc_similarity(self, Hbits, C_acc, kn: hdc_knobs_t, s_dtype=None):
        N = Hbits.shape[0]
        K, D = C_acc.shape
        if s_dtype is None:
            s_dtype = torch.int32 if kn.sim == HDC_SIM_HAMMING else torch.float32
        S = torch.empty((N, K), dtype=s_dtype, device=self.device)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_SIMILARITY, N, 0, D, K, kn))
        rc = self._L.hdc_similarity(self._h, _ptr(Hbits), N, _rowmajor(Hbits, "Hbits"), _ptr(C_acc), K,
                                    _rowmajor(C_acc, "C_acc"), D, C.byref(kn), _ptr(S), _DT[s_dtype],
                                    S.stride(0) if N > 1 else K, ws, wsb, self._stream())
        self._check(rc)
        return S

    def hdc_similarity_adc(self, Hbits, C_acc, kn: hdc_knobs_t, res: int, step: int, floor: int, ceil: int,
                           want_scores: bool = True, want_labels: bool = True):
        """Chunked ADC-quantised dot (SpecPCM simulator, include/hdc.h (2')): returns (S int32 [N][K] or None,
        labels int32 [N] or None)."""
        N = Hbits.shape[0]
        K, D = C_acc.shape
        S = torch.empty((N, K), dtype=torch.int32, device=self.device) if want_scores else None
        labels = torch.empty(N, dtype=torch.int32, device=self.device) if want_labels else None
        adc = hdc_adc_t(int(res), int(step), int(floor), int(ceil))
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_SIMILARITY, N, 0, D, K, kn))
        rc = self._L.hdc_similarity_adc(self._h, _ptr(Hbits), N, _rowmajor(Hbits, "Hbits"), _ptr(C_acc), K,
                                        _rowmajor(C_acc, "C_acc"), D, C.byref(kn), C.byref(adc), _ptr(S), K,
                                        _ptr(labels), ws, wsb, self._stream())
        self._check(rc)
        return S, labels

    # -------------------------------------------------------------------------------- (2+3a)
    def hdc_classify(self, Hbits, C_acc, kn: hdc_knobs_t, want_scores: bool = False, labels=None):
        N = Hbits.shape[0]
        K, D = C_acc.shape
        if labels is None:
            labels = torch.empty(N, dtype=torch.int32, device=self.device)
        best = second = None
        if want_scores:
            best = torch.empty(N, dtype=torch.float32, device=self.device)
            second = torch.empty(N, dtype=torch.float32, device=self.device)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_CLASSIFY, N, 0, D, K, kn))
        rc = self._L.hdc_classify(self._h, _ptr(Hbits), N, _rowmajor(Hbits, "Hbits"), _ptr(C_acc), K,
                                  _rowmajor(C_acc, "C_acc"), D, C.byref(kn), _ptr(labels), _ptr(best),
                                  _ptr(second), ws, wsb, self._stream())
        self._check(rc)
        return (labels, best, second) if want_scores else labels

    def hdc_classify_hamming_static(self, Hbits, C_acc, kn: hdc_knobs_t, want_scores: bool = False, labels=None,
                                    best=None, second=None):
        """hdc_classify (Hamming, 1-bit classes) with the library's fixed scratch array: no workspace argument, no
        allocation inside the call (pass labels / best / second to allocate nothing on the torch side either)."""
        N = Hbits.shape[0]
        K, D = C_acc.shape
        if labels is None:
            labels = torch.empty(N, dtype=torch.int32, device=self.device)
        if want_scores and best is None:
            best = torch.empty(N, dtype=torch.float32, device=self.device)
        if want_scores and second is None:
            second = torch.empty(N, dtype=torch.float32, device=self.device)
        rc = self._L.hdc_classify_hamming_static(self._h, _ptr(Hbits), N, _rowmajor(Hbits, "Hbits"), _ptr(C_acc), K,
                                                 _rowmajor(C_acc, "C_acc"), D, C.byref(kn), _ptr(labels), _ptr(best),
                                                 _ptr(second), self._stream())
        self._check(rc)
        return (labels, best, second) if want_scores else labels

    # -------------------------------------------------------------------------------- (3b, 3c)
    def hdc_train_epoch(self, mode: int, Hbits, y, C_acc, kn: hdc_knobs_t, lr: float = 1.0,
                        batch: int = 0, pred=None, n_wrong=None):
        N = Hbits.shape[0]
        K, D = C_acc.shape
        B = N if batch in (0, None) or batch > N else batch
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_TRAIN_EPOCH, N if mode == HDC_TRAIN_KMEANS else B, 0, D, K, kn))
        rc = self._L.hdc_train_epoch(self._h, mode, _ptr(Hbits), N, _rowmajor(Hbits, "Hbits"), _ptr(y),
                                     _ptr(C_acc), K, _rowmajor(C_acc, "C_acc"), D, C.byref(kn),
                                     C.c_float(lr), int(batch or 0), _ptr(pred), _ptr(n_wrong), ws, wsb,
                                     self._stream())
        self._check(rc)
        return C_acc

    def hdc_train_delta(self, Hbits, y, C_acc, kn: hdc_knobs_t, delta=None, pred=None, n_wrong=None):
        """int32 [K][W*32] class update of these samples against the current C_acc (not applied)."""
        N = Hbits.shape[0]
        K, D = C_acc.shape
        W = (kn.D_eff + 31) // 32
        if delta is None:
            delta = torch.empty((K, W * 32), dtype=torch.int32, device=self.device)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_TRAIN_EPOCH, max(N, 1), 0, D, K, kn))
        rc = self._L.hdc_train_delta(self._h, _ptr(Hbits), N, _rowmajor(Hbits, "Hbits") if N else W, _ptr(y),
                                     _ptr(C_acc), K, _rowmajor(C_acc, "C_acc"), D, C.byref(kn), _ptr(delta),
                                     _ptr(pred), _ptr(n_wrong), ws, wsb, self._stream())
        self._check(rc)
        return delta

    def hdc_train_apply(self, C_acc, kn: hdc_knobs_t, delta, lr: float):
        K, D = C_acc.shape
        rc = self._L.hdc_train_apply(self._h, _ptr(C_acc), K, _rowmajor(C_acc, "C_acc"), D, C.byref(kn),
                                     _ptr(delta), C.c_float(lr), self._stream())
        self._check(rc)
        return C_acc

    def stat(self, stat_id: int) -> int:
        return int(self._L.hdc_stat(self._h, int(stat_id)))

    # -------------------------------------------------------------------------------- (1a)+(2)+(3a)
    def hdc_infer_rp(self, X, P, C_acc, kn: hdc_knobs_t, labels=None, want_scores: bool = False, Hbits=None):
        """encode + similarity + arg-max in one call (fused into one kernel for small K, large N)."""
        N, F = X.shape
        D = P.shape[0]
        K = C_acc.shape[0]
        if labels is None:
            labels = torch.empty(N, dtype=torch.int32, device=self.device)
        best = second = None
        if want_scores:
            best = torch.empty(N, dtype=torch.float32, device=self.device)
            second = torch.empty(N, dtype=torch.float32, device=self.device)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_INFER_RP, N, F, D, K, kn))
        rc = self._L.hdc_infer_rp(self._h, _ptr(X), _DT[X.dtype], N, F, _rowmajor(X, "X"), _ptr(P), _DT[P.dtype], D,
                                  _rowmajor(P, "P"), _ptr(C_acc), K, _rowmajor(C_acc, "C_acc"), C.byref(kn),
                                  _ptr(labels), _ptr(best), _ptr(second), _ptr(Hbits),
                                  0 if Hbits is None else _rowmajor(Hbits, "Hbits"), ws, wsb, self._stream())
        self._check(rc)
        return (labels, best, second) if want_scores else labels

    # -------------------------------------------------------------------------------- prepared model
    def hdc_model_prepare(self, P, C_acc, kn: hdc_knobs_t) -> "Model":
        """Converts the query-independent operands once (include/hdc.h "prepared model").  P or C_acc may be None."""
        D = P.shape[0] if P is not None else C_acc.shape[1]
        F = P.shape[1] if P is not None else 1
        K = C_acc.shape[0] if C_acc is not None else 1
        nbytes = int(self._L.hdc_model_bytes(self._h, F, D, K, C.byref(kn)))
        blob = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-blob.data_ptr()) % 256
        desc = hdc_model_t()
        rc = self._L.hdc_model_prepare(self._h, _ptr(P), _DT[P.dtype] if P is not None else HDC_F32, F, D,
                                       _rowmajor(P, "P") if P is not None else F, _ptr(C_acc), K,
                                       _rowmajor(C_acc, "C_acc") if C_acc is not None else D, C.byref(kn),
                                       C.c_void_p(blob.data_ptr() + off), nbytes, C.byref(desc), self._stream())
        self._check(rc)
        return Model(desc, (blob, P, C_acc), kn)

    def hdc_encode_rp_m(self, X, m: "Model", Hbits=None):
        N, F = X.shape
        kn = m.kn
        if Hbits is None:
            Hbits = self.alloc_hbits(N, kn.D_eff)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_ENCODE_RP, N, F, m.desc.D, 0, kn))
        rc = self._L.hdc_encode_rp_m(self._h, _ptr(X), _DT[X.dtype], N, _rowmajor(X, "X"), C.byref(m.desc), _ptr(Hbits),
                                     _rowmajor(Hbits, "Hbits"), ws, wsb, self._stream())
        self._check(rc)
        return Hbits

    def hdc_classify_m(self, Hbits, m: "Model", want_scores: bool = False, labels=None):
        N = Hbits.shape[0]
        if labels is None:
            labels = torch.empty(N, dtype=torch.int32, device=self.device)
        best = second = None
        if want_scores:
            best = torch.empty(N, dtype=torch.float32, device=self.device)
            second = torch.empty(N, dtype=torch.float32, device=self.device)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_CLASSIFY, N, 0, m.desc.D, m.desc.K, m.kn))
        rc = self._L.hdc_classify_m(self._h, _ptr(Hbits), N, _rowmajor(Hbits, "Hbits"), C.byref(m.desc), _ptr(labels),
                                    _ptr(best), _ptr(second), ws, wsb, self._stream())
        self._check(rc)
        return (labels, best, second) if want_scores else labels

    def hdc_infer_rp_m(self, X, m: "Model", labels=None, want_scores: bool = False, Hbits=None):
        N, F = X.shape
        if labels is None:
            labels = torch.empty(N, dtype=torch.int32, device=self.device)
        best = second = None
        if want_scores:
            best = torch.empty(N, dtype=torch.float32, device=self.device)
            second = torch.empty(N, dtype=torch.float32, device=self.device)
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_INFER_RP, N, F, m.desc.D, m.desc.K, m.kn))
        rc = self._L.hdc_infer_rp_m(self._h, _ptr(X), _DT[X.dtype], N, _rowmajor(X, "X"), C.byref(m.desc), _ptr(labels),
                                    _ptr(best), _ptr(second), _ptr(Hbits),
                                    0 if Hbits is None else _rowmajor(Hbits, "Hbits"), ws, wsb, self._stream())
        self._check(rc)
        return (labels, best, second) if want_scores else labels

    # -------------------------------------------------------------------------------- host e2e
    def hdc_infer_rp_host(self, X_host, P, C_acc, kn: hdc_knobs_t, labels_host=None):
        """X_host: CPU tensor (pinned for full speed); returns CPU int32 labels.  Synchronises."""
        N, F = X_host.shape
        D = P.shape[0]
        K = C_acc.shape[0]
        if labels_host is None:
            labels_host = torch.empty(N, dtype=torch.int32).pin_memory()
        ws, wsb = self._workspace(self.workspace_bytes(HDC_OP_INFER_RP_HOST, N, F, D, K, kn))
        rc = self._L.hdc_infer_rp_host(self._h, _ptr(X_host), _DT[X_host.dtype], N, F,
                                       _rowmajor(X_host, "X_host"), _ptr(P), _DT[P.dtype], D,
                                       _rowmajor(P, "P"), _ptr(C_acc), K, _rowmajor(C_acc, "C_acc"),
                                       C.byref(kn), _ptr(labels_host), ws, wsb, self._stream())
        self._check(rc)
        return labels_host


class Model:
    """hdc_model_t descriptor plus the tensors it points into (kept alive with it)."""

    def __init__(self, desc: hdc_model_t, keep, kn: hdc_knobs_t):
        self.desc, self._keep, self.kn = desc, keep, kn
