"""Thin Python binding over libkairos.so (include/kairos.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch is used for device memory and streams.
Importing this module loads the shared library and raises if it is missing: there is no CPU fallback and
nothing here ever touches oracle/.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkairos.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is not built: run `python -m paper_2607_02043_b200.build` (nvcc, sm_100a). "
        "There is no CPU fallback.")

_lib = ctypes.CDLL(LIB_PATH)
_c = ctypes
_vp = _c.c_void_p
_i32 = _c.c_int32


class KairosConfig(_c.Structure):
    _fields_ = [("num_heads", _i32), ("latent_dim", _i32), ("rope_dim", _i32), ("page_size", _i32),
                ("softmax_scale", _c.c_float), ("pool", _vp), ("num_pages", _i32), ("workspace", _vp),
                ("workspace_bytes", _c.c_size_t), ("device", _i32)]


_lib.kairos_workspace_bytes.argtypes = [_i32, _i32]
_lib.kairos_workspace_bytes.restype = _c.c_size_t
_lib.kairos_create.argtypes = [_c.POINTER(KairosConfig), _c.POINTER(_vp)]
_lib.kairos_create.restype = _c.c_int
_lib.kairos_destroy.argtypes = [_vp]
_lib.kairos_destroy.restype = _c.c_int
_lib.kairos_append_latent.argtypes = [_vp, _vp, _vp, _i32, _vp, _i32, _i32, _vp]
_lib.kairos_append_latent.restype = _c.c_int
_lib.kairos_append_decode_tokens.argtypes = [_vp, _vp, _vp, _i32, _vp, _i32, _vp, _vp]
_lib.kairos_append_decode_tokens.restype = _c.c_int
_lib.kairos_gather_latent.argtypes = [_vp, _vp, _i32, _i32, _vp, _vp]
_lib.kairos_gather_latent.restype = _c.c_int
_lib.kairos_mixed_step.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp, _i32, _i32, _vp, _vp, _i32, _vp, _vp, _vp, _vp, _vp]
_lib.kairos_mixed_step.restype = _c.c_int
_lib.kairos_mixed_step_host.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp, _i32, _i32, _vp, _vp, _vp, _vp, _i32, _vp, _vp,
                                        _vp, _vp, _vp, _vp, _vp]
_lib.kairos_mixed_step_host.restype = _c.c_int
_lib.kairos_step_latency_table.argtypes = [_vp, _vp, _i32, _vp, _i32, _vp, _i32, _i32, _i32, _i32, _i32, _vp, _vp, _vp]
_lib.kairos_step_latency_table.restype = _c.c_int
_lib.kairos_plan_dump.argtypes = [_vp, _i32, _i32, _i32, _i32, _i32, _vp, _i32, _vp, _vp, _vp]
_lib.kairos_plan_dump.restype = _c.c_int
_lib.kairos_last_plan_info.argtypes = [_vp, _vp, _i32]
_lib.kairos_last_plan_info.restype = _c.c_int
_lib.kairos_profile_enable.argtypes = [_vp, _i32]
_lib.kairos_profile_enable.restype = _c.c_int
_lib.kairos_profile_read.argtypes = [_vp, _vp, _vp]
_lib.kairos_profile_read.restype = _c.c_int


class StepModel(_c.Structure):
    """kairos_step_model (Eq. 4): T0 = a0 + a1*B + a2*Kd; dT_pf = b0 + b1*C + b2*C*(P + (C+1)/2) + b3*Kd for C > 0."""
    _fields_ = [("a", _c.c_double * 3), ("b", _c.c_double * 4)]


class PrefillModel(_c.Structure):
    """kairos_prefill_model: T = p0 + p1*tokens + p2*cached + p3*tokens*cached."""
    _fields_ = [("p", _c.c_double * 4)]


class DecideInput(_c.Structure):
    _fields_ = [("prompt_len", _i32), ("queue_lens", _vp), ("n_queue", _i32), ("chi_p", _i32), ("node_B", _vp),
                ("node_K", _vp), ("n_nodes", _i32), ("candidates", _vp), ("n_candidates", _i32), ("tbt_slo", _c.c_double),
                ("beta", _c.c_double), ("alpha", _c.c_double), ("ttft_slo", _c.c_double)]


class DecideOutput(_c.Structure):
    _fields_ = [("decision", _i32), ("node", _i32), ("n_steps", _i32), ("ttft_pf", _c.c_double), ("ttft_dec", _c.c_double)]


class SimRequest(_c.Structure):
    _fields_ = [("arrival", _c.c_double), ("prompt_len", _i32), ("output_len", _i32)]


class SimConfig(_c.Structure):
    _fields_ = [("n_prefill", _i32), ("n_decode", _i32), ("chi_p", _i32), ("policy", _i32), ("param", _i32),
                ("static_chi", _i32), ("candidates", _vp), ("n_candidates", _i32), ("tbt_slo", _c.c_double),
                ("beta", _c.c_double), ("alpha", _c.c_double), ("ttft_slo", _c.c_double), ("transfer_per_token", _c.c_double)]


class SimResult(_c.Structure):
    _fields_ = [("n_requests", _i32), ("n_deflected", _i32), ("p95_ttft", _c.c_double), ("mean_ttft", _c.c_double),
                ("decode_steps", _c.c_int64), ("tbt_violations", _c.c_int64), ("slo_attainment", _c.c_double),
                ("makespan", _c.c_double)]


_lib.kairos_simulate.argtypes = [_c.POINTER(StepModel), _c.POINTER(PrefillModel), _c.POINTER(SimConfig), _vp, _i32, _vp,
                                 _c.POINTER(SimResult)]
_lib.kairos_simulate.restype = _c.c_int
_lib.kairos_fit_latency_model.argtypes = [_vp, _vp, _vp, _vp, _vp, _i32, _c.POINTER(StepModel), _vp]
_lib.kairos_fit_latency_model.restype = _c.c_int
_lib.kairos_predict_step.argtypes = [_c.POINTER(StepModel), _c.c_int64, _c.c_int64, _c.c_int64, _c.c_int64]
_lib.kairos_predict_step.restype = _c.c_double
_lib.kairos_decide.argtypes = [_c.POINTER(StepModel), _c.POINTER(PrefillModel), _c.POINTER(DecideInput), _vp, _i32,
                               _c.POINTER(DecideOutput)]
_lib.kairos_decide.restype = _c.c_int
_lib.kairos_run_schedule.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp, _vp, _vp, _i32, _vp, _i32, _vp, _vp, _vp, _vp, _i32, _i32,
                                     _vp, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.kairos_run_schedule.restype = _c.c_int
_lib.kairos_absorb_q.argtypes = [_vp, _vp, _vp, _vp, _i32, _vp, _vp]
_lib.kairos_absorb_q.restype = _c.c_int
_lib.kairos_project_out.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp]
_lib.kairos_project_out.restype = _c.c_int
_lib.kairos_tune_step.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp, _i32, _i32, _vp, _vp, _i32, _vp, _vp, _i32, _vp, _vp, _vp, _vp]
_lib.kairos_tune_step.restype = _c.c_int
_lib.kairos_fp8_attach.argtypes = [_vp, _vp, _i32]
_lib.kairos_fp8_attach.restype = _c.c_int
_lib.kairos_fp8_append.argtypes = [_vp, _vp, _vp, _i32, _vp, _i32, _i32, _vp]
_lib.kairos_fp8_append.restype = _c.c_int
_lib.kairos_fp8_append_decode_tokens.argtypes = [_vp, _vp, _vp, _i32, _vp, _i32, _vp, _vp]
_lib.kairos_fp8_append_decode_tokens.restype = _c.c_int
_lib.kairos_fp8_mixed_step.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp, _i32, _i32, _vp, _vp, _i32, _vp, _vp, _vp, _vp, _vp]
_lib.kairos_fp8_mixed_step.restype = _c.c_int
_lib.kairos_fp8_decode.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp, _vp, _vp, _vp]
_lib.kairos_fp8_decode.restype = _c.c_int
_lib.kairos_decode_static.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp, _vp, _vp, _vp]
_lib.kairos_decode_static.restype = _c.c_int
_lib.kairos_debug_set.argtypes = [_vp, _c.c_char_p, _i32]
_lib.kairos_debug_set.restype = _c.c_int
_lib.kairos_last_error.argtypes = []
_lib.kairos_last_error.restype = _c.c_char_p
_lib.kairos_version.argtypes = []
_lib.kairos_version.restype = _c.c_char_p

EXPORTS = ["kairos_workspace_bytes", "kairos_create", "kairos_destroy", "kairos_append_latent",
           "kairos_append_decode_tokens", "kairos_gather_latent", "kairos_mixed_step", "kairos_mixed_step_host",
           "kairos_step_latency_table", "kairos_plan_dump", "kairos_last_plan_info", "kairos_profile_enable", "kairos_profile_read", "kairos_debug_set",
           "kairos_fit_latency_model", "kairos_predict_step", "kairos_decide", "kairos_run_schedule", "kairos_absorb_q", "kairos_project_out", "kairos_simulate", "kairos_tune_step",
           "kairos_fp8_attach", "kairos_fp8_append", "kairos_fp8_append_decode_tokens", "kairos_fp8_mixed_step", "kairos_decode_static", "kairos_fp8_decode",
           "kairos_last_error", "kairos_version"]

STATUS = {0: "KAIROS_OK", -1: "KAIROS_ERR_INVALID_ARG", -2: "KAIROS_ERR_UNSUPPORTED", -3: "KAIROS_ERR_WORKSPACE",
          -4: "KAIROS_ERR_CUDA"}


class KairosError(RuntimeError):
    def __init__(self, code: int):
        self.code = code
        super().__init__(f"{STATUS.get(code, code)}: {_lib.kairos_last_error().decode()}")


def _check(rc: int) -> None:
    if rc != 0:
        raise KairosError(rc)


def version() -> str:
    return _lib.kairos_version().decode()


FP8_PAGE_BYTES = 41216  # KAIROS_FP8_PAGE_BYTES
STATIC_MAX_DECODES = 128  # KAIROS_STATIC_MAX_DECODES


def workspace_bytes(max_decodes: int, max_chunk: int) -> int:
    return int(_lib.kairos_workspace_bytes(int(max_decodes), int(max_chunk)))


def _dp(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None or t.numel() == 0:
        return None
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensors only"
    return t.data_ptr()


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> Optional[int]:
    if stream is None:  # torch's current stream on the current device, through the fast C accessor
        return torch._C._cuda_getCurrentRawStream(torch.cuda.current_device()) or None
    return stream.cuda_stream or None


class Kairos:
    """One context = one paged latent pool + workspace on one device (kairos_create / kairos_destroy)."""

    def __init__(self, pool: torch.Tensor, workspace: torch.Tensor, softmax_scale: float = 1.0 / 192.0 ** 0.5):
        assert pool.is_cuda and pool.dtype == torch.bfloat16 and pool.is_contiguous()
        assert pool.dim() == 3 and pool.shape[1] == 64 and pool.shape[2] == 576
        assert workspace.is_cuda and workspace.is_contiguous()
        self.pool, self.workspace = pool, workspace  # keep the caller's buffers alive
        cfg = KairosConfig(16, 512, 64, 64, float(softmax_scale), pool.data_ptr(), int(pool.shape[0]),
                           workspace.data_ptr(), workspace.numel() * workspace.element_size(), pool.device.index or 0)
        h = _vp()
        _check(_lib.kairos_create(_c.byref(cfg), _c.byref(h)))
        self._h = h

    def close(self) -> None:
        if getattr(self, "_h", None):
            _lib.kairos_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- a1
    def append_latent(self, latent: torch.Tensor, k_rope: torch.Tensor, page_table: torch.Tensor, start_pos: int,
                      stream: Optional[torch.cuda.Stream] = None) -> None:
        n = int(latent.shape[0])
        _check(_lib.kairos_append_latent(self._h, _dp(latent), _dp(k_rope), n, _dp(page_table),
                                         int(page_table.numel()), int(start_pos), _stream_ptr(stream)))

    def append_decode_tokens(self, latent, k_rope, page_tables, positions, stream=None) -> None:
        n = int(latent.shape[0])
        _check(_lib.kairos_append_decode_tokens(self._h, _dp(latent), _dp(k_rope), n, _dp(page_tables),
                                                int(page_tables.shape[1]) if n else 1, _dp(positions),
                                                _stream_ptr(stream)))

    def gather_latent(self, page_table: torch.Tensor, n_tokens: int, stream=None) -> torch.Tensor:
        out = torch.empty((n_tokens, 576), dtype=torch.bfloat16, device=self.pool.device)
        _check(_lib.kairos_gather_latent(self._h, _dp(page_table), int(page_table.numel()), int(n_tokens), _dp(out),
                                         _stream_ptr(stream)))
        return out

    # -- a2..a10
    def mixed_step(self, q_dec, dec_page_tables, dec_ctx_lens: Sequence[int], q_chunk, chunk_page_table,
                   chunk_len: int, prefix_len: int, out_dec=None, out_chunk=None, lse_dec=None, lse_chunk=None,
                   want_lse: bool = True, stream=None):
        dev = self.pool.device
        lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
        B, C = int(lens.shape[0]), int(chunk_len)
        if out_dec is None:
            out_dec = torch.empty((B, 16, 512), dtype=torch.bfloat16, device=dev)
        if out_chunk is None:
            out_chunk = torch.empty((C, 16, 512), dtype=torch.bfloat16, device=dev)
        if want_lse and lse_dec is None:
            lse_dec = torch.empty((B, 16), dtype=torch.float32, device=dev)
        if want_lse and lse_chunk is None:
            lse_chunk = torch.empty((C, 16), dtype=torch.float32, device=dev)
        stride = int(dec_page_tables.shape[1]) if B else 1
        _check(_lib.kairos_mixed_step(self._h, B, _dp(q_dec), _dp(dec_page_tables), stride,
                                      lens.ctypes.data_as(_vp), C, int(prefix_len), _dp(q_chunk),
                                      _dp(chunk_page_table), int(chunk_page_table.numel()) if C else 0, _dp(out_dec),
                                      _dp(out_chunk), _dp(lse_dec), _dp(lse_chunk), _stream_ptr(stream)))
        return out_dec, out_chunk, lse_dec, lse_chunk

    # -- fp8 latent cache
    def fp8_attach(self, pool8: torch.Tensor) -> None:
        """pool8: uint8 [num_pages, 41216] on the device (kept alive by this object)."""
        assert pool8.dtype == torch.uint8 and pool8.dim() == 2 and pool8.shape[1] == FP8_PAGE_BYTES
        self._pool8 = pool8
        _check(_lib.kairos_fp8_attach(self._h, _dp(pool8), int(pool8.shape[0])))

    def fp8_append(self, latent: torch.Tensor, k_rope: torch.Tensor, page_table: torch.Tensor, start_pos: int, stream=None) -> None:
        _check(_lib.kairos_fp8_append(self._h, _dp(latent), _dp(k_rope), int(latent.shape[0]), _dp(page_table),
                                      int(page_table.numel()), int(start_pos), _stream_ptr(stream)))

    def fp8_append_decode_tokens(self, latent, k_rope, page_tables, positions, stream=None) -> None:
        n = int(latent.shape[0])
        _check(_lib.kairos_fp8_append_decode_tokens(self._h, _dp(latent), _dp(k_rope), n, _dp(page_tables),
                                                    int(page_tables.shape[1]) if n else 1, _dp(positions), _stream_ptr(stream)))

    def fp8_mixed_step(self, q_dec, dec_page_tables, dec_ctx_lens: Sequence[int], q_chunk, chunk_page_table, chunk_len: int,
                       prefix_len: int, out_dec=None, out_chunk=None, lse_dec=None, lse_chunk=None, want_lse: bool = True, stream=None):
        """kairos_fp8_mixed_step: as mixed_step, over the attached fp8 pool."""
        lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
        B, C = int(lens.shape[0]), int(chunk_len)
        dev = self._pool8.device
        if out_dec is None:
            out_dec = torch.empty((B, 16, 512), dtype=torch.bfloat16, device=dev)
        if out_chunk is None:
            out_chunk = torch.empty((C, 16, 512), dtype=torch.bfloat16, device=dev)
        if want_lse and lse_dec is None:
            lse_dec = torch.empty((B, 16), dtype=torch.float32, device=dev)
        if want_lse and lse_chunk is None:
            lse_chunk = torch.empty((C, 16), dtype=torch.float32, device=dev)
        _check(_lib.kairos_fp8_mixed_step(self._h, B, _dp(q_dec), _dp(dec_page_tables), int(dec_page_tables.shape[1]) if B else 1,
                                          lens.ctypes.data_as(_vp), C, int(prefix_len), _dp(q_chunk), _dp(chunk_page_table),
                                          int(chunk_page_table.numel()) if C else 0, _dp(out_dec), _dp(out_chunk), _dp(lse_dec),
                                          _dp(lse_chunk), _stream_ptr(stream)))
        return out_dec, out_chunk, lse_dec, lse_chunk

    def fp8_decode(self, q_dec, dec_page_tables, dec_ctx_lens: Sequence[int], out_dec=None, lse_dec=None, want_lse: bool = True,
                   stream=None):
        lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
        B = int(lens.shape[0])
        dev = q_dec.device
        if out_dec is None:
            out_dec = torch.empty((B, 16, 512), dtype=torch.bfloat16, device=dev)
        if want_lse and lse_dec is None:
            lse_dec = torch.empty((B, 16), dtype=torch.float32, device=dev)
        _check(_lib.kairos_fp8_decode(self._h, B, _dp(q_dec), _dp(dec_page_tables), int(dec_page_tables.shape[1]) if B else 1,
                                      lens.ctypes.data_as(_vp), _dp(out_dec), _dp(lse_dec), _stream_ptr(stream)))
        return out_dec, lse_dec

    def decode_static(self, q_dec, dec_page_tables, dec_ctx_lens: Sequence[int], out_dec, lse_dec=None, stream=None) -> None:
        """kairos_decode_static: decode attention with no allocation (scratch is a fixed device array of the library; at most
        STATIC_MAX_DECODES requests; calls that overlap on the GPU race).  The caller passes the output tensors."""
        lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
        B = int(lens.shape[0])
        _check(_lib.kairos_decode_static(self._h, B, _dp(q_dec), _dp(dec_page_tables), int(dec_page_tables.shape[1]) if B else 1,
                                         lens.ctypes.data_as(_vp), _dp(out_dec), _dp(lse_dec), _stream_ptr(stream)))

    def tune_step(self, q_dec, dec_page_tables, dec_ctx_lens: Sequence[int], q_chunk, chunk_page_table, chunk_len: int,
                  prefix_len: int, out_dec, out_chunk, reps: int = 5, stream=None):
        """kairos_tune_step: (pinned order or -1, its median us, the planner's own order's median us).  Synchronises."""
        lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
        B, C = int(lens.shape[0]), int(chunk_len)
        stride = int(dec_page_tables.shape[1]) if B else 1
        mode, us, dus = _i32(-1), _c.c_double(0.0), _c.c_double(0.0)
        _check(_lib.kairos_tune_step(self._h, B, _dp(q_dec), _dp(dec_page_tables), stride, lens.ctypes.data_as(_vp), C,
                                     int(prefix_len), _dp(q_chunk), _dp(chunk_page_table),
                                     int(chunk_page_table.numel()) if C else 0, _dp(out_dec), _dp(out_chunk), int(reps),
                                     _c.byref(mode), _c.byref(us), _c.byref(dus), _stream_ptr(stream)))
        return int(mode.value), float(us.value), float(dus.value)

    def bind_step(self, q_dec, dec_page_tables, dec_ctx_lens: Sequence[int], q_chunk, chunk_page_table, chunk_len: int,
                  prefix_len: int, out_dec, out_chunk, lse_dec=None, lse_chunk=None, chunk_latent=None, chunk_k_rope=None):
        """Marshals the arguments of a step ONCE (a serving loop passes the same buffers step after step) and returns a
        BoundStep whose run() makes the C call -- kairos_mixed_step, or, when chunk_latent / chunk_k_rope are given, the
        one-step kairos_run_schedule that appends the chunk and runs the step -- with no per-call tensor inspection.  The tensors are kept alive by the object."""
        return BoundStep(self, q_dec, dec_page_tables, dec_ctx_lens, q_chunk, chunk_page_table, chunk_len, prefix_len,
                         out_dec, out_chunk, lse_dec, lse_chunk, chunk_latent, chunk_k_rope)

    def mixed_step_host(self, q_dec: np.ndarray, dec_page_tables: np.ndarray, dec_ctx_lens: np.ndarray,
                        q_chunk: np.ndarray, chunk_latent: np.ndarray, chunk_k_rope: np.ndarray,
                        chunk_page_table: np.ndarray, chunk_len: int, prefix_len: int, out_dec: np.ndarray,
                        out_chunk: np.ndarray, stream=None, lse_dec: Optional[np.ndarray] = None,
                        lse_chunk: Optional[np.ndarray] = None):
        """HOST buffers in, HOST buffers out (numpy uint16 views of bf16; pin them with torch for speed); lse_* = optional
        float32 HOST arrays [n_dec, 16] / [chunk_len, 16]."""
        lens = np.ascontiguousarray(dec_ctx_lens, dtype=np.int32)
        B, C = int(lens.shape[0]), int(chunk_len)
        h2d, d2h = _c.c_uint64(0), _c.c_uint64(0)

        def hp(a):
            return None if a is None or a.size == 0 else a.ctypes.data_as(_vp)
        stride = int(dec_page_tables.shape[1]) if B else 1
        _check(_lib.kairos_mixed_step_host(self._h, B, hp(q_dec), hp(dec_page_tables), stride, hp(lens), C,
                                           int(prefix_len), hp(q_chunk), hp(chunk_latent), hp(chunk_k_rope),
                                           hp(chunk_page_table), int(chunk_page_table.size) if C else 0, hp(out_dec),
                                           hp(out_chunk), hp(lse_dec), hp(lse_chunk), _c.byref(h2d), _c.byref(d2h),
                                           _stream_ptr(stream)))
        return int(h2d.value), int(d2h.value)

    # -- SURVEY.md 8(f) row 2
    def absorb_q(self, q_nope, q_rope, w_uk_t, q_out=None, stream=None):
        n = int(q_nope.shape[0])
        if q_out is None:
            q_out = torch.empty((n, 16, 576), dtype=torch.bfloat16, device=self.pool.device)
        _check(_lib.kairos_absorb_q(self._h, _dp(q_nope), _dp(q_rope), _dp(w_uk_t), n, _dp(q_out), _stream_ptr(stream)))
        return q_out

    def project_out(self, o_lat, w_uv_t, v_out=None, stream=None):
        n = int(o_lat.shape[0])
        if v_out is None:
            v_out = torch.empty((n, 16, 128), dtype=torch.bfloat16, device=self.pool.device)
        _check(_lib.kairos_project_out(self._h, _dp(o_lat), _dp(w_uv_t), n, _dp(v_out), _stream_ptr(stream)))
        return v_out

    # -- SURVEY.md 8(f) row 3
    def run_schedule(self, q_dec, dec_page_tables, dec_ctx_lens, dec_latent, dec_k_rope, chunk_sizes, q_prompt,
                     prompt_latent, prompt_k_rope, prompt_page_table, prefix_len: int = 0, out_dec=None, out_prompt=None,
                     lse_dec=None, lse_prompt=None, time_steps: bool = False, timed: bool = True, stream=None):
        """kairos_run_schedule.  Returns (out_dec [m,B,16,512], out_prompt [l,16,512], lse_dec, lse_prompt, ttft_us, step_us)."""
        dev = self.pool.device
        lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
        cs = np.ascontiguousarray(np.asarray(chunk_sizes, dtype=np.int32))
        B, m, L = int(lens.shape[0]), int(cs.shape[0]), int(cs.sum())
        if out_dec is None:
            out_dec = torch.empty((m, B, 16, 512), dtype=torch.bfloat16, device=dev)
        if out_prompt is None:
            out_prompt = torch.empty((L, 16, 512), dtype=torch.bfloat16, device=dev)
        if lse_dec is None:
            lse_dec = torch.empty((m, B, 16), dtype=torch.float32, device=dev)
        if lse_prompt is None:
            lse_prompt = torch.empty((L, 16), dtype=torch.float32, device=dev)
        ttft = _c.c_double(0.0)
        steps = np.zeros(m, dtype=np.float64)
        stride = int(dec_page_tables.shape[1]) if B else 1
        _check(_lib.kairos_run_schedule(self._h, B, _dp(q_dec), _dp(dec_page_tables), stride, lens.ctypes.data_as(_vp),
                                        _dp(dec_latent), _dp(dec_k_rope), L, cs.ctypes.data_as(_vp), m, _dp(q_prompt),
                                        _dp(prompt_latent), _dp(prompt_k_rope), _dp(prompt_page_table),
                                        int(prompt_page_table.numel()), int(prefix_len), _dp(out_dec), _dp(out_prompt),
                                        _dp(lse_dec), _dp(lse_prompt), steps.ctypes.data_as(_vp) if time_steps else None,
                                        _c.byref(ttft) if (timed or time_steps) else None, _stream_ptr(stream)))
        return out_dec, out_prompt, lse_dec, lse_prompt, float(ttft.value), (steps if time_steps else None)

    # -- a11
    def step_latency_table(self, Bs: Sequence[int], Ks: Sequence[int], Cs: Sequence[int], prefix_len: int = 0,
                           warmup: int = 5, reps: int = 20, flush_l2: bool = True, stream=None):
        Bs_, Ks_, Cs_ = (np.ascontiguousarray(np.asarray(x, dtype=np.int32)) for x in (Bs, Ks, Cs))
        med = np.zeros((len(Bs_), len(Ks_), len(Cs_)), dtype=np.float64)
        mn = np.zeros_like(med)
        _check(_lib.kairos_step_latency_table(self._h, Bs_.ctypes.data_as(_vp), len(Bs_), Ks_.ctypes.data_as(_vp),
                                              len(Ks_), Cs_.ctypes.data_as(_vp), len(Cs_), int(prefix_len),
                                              int(warmup), int(reps), int(bool(flush_l2)), med.ctypes.data_as(_vp),
                                              mn.ctypes.data_as(_vp), _stream_ptr(stream)))
        return med, mn

    def profile_enable(self, on: bool) -> None:
        _check(_lib.kairos_profile_enable(self._h, int(bool(on))))

    def profile_read(self):
        """(summed main-kernel microseconds, launches) since the last read; synchronises the recorded events."""
        us, n = _c.c_double(0.0), _c.c_int64(0)
        _check(_lib.kairos_profile_read(self._h, _c.byref(us), _c.byref(n)))
        return float(us.value), int(n.value)

    def last_plan_info(self) -> dict:
        info = (_c.c_int64 * 10)()
        _check(_lib.kairos_last_plan_info(self._h, info, 10))
        keys = ["work_items", "decode_splits", "chunk_tiles", "ctas", "kernels", "workspace_bytes", "chunk_pairs",
                "plan_cache", "graph", "dec_ctas_first"]
        return dict(zip(keys, (int(x) for x in info)))

    def debug_set(self, key: str, value: int) -> None:
        """Test-only knobs (kairos_debug_set)."""
        _check(_lib.kairos_debug_set(self._h, key.encode(), int(value)))


class BoundStep:
    """Pre-marshalled (append, mixed step) pair: see Kairos.bind_step.  Argument marshalling only."""

    def __init__(self, ctx, q_dec, dec_page_tables, dec_ctx_lens, q_chunk, chunk_page_table, chunk_len, prefix_len, out_dec,
                 out_chunk, lse_dec, lse_chunk, chunk_latent, chunk_k_rope):
        self._keep = (ctx, q_dec, dec_page_tables, q_chunk, chunk_page_table, out_dec, out_chunk, lse_dec, lse_chunk,
                      chunk_latent, chunk_k_rope)
        self._lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
        B, C = int(self._lens.shape[0]), int(chunk_len)
        stride = int(dec_page_tables.shape[1]) if B else 1
        self._h = ctx._h
        self._step_args = (B, _dp(q_dec), _dp(dec_page_tables), stride, self._lens.ctypes.data_as(_vp), C, int(prefix_len),
                           _dp(q_chunk), _dp(chunk_page_table), int(chunk_page_table.numel()) if C else 0, _dp(out_dec),
                           _dp(out_chunk), _dp(lse_dec), _dp(lse_chunk))
        self._sched_args = None
        if C and chunk_latent is not None:
            # append + step as a one-step chunk schedule: kairos_run_schedule captures the append, the attention grid(s) and
            # the combine into ONE graph (one launch per step instead of an append launch plus a graph launch)
            self._cs = np.array([C], dtype=np.int32)
            self._sched_args = (B, _dp(q_dec), _dp(dec_page_tables), stride, self._lens.ctypes.data_as(_vp), None, None, C,
                                self._cs.ctypes.data_as(_vp), 1, _dp(q_chunk), _dp(chunk_latent), _dp(chunk_k_rope),
                                _dp(chunk_page_table), int(chunk_page_table.numel()), int(prefix_len), _dp(out_dec),
                                _dp(out_chunk), _dp(lse_dec), _dp(lse_chunk), None, None)

    def run(self, stream: Optional[torch.cuda.Stream] = None) -> None:
        sp = _stream_ptr(stream)
        if self._sched_args is not None:
            rc = _lib.kairos_run_schedule(self._h, *self._sched_args, sp)
        else:
            rc = _lib.kairos_mixed_step(self._h, *self._step_args, sp)
        if rc:
            raise KairosError(rc)


def plan_dump(dec_ctx_lens: Sequence[int], chunk_len: int, prefix_len: int, n_ctas: int = 148, pair_mode: int = 0,
              with_pairs: bool = False):
    """Host planner alone (kairos_plan_dump): (items int32 [n, 8], n_partial_slots[, n_pairs]). No GPU needed."""
    lens = np.ascontiguousarray(np.asarray(dec_ctx_lens, dtype=np.int32))
    n, slots, pairs = _c.c_int32(0), _c.c_int32(0), _c.c_int32(0)
    lp = lens.ctypes.data_as(_vp) if lens.size else None
    args = (lp, int(lens.size), int(chunk_len), int(prefix_len), int(n_ctas), int(pair_mode))
    _check(_lib.kairos_plan_dump(*args, None, 0, _c.byref(n), _c.byref(slots), _c.byref(pairs)))
    items = np.zeros((int(n.value), 8), dtype=np.int32)
    _check(_lib.kairos_plan_dump(*args, items.ctypes.data_as(_vp), int(n.value), _c.byref(n), _c.byref(slots),
                                 _c.byref(pairs)))
    if with_pairs:
        return items, int(slots.value), int(pairs.value)
    return items, int(slots.value)


# -- latency model, chunk schedule, deflection decision (host only)
def fit_latency_model(B, Kd, C, P, T):
    """kairos_fit_latency_model: (StepModel, in-sample MAPE)."""
    arr = [np.ascontiguousarray(np.asarray(x, dtype=np.int64)) for x in (B, Kd, C, P)]
    Tn = np.ascontiguousarray(np.asarray(T, dtype=np.float64))
    m, mape = StepModel(), _c.c_double(0.0)
    _check(_lib.kairos_fit_latency_model(*(a.ctypes.data_as(_vp) for a in arr), Tn.ctypes.data_as(_vp), int(Tn.size),
                                         _c.byref(m), _c.byref(mape)))
    return m, float(mape.value)


def step_model(a, b) -> StepModel:
    m = StepModel()
    m.a[:] = [float(x) for x in a]
    m.b[:] = [float(x) for x in b]
    return m


def prefill_model(p) -> PrefillModel:
    m = PrefillModel()
    m.p[:] = [float(x) for x in p]
    return m


def predict_step(model: StepModel, B: int, Kd: int, C: int, P: int) -> float:
    return float(_lib.kairos_predict_step(_c.byref(model), int(B), int(Kd), int(C), int(P)))


def decide(model: StepModel, prefill: PrefillModel, prompt_len: int, queue_lens, chi_p: int, nodes, candidates,
           tbt_slo: float, beta: float, alpha: float, ttft_slo: float, max_schedule: int = 4096):
    """kairos_decide (Algorithm 1): (decision 'KEEP'|'DEFLECT', n_star, X_star, ttft_pf, ttft_dec)."""
    q = np.ascontiguousarray(np.asarray(queue_lens, dtype=np.int32))
    nb = np.ascontiguousarray(np.asarray([n[0] for n in nodes], dtype=np.int32))
    nk = np.ascontiguousarray(np.asarray([n[1] for n in nodes], dtype=np.int64))
    cand = np.ascontiguousarray(np.asarray(candidates, dtype=np.int32))
    ptr = lambda a: a.ctypes.data_as(_vp) if a.size else None
    inp = DecideInput(int(prompt_len), ptr(q), int(q.size), int(chi_p), ptr(nb), ptr(nk), int(nb.size), ptr(cand),
                      int(cand.size), float(tbt_slo), float(beta), float(alpha), float(ttft_slo))
    sched = np.zeros(max_schedule, dtype=np.int32)
    out = DecideOutput()
    _check(_lib.kairos_decide(_c.byref(model), _c.byref(prefill), _c.byref(inp), sched.ctypes.data_as(_vp), max_schedule,
                              _c.byref(out)))
    return ("DEFLECT" if out.decision else "KEEP"), int(out.node), sched[:out.n_steps].tolist(), float(out.ttft_pf), float(out.ttft_dec)


POLICIES = {"baseline": 0, "sq": 1, "sl": 2, "oracle": 3}


def simulate(model: StepModel, prefill: PrefillModel, reqs, n_prefill: int, n_decode: int, chi_p: int, policy: str,
             param: int = 0, static_chi: int = 128, candidates=(2048, 1024, 512, 256, 128), tbt_slo: float = 1e30,
             beta: float = 1.0, alpha: float = 1.0, ttft_slo: float = 1e30, transfer_per_token: float = 0.0):
    """kairos_simulate: reqs = sequence of (arrival, prompt_len, output_len) sorted by arrival.  Returns (dict, ttft array)."""
    n = len(reqs)
    arr = (SimRequest * max(n, 1))()
    for i, (t, l, o) in enumerate(reqs):
        arr[i] = SimRequest(float(t), int(l), int(o))
    cand = np.ascontiguousarray(np.asarray(candidates, dtype=np.int32))
    cfg = SimConfig(int(n_prefill), int(n_decode), int(chi_p), POLICIES[policy], int(param), int(static_chi),
                    cand.ctypes.data_as(_vp), int(cand.size), float(tbt_slo), float(beta), float(alpha), float(ttft_slo),
                    float(transfer_per_token))
    ttft = np.zeros(max(n, 1), dtype=np.float64)
    res = SimResult()
    _check(_lib.kairos_simulate(_c.byref(model), _c.byref(prefill), _c.byref(cfg), arr, n, ttft.ctypes.data_as(_vp),
                                _c.byref(res)))
    return {k: getattr(res, k) for k, _ in SimResult._fields_}, ttft[:n]


def bf16_tensor(bits: np.ndarray, device="cuda") -> torch.Tensor:
    """numpy uint16 bf16 bit patterns -> torch.bfloat16 tensor on `device` (bit-exact)."""
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device).view(torch.bfloat16)


def bf16_bits(t: torch.Tensor) -> np.ndarray:
    """torch.bfloat16 tensor -> numpy uint16 bit patterns (bit-exact)."""
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
