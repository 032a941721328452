"""Thin ctypes binding over libdwkv.so (include/dwkv.h). Argument marshalling only: every step of the hot path runs in
the CUDA kernels behind the C ABI. torch is used for device memory (tensor.data_ptr()) and the current stream.

There is no CPU fallback: if libdwkv.so is missing or cannot be loaded this module raises at import time.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdwkv.so")

DWKV_OK, DWKV_E_INVALID, DWKV_E_STATE, DWKV_E_CAPACITY, DWKV_E_EMPTY, DWKV_E_CUDA = 0, -1, -2, -3, -4, -5
_ERR_NAMES = {-1: "DWKV_E_INVALID", -2: "DWKV_E_STATE", -3: "DWKV_E_CAPACITY", -4: "DWKV_E_EMPTY", -5: "DWKV_E_CUDA"}

EXPORTED = [
    "dwkv_create", "dwkv_destroy", "dwkv_set_basis", "dwkv_set_gates", "dwkv_append_compress", "dwkv_decode_attention",
    "dwkv_append_raw", "dwkv_export_tokens", "dwkv_reset_seq", "dwkv_seq_len", "dwkv_footprint", "dwkv_set_option",
    "dwkv_launch_count", "dwkv_get_stat", "dwkv_last_error", "dwkv_dense_workspace_bytes", "dwkv_dense_decode_attention",
    "dwkv_build_basis", "dwkv_export_basis", "dwkv_probe_error", "dwkv_route_tokens", "dwkv_router_thresholds",
    "dwkv_probe_token_stats", "dwkv_controller_create", "dwkv_controller_destroy", "dwkv_controller_step", "dwkv_controller_state",
    "dwkv_controller_thresholds", "dwkv_dense_decode_attention_static", "dwkv_retier_seq",
]


class DwkvError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class dwkv_config(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("group_size", C.c_int32), ("n_kv_heads", C.c_int32), ("n_q_heads", C.c_int32),
                ("d_head", C.c_int32), ("n_tiers", C.c_int32), ("tier_rank", C.c_int32 * 4), ("max_seqs", C.c_int32),
                ("max_tokens_per_seq", C.c_int64), ("softmax_scale", C.c_float), ("device", C.c_int32),
                ("arena", C.c_void_p), ("arena_bytes", C.c_uint64)]


class dwkv_controller_config(C.Structure):
    _fields_ = [("n_windows", C.c_int32), ("patience", C.c_int32), ("tol_default", C.c_float), ("tol", C.c_void_p),
                ("step_down", C.c_float), ("step_up", C.c_float), ("delta_min", C.c_float), ("delta_max", C.c_float)]


class dwkv_raw_tokens(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("coefK", "coefV", "residK", "residV", "codeK", "codeV", "scaleK", "scaleV")]


class dwkv_token_dump(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("tier", "flag", "slot", "coefK", "coefV", "codeK", "codeV", "scaleK", "scaleV",
                                          "deqK", "deqV")]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2607_06523_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
    lib.dwkv_create.argtypes = [C.POINTER(dwkv_config), C.POINTER(vp)]
    lib.dwkv_destroy.argtypes = [vp]
    lib.dwkv_destroy.restype = None
    lib.dwkv_set_basis.argtypes = [vp, vp, vp, vp]
    lib.dwkv_set_gates.argtypes = [vp, vp, vp, vp]
    lib.dwkv_build_basis.argtypes = [vp, i32, vp, vp, vp, i32, vp]
    lib.dwkv_export_basis.argtypes = [vp, vp, vp, vp]
    lib.dwkv_probe_error.argtypes = [vp, i32, i32, i32, vp, vp, vp, C.c_float, vp, vp]
    lib.dwkv_route_tokens.argtypes = [i64, vp, vp, i32, vp, C.c_float, vp, vp]
    lib.dwkv_router_thresholds.argtypes = [i64, vp, vp, i32, vp, C.c_float, vp, vp]
    lib.dwkv_probe_token_stats.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    lib.dwkv_controller_create.argtypes = [C.POINTER(dwkv_controller_config), C.POINTER(vp)]
    lib.dwkv_controller_destroy.argtypes = [vp]
    lib.dwkv_controller_destroy.restype = None
    lib.dwkv_controller_step.argtypes = [vp, i32, vp, vp]
    lib.dwkv_controller_state.argtypes = [vp, vp, vp]
    lib.dwkv_controller_thresholds.argtypes = [vp, i32, vp, C.c_float, vp, vp]
    lib.dwkv_append_compress.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.dwkv_decode_attention.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    lib.dwkv_append_raw.argtypes = [vp, i32, i32, vp, vp, C.POINTER(dwkv_raw_tokens), vp]
    lib.dwkv_export_tokens.argtypes = [vp, i32, i64, i64, C.POINTER(dwkv_token_dump), vp]
    lib.dwkv_reset_seq.argtypes = [vp, i32]
    lib.dwkv_retier_seq.argtypes = [vp, i32, vp, vp, vp]
    lib.dwkv_seq_len.argtypes = [vp, i32]
    lib.dwkv_seq_len.restype = i64
    lib.dwkv_footprint.argtypes = [vp, C.POINTER(u64), C.POINTER(u64), C.POINTER(u64)]
    lib.dwkv_set_option.argtypes = [vp, C.c_char_p, i64]
    lib.dwkv_launch_count.argtypes = [vp]
    lib.dwkv_launch_count.restype = i64
    lib.dwkv_get_stat.argtypes = [vp, C.c_char_p]
    lib.dwkv_get_stat.restype = C.c_double
    lib.dwkv_last_error.restype = C.c_char_p
    lib.dwkv_dense_workspace_bytes.argtypes = [i32, i32, i32, i32, i64]
    lib.dwkv_dense_workspace_bytes.restype = u64
    lib.dwkv_dense_decode_attention.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i64, C.c_float, vp]
    lib.dwkv_dense_decode_attention_static.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, i64, C.c_float, vp]
    for name in EXPORTED:
        getattr(lib, name)
    return lib


lib = _load()


def _check(rc: int):
    if rc != 0:
        raise DwkvError(rc, (lib.dwkv_last_error() or b"").decode())


def _ptr(t: Optional[torch.Tensor], dtype=None) -> Optional[int]:
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device-resident contiguous tensor required"
    if dtype is not None:
        assert t.dtype == dtype, f"expected {dtype}, got {t.dtype}"
    return t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _u8(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.uint8))


class DwkvCache:
    """Handle of one dwkv_cache. Method names follow the C ABI (dwkv_<name>)."""

    def __init__(self, n_layers, group_size, n_kv_heads, n_q_heads, d_head, tier_ranks: Sequence[int], max_seqs,
                 max_tokens_per_seq, softmax_scale: float = 0.0, device: int = 0, arena: Optional[torch.Tensor] = None,
                 arena_bytes: int = 0):
        cfg = dwkv_config()
        cfg.n_layers, cfg.group_size, cfg.n_kv_heads, cfg.n_q_heads = n_layers, group_size, n_kv_heads, n_q_heads
        cfg.d_head, cfg.n_tiers = d_head, len(tier_ranks)
        for i in range(4):
            cfg.tier_rank[i] = tier_ranks[i] if i < len(tier_ranks) else 0
        cfg.max_seqs, cfg.max_tokens_per_seq, cfg.softmax_scale, cfg.device = max_seqs, max_tokens_per_seq, softmax_scale, device
        self._arena = arena
        cfg.arena = arena.data_ptr() if arena is not None else None
        cfg.arena_bytes = arena.numel() * arena.element_size() if arena is not None else arena_bytes
        self.L, self.H, self.Hq, self.d, self.r = n_layers, n_kv_heads, n_q_heads, d_head, tier_ranks[-1]
        self.w = group_size
        h = C.c_void_p()
        _check(lib.dwkv_create(C.byref(cfg), C.byref(h)))
        self._h = h

    def destroy(self):
        if getattr(self, "_h", None):
            lib.dwkv_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_basis(self, BK: torch.Tensor, BV: torch.Tensor):
        _check(lib.dwkv_set_basis(self._h, _ptr(BK, torch.bfloat16), _ptr(BV, torch.bfloat16), _stream()))

    def build_basis(self, k_dense: torch.Tensor, v_dense: torch.Tensor, omega: torch.Tensor):
        """k_dense, v_dense: bf16 [n, L, H_kv, d]; omega: bf16 [w, n_sketch, n] (the random test matrix, an input)."""
        n, n_sketch = int(k_dense.shape[0]), int(omega.shape[1])
        assert k_dense.shape == v_dense.shape and omega.shape[2] == n
        _check(lib.dwkv_build_basis(self._h, n, _ptr(k_dense, torch.bfloat16), _ptr(v_dense, torch.bfloat16),
                                    _ptr(omega, torch.bfloat16), n_sketch, _stream()))

    def export_basis(self, M: int, H: int, r: int, d: int):
        BK = torch.empty(M, H, r, d, dtype=torch.bfloat16, device=torch.device("cuda", torch.cuda.current_device()))
        BV = torch.empty_like(BK)
        _check(lib.dwkv_export_basis(self._h, _ptr(BK, torch.bfloat16), _ptr(BV, torch.bfloat16), _stream()))
        return BK, BV

    def probe_error(self, layer: int, seq_id: int, q: torch.Tensor, K_ref: torch.Tensor, V_ref: torch.Tensor, eps: float = 1e-6):
        """q: bf16 [n_q, H_q, d]; K_ref, V_ref: bf16 [H_kv, T, d]. Returns fp32 [H_kv] (Eq. 3 of the paper)."""
        e = torch.empty(K_ref.shape[0], dtype=torch.float32, device=q.device)
        _check(lib.dwkv_probe_error(self._h, layer, seq_id, int(q.shape[0]), _ptr(q, torch.bfloat16), _ptr(K_ref, torch.bfloat16),
                                    _ptr(V_ref, torch.bfloat16), float(eps), _ptr(e, torch.float32), _stream()))
        return e

    def probe_token_stats(self, layer: int, seq_id: int, q: torch.Tensor, mass: torch.Tensor, spike: torch.Tensor):
        """q: bf16 [H_q, d]; mass, spike: fp32 [T] on the device, updated in place (mass += sum_hq p, spike = max(spike, max_hq p))."""
        _check(lib.dwkv_probe_token_stats(self._h, layer, seq_id, _ptr(q, torch.bfloat16), _ptr(mass, torch.float32),
                                          _ptr(spike, torch.float32), _stream()))

    def set_gates(self, gK: torch.Tensor, gV: torch.Tensor):
        _check(lib.dwkv_set_gates(self._h, _ptr(gK, torch.bfloat16), _ptr(gV, torch.bfloat16), _stream()))

    def append_compress(self, seq_ids, n_new, k_new: torch.Tensor, v_new: torch.Tensor, tier, flag):
        s, n, t, f = _i32(seq_ids), _i32(n_new), _u8(tier), _u8(flag)
        assert len(t) == int(n.sum()) == len(f)
        _check(lib.dwkv_append_compress(self._h, len(s), s.ctypes.data, n.ctypes.data, _ptr(k_new, torch.bfloat16),
                                        _ptr(v_new, torch.bfloat16), t.ctypes.data, f.ctypes.data, _stream()))

    def append_raw(self, seq_id: int, tier, flag, coefK, coefV, residK=None, residV=None, codeK=None, codeV=None,
                   scaleK=None, scaleV=None):
        t, f = _u8(tier), _u8(flag)
        raw = dwkv_raw_tokens(_ptr(coefK, torch.bfloat16), _ptr(coefV, torch.bfloat16), _ptr(residK, torch.float32),
                              _ptr(residV, torch.float32), _ptr(codeK, torch.uint8), _ptr(codeV, torch.uint8),
                              _ptr(scaleK, torch.float16), _ptr(scaleV, torch.float16))
        _check(lib.dwkv_append_raw(self._h, seq_id, len(t), t.ctypes.data, f.ctypes.data, C.byref(raw), _stream()))

    def decode_attention(self, layer: int, seq_ids, q: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        s = _i32(seq_ids)
        if out is None:
            out = torch.empty(q.shape, dtype=torch.float32, device=q.device)
        _check(lib.dwkv_decode_attention(self._h, layer, len(s), s.ctypes.data, _ptr(q, torch.bfloat16),
                                         _ptr(out, torch.float32), _stream()))
        return out

    def export_tokens(self, seq_id: int, t0: int, n: int, want=("tier", "flag", "slot", "coefK", "coefV", "codeK", "codeV",
                                                                "scaleK", "scaleV", "deqK", "deqV")):
        dev = torch.device("cuda", torch.cuda.current_device())
        L, H, d, r = self.L, self.H, self.d, self.r
        shapes = dict(tier=((n,), torch.uint8), flag=((n,), torch.uint8), slot=((n,), torch.int32),
                      coefK=((n, L, H, r), torch.bfloat16), coefV=((n, L, H, r), torch.bfloat16),
                      codeK=((n, L, H, d // 2), torch.uint8), codeV=((n, L, H, d // 2), torch.uint8),
                      scaleK=((n, L, H, d // 16), torch.float16), scaleV=((n, L, H, d // 16), torch.float16),
                      deqK=((n, L, H, d), torch.float32), deqV=((n, L, H, d), torch.float32))
        out = {k: torch.empty(shapes[k][0], dtype=shapes[k][1], device=dev) for k in want}
        dump = dwkv_token_dump(*[out[k].data_ptr() if k in out else None for k, _ in dwkv_token_dump._fields_])
        _check(lib.dwkv_export_tokens(self._h, seq_id, t0, n, C.byref(dump), _stream()))
        return out

    def reset_seq(self, seq_id: int):
        _check(lib.dwkv_reset_seq(self._h, seq_id))

    def retier_seq(self, seq_id: int, new_tier, new_flag):
        """Lower the class of stored tokens (dwkv_retier_seq): new_tier / new_flag host uint8 [seq_len], element-wise <= the stored ones."""
        t, f = _u8(new_tier), _u8(new_flag)
        n = self.seq_len(seq_id)
        if len(t) != n or len(f) != n:
            raise ValueError(f"retier_seq needs {n} tiers and flags")
        _check(lib.dwkv_retier_seq(self._h, seq_id, t.ctypes.data, f.ctypes.data, _stream()))

    def seq_len(self, seq_id: int) -> int:
        n = lib.dwkv_seq_len(self._h, seq_id)
        if n < 0:
            _check(int(n))
        return int(n)

    def footprint(self):
        a, b, c = C.c_uint64(), C.c_uint64(), C.c_uint64()
        _check(lib.dwkv_footprint(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return dict(used_bytes=a.value, reserved_bytes=b.value, dense_equiv_bytes=c.value)

    def set_option(self, key: str, value: int):
        _check(lib.dwkv_set_option(self._h, key.encode(), int(value)))

    def get_stat(self, key: str) -> float:
        return float(lib.dwkv_get_stat(self._h, key.encode()))

    def launch_count(self) -> int:
        return int(lib.dwkv_launch_count(self._h))


def dense_decode_attention(K: torch.Tensor, V: torch.Tensor, q: torch.Tensor, n_kv_heads: int, softmax_scale: float = 0.0,
                           workspace: Optional[torch.Tensor] = None, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """K, V bf16 [n_seqs, L, H_kv, T, d]; q bf16 [n_seqs, L, H_q, d] -> fp32 [n_seqs, L, H_q, d]."""
    n_seqs, L, H, T, d = K.shape
    Hq = q.shape[2]
    if workspace is None:
        workspace = torch.empty(lib.dwkv_dense_workspace_bytes(n_seqs, L, Hq, d, T), dtype=torch.uint8, device=K.device)
    if out is None:
        out = torch.empty(q.shape, dtype=torch.float32, device=q.device)
    _check(lib.dwkv_dense_decode_attention(_ptr(K, torch.bfloat16), _ptr(V, torch.bfloat16), _ptr(q, torch.bfloat16),
                                           _ptr(out, torch.float32), _ptr(workspace), n_seqs, L, H, Hq, d, T,
                                           softmax_scale, _stream()))
    return out


DENSE_STATIC_SCRATCH_BYTES = 16 << 20      # DWKV_DENSE_STATIC_SCRATCH_BYTES of include/dwkv.h


def dense_decode_attention_static(K: torch.Tensor, V: torch.Tensor, q: torch.Tensor, n_kv_heads: int, out: torch.Tensor,
                                  softmax_scale: float = 0.0) -> torch.Tensor:
    """dwkv_dense_decode_attention_static: the dense kernel with its split partials in the library's static device array; the
    call allocates nothing (so `out` is the caller's). Calls that overlap on the GPU race on that array."""
    n_seqs, L, H, T, d = K.shape
    _check(lib.dwkv_dense_decode_attention_static(_ptr(K, torch.bfloat16), _ptr(V, torch.bfloat16), _ptr(q, torch.bfloat16),
                                                  _ptr(out, torch.float32), n_seqs, L, H, q.shape[2], d, T, softmax_scale, _stream()))
    return out


class Controller:
    """Probe-driven threshold controller (dwkv_controller_* of the C ABI). Host-only."""

    def __init__(self, n_windows: int, tol, step_down: float, step_up: float, patience: int, delta_min: float, delta_max: float):
        cfg = dwkv_controller_config()
        cfg.n_windows, cfg.patience = n_windows, patience
        tol_arr = None
        if np.ndim(tol) == 0:
            cfg.tol_default, cfg.tol = float(tol), None
        else:
            tol_arr = np.ascontiguousarray(tol, np.float32)
            assert tol_arr.shape == (n_windows,)
            cfg.tol_default, cfg.tol = 0.0, tol_arr.ctypes.data
        cfg.step_down, cfg.step_up, cfg.delta_min, cfg.delta_max = step_down, step_up, delta_min, delta_max
        self.n_windows = n_windows
        h = C.c_void_p()
        rc = lib.dwkv_controller_create(C.byref(cfg), C.byref(h))
        if rc:
            raise DwkvError(rc, "dwkv_controller_create")
        self._h = h

    def destroy(self):
        if getattr(self, "_h", None):
            lib.dwkv_controller_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def step(self, window, e):
        w = _i32(window); x = np.ascontiguousarray(e, np.float32)
        assert len(w) == len(x)
        rc = lib.dwkv_controller_step(self._h, len(w), w.ctypes.data, x.ctypes.data)
        if rc:
            raise DwkvError(rc, "dwkv_controller_step")

    def state(self):
        d = np.zeros(self.n_windows, np.float32); q = np.zeros(self.n_windows, np.int32)
        rc = lib.dwkv_controller_state(self._h, d.ctypes.data, q.ctypes.data)
        if rc:
            raise DwkvError(rc, "dwkv_controller_state")
        return d, q

    def thresholds(self, base_tau_logit, base_flag_logit: float):
        base = np.ascontiguousarray(base_tau_logit, np.float32)
        tau = np.zeros(max(len(base), 1), np.float32); tf = C.c_float(0.0)
        rc = lib.dwkv_controller_thresholds(self._h, len(base) + 1, base.ctypes.data if len(base) else None, float(base_flag_logit),
                                            tau.ctypes.data, C.addressof(tf))
        if rc:
            raise DwkvError(rc, "dwkv_controller_thresholds")
        return tau[:len(base)], float(tf.value)


def route_tokens(phi: np.ndarray, u: np.ndarray, tau_logit, tau_flag_logit: float, n_tiers: int):
    """Host router (Eq. 2 of the paper): phi fp32 [n, 4], u fp32 [4]. Returns (tier u8 [n], flag u8 [n])."""
    phi = np.ascontiguousarray(phi, np.float32); u = np.ascontiguousarray(u, np.float32)
    tau = np.ascontiguousarray(tau_logit, np.float32)
    n = phi.shape[0]
    tier = np.zeros(n, np.uint8); flag = np.zeros(n, np.uint8)
    _check(lib.dwkv_route_tokens(n, phi.ctypes.data, u.ctypes.data, n_tiers, tau.ctypes.data if tau.size else None,
                                 float(tau_flag_logit), tier.ctypes.data, flag.ctypes.data))
    return tier, flag


def router_thresholds(phi: np.ndarray, u: np.ndarray, tier_frac, flag_frac: float):
    """Thresholds (logit space) that route the given fractions of the tokens: returns (tau_logit fp32 [n_tiers-1], tau_flag_logit)."""
    phi = np.ascontiguousarray(phi, np.float32); u = np.ascontiguousarray(u, np.float32)
    frac = np.ascontiguousarray(tier_frac, np.float32)
    tau = np.zeros(max(len(frac) - 1, 1), np.float32); tf = C.c_float(0.0)
    _check(lib.dwkv_router_thresholds(phi.shape[0], phi.ctypes.data, u.ctypes.data, len(frac), frac.ctypes.data, float(flag_frac),
                                      tau.ctypes.data, C.addressof(tf)))
    return tau[:len(frac) - 1], float(tf.value)
