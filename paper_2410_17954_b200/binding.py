"""ctypes binding of libef.so: same names as include/ef.h, argument marshalling only.

Device tensors are torch tensors (their ``data_ptr()`` is passed through); host arrays are numpy.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIBS: dict = {}

# include/ef.h
DECLARED_SYMBOLS = [
    "ef_create", "ef_destroy", "ef_host_expert_register", "ef_host_expert_alias", "ef_route_topk", "ef_permute",
    "ef_expert_ffn_grouped", "ef_expert_ffn_grouped_resident", "ef_shared_ffn", "ef_combine", "ef_rmsnorm",
    "ef_cache_prefetch", "ef_cache_evict", "ef_cache_get_stats", "ef_cache_reset_stats", "ef_cache_snapshot",
    "ef_cache_clear", "ef_set_cache_policy", "ef_copy_busy_ms", "ef_token_schedule", "ef_reindex_rows", "ef_path_hamming",
    "ef_path_hamming_static",
    "ef_sync", "ef_last_error", "ef_launch_count", "ef_set_kernel_timing", "ef_get_kernel_times", "ef_get_launch_log",
    "ef_set_option",
]
# include/ef_diag.h: only libef_diag.so (the diagnostic build) has these
DIAG_SYMBOLS = ["ef_diag_set_simt_ffn", "ef_diag_tma_fill_gbs", "ef_diag_pair_handoff_gbs", "ef_diag_kprof"]

EF_OPT_SPLITK, EF_OPT_WAVE_BYTES, EF_OPT_CHUNK_MIN_BYTES, EF_OPT_FUSED_WAVES, EF_OPT_TOKEN_SCHED_PATH, EF_OPT_COPY_ORDER = 1, 2, 3, 4, 5, 6
EF_OPT_EARLY_RELEASE = 7


class EfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libef error {code}: {msg}")
        self.code = code


class EfConfig(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("n_layers", "n_experts", "top_k", "d_model", "d_ff", "n_slots",
                                               "n_shared", "max_tokens", "prefetch_horizon", "device", "expert_kind")]


class CacheStats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in ("lookups", "hits", "misses", "prefetch_issued", "prefetch_used",
                                                "prefetch_wasted", "ondemand_loads", "evictions", "bytes_h2d")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class KernelTimes(ctypes.Structure):
    _fields_ = ([(n, ctypes.c_double) for n in ("gemm1_ms", "gemm2_ms", "wave_ms")] +
                [(n, ctypes.c_int64) for n in ("gemm1_launches", "gemm2_launches", "wave_launches", "gemm1_rows", "gemm2_rows",
                                               "wave_rows", "gemm1_groups", "gemm2_groups", "wave_groups",
                                               "gemm1_fill_bytes", "gemm2_fill_bytes")])

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class LaunchRecord(ctypes.Structure):
    _fields_ = [("which", ctypes.c_int32), ("groups", ctypes.c_int32), ("rows", ctypes.c_int64), ("ms", ctypes.c_float)]


def library_path(diag: bool = False) -> str:
    return os.path.join(_PKG, "libef_diag.so" if diag else "libef.so")


def load_library(diag: bool = False) -> ctypes.CDLL:
    """Load libef.so (built by ``python -m paper_2410_17954_b200.build``), or with diag=True the diagnostic build
    libef_diag.so (``... .build --diag``; include/ef_diag.h).  Fails loudly if absent."""
    if diag not in _LIBS:
        path = library_path(diag)
        if not os.path.exists(path):
            raise EfError(-100, f"{path} not found: build it with `python -m paper_2410_17954_b200.build"
                                f"{' --diag' if diag else ''}` (there is no CPU fallback)")
        lib = ctypes.CDLL(path)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        sig = {
            "ef_create": [ctypes.POINTER(EfConfig), ctypes.POINTER(vp)],
            "ef_destroy": [vp],
            "ef_host_expert_register": [vp, i32, i32, vp, vp, vp],
            "ef_host_expert_alias": [vp, i32, i32, i32, i32],
            "ef_route_topk": [vp, vp, vp, vp, vp, i64, i32, i32, vp, vp, vp],
            "ef_permute": [vp, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp],
            "ef_expert_ffn_grouped": [vp, vp, i64, i32, vp, vp, vp],
            "ef_expert_ffn_grouped_resident": [vp, vp, vp, i32, vp, vp, vp, vp],
            "ef_shared_ffn": [vp, vp, i32, vp, i32, vp],
            "ef_combine": [vp, vp, vp, vp, vp, i32, vp, vp, vp],
            "ef_rmsnorm": [vp, vp, vp, i32, ctypes.c_float, vp],
            "ef_cache_prefetch": [vp, i64, vp, i32],
            "ef_cache_evict": [vp, i32, vp, i32],
            "ef_cache_get_stats": [vp, ctypes.POINTER(CacheStats)],
            "ef_cache_reset_stats": [vp],
            "ef_cache_snapshot": [vp, vp],
            "ef_cache_clear": [vp],
            "ef_copy_busy_ms": [vp, ctypes.POINTER(ctypes.c_float)],
            "ef_sync": [vp],
            "ef_set_kernel_timing": [vp, i32],
            "ef_get_kernel_times": [vp, ctypes.POINTER(KernelTimes), i32],
            "ef_get_launch_log": [vp, ctypes.POINTER(LaunchRecord), i32, ctypes.POINTER(i32), i32],
            "ef_token_schedule": [vp, vp, vp, i32, i32, i32, i32, i32, vp, vp, vp, vp],
            "ef_reindex_rows": [vp, vp, vp, vp, i32, i64, vp],
            "ef_path_hamming": [vp, vp, vp, i32, i32, vp],
            "ef_path_hamming_static": [vp, vp, vp, i32, i32, vp],
            "ef_set_cache_policy": [vp, i32],
            "ef_set_option": [vp, i32, i64],
        }
        if diag:
            sig.update({"ef_diag_set_simt_ffn": [vp, i32], "ef_diag_kprof": [vp, i32, vp],
                        "ef_diag_tma_fill_gbs": [vp, i64, i32, ctypes.POINTER(ctypes.c_double)],
                        "ef_diag_pair_handoff_gbs": [vp, i64, i32, i32, i32, ctypes.POINTER(ctypes.c_double)]})
        for name, args in sig.items():
            fn = getattr(lib, name)
            fn.argtypes = args
            fn.restype = i32
        lib.ef_last_error.argtypes = [vp]
        lib.ef_last_error.restype = ctypes.c_char_p
        lib.ef_launch_count.argtypes = [vp]
        lib.ef_launch_count.restype = i64
        _LIBS[diag] = lib
    return _LIBS[diag]


def exported_symbols(diag: bool = False) -> list[str]:
    lib = load_library(diag)
    return [s for s in DECLARED_SYMBOLS + DIAG_SYMBOLS if hasattr(lib, s)]


def _dp(t):
    """device pointer of a torch tensor (or None)"""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    return ctypes.c_void_p(t.data_ptr())


def _hp(a):
    if a is None:
        return None
    assert isinstance(a, np.ndarray) and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


class EfContext:
    """One ef_ctx.  Method names and argument order follow include/ef.h."""

    def __init__(self, n_layers, n_experts, top_k, d_model, d_ff, n_slots, n_shared=0, max_tokens=1,
                 prefetch_horizon=0, device=0, expert_kind=0, diag=False):
        self.lib = load_library(diag)
        self.diag = diag
        self.cfg = EfConfig(n_layers, n_experts, top_k, d_model, d_ff, n_slots, n_shared, max_tokens,
                            prefetch_horizon, device, expert_kind)
        h = ctypes.c_void_p()
        rc = self.lib.ef_create(ctypes.byref(self.cfg), ctypes.byref(h))
        if rc != 0:
            raise EfError(rc, self.lib.ef_last_error(None).decode())
        self.h = h

    # -- plumbing
    def _chk(self, rc):
        if rc != 0:
            raise EfError(rc, self.lib.ef_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.lib.ef_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- registration
    def ef_host_expert_register(self, layer, expert, w_gate, w_up, w_down):
        for a in (w_gate, w_up, w_down):
            assert a is None or (a.dtype == np.uint16 and a.flags["C_CONTIGUOUS"])
        self._chk(self.lib.ef_host_expert_register(self.h, layer, expert, _hp(w_gate), _hp(w_up), _hp(w_down)))

    def ef_host_expert_alias(self, layer, expert, src_layer, src_expert):
        self._chk(self.lib.ef_host_expert_alias(self.h, layer, expert, src_layer, src_expert))

    # -- a1
    def ef_route_topk(self, x, w_router, bias, T, renorm, topk_idx, topk_w, logits_out=None):
        stride, bp = 0, None
        if bias is not None:
            if bias.dim() == 2:      # per-token rows; a row stride above E selects one layer of a [T, L, E] tensor
                assert bias.is_cuda and bias.stride(1) == 1
                stride, bp = bias.stride(0), ctypes.c_void_p(bias.data_ptr())
            else:
                bp = _dp(bias)
        self._chk(self.lib.ef_route_topk(self.h, _stream(), _dp(x), _dp(w_router), bp, stride, T, renorm,
                                         _dp(topk_idx), _dp(topk_w), _dp(logits_out)))

    # -- a2
    def ef_permute(self, topk_idx, x, T, x_perm, counts, offsets, src, inv, counts_host_pinned=None):
        chp = None
        if counts_host_pinned is not None:
            assert counts_host_pinned.is_pinned()
            chp = ctypes.c_void_p(counts_host_pinned.data_ptr())
        self._chk(self.lib.ef_permute(self.h, _stream(), _dp(topk_idx), _dp(x), T, _dp(x_perm), _dp(counts),
                                      _dp(offsets), _dp(src), _dp(inv), chp))

    # -- a3 + a4
    def ef_expert_ffn_grouped(self, visit, layer, x_perm, counts_host, y_perm):
        ch = None if counts_host is None else _hp(np.ascontiguousarray(counts_host, dtype=np.int32))
        self._chk(self.lib.ef_expert_ffn_grouped(self.h, _stream(), visit, layer, _dp(x_perm), ch, _dp(y_perm)))

    def ef_expert_ffn_grouped_resident(self, x_perm, row_begin, rows, slots, y_perm):
        rb = np.ascontiguousarray(row_begin, dtype=np.int32)
        rw = np.ascontiguousarray(rows, dtype=np.int32)
        sl = np.ascontiguousarray(slots, dtype=np.int32)
        self._chk(self.lib.ef_expert_ffn_grouped_resident(self.h, _stream(), _dp(x_perm), len(rb), _hp(rb), _hp(rw),
                                                          _hp(sl), _dp(y_perm)))

    def ef_shared_ffn(self, layer, x, T, y_shared):
        self._chk(self.lib.ef_shared_ffn(self.h, _stream(), layer, _dp(x), T, _dp(y_shared)))

    # -- a5, a8
    def ef_combine(self, y_perm, inv, topk_w, T, residual, y_shared, out):
        self._chk(self.lib.ef_combine(self.h, _stream(), _dp(y_perm), _dp(inv), _dp(topk_w), T, _dp(residual),
                                      _dp(y_shared), _dp(out)))

    def ef_rmsnorm(self, x, T, eps, out):
        self._chk(self.lib.ef_rmsnorm(self.h, _stream(), _dp(x), T, eps, _dp(out)))

    # -- a6, a7
    def ef_cache_prefetch(self, visit_now, predicted):
        p = np.ascontiguousarray(predicted, dtype=np.uint8)
        if p.ndim == 1:
            p = p[None, :]
        self._chk(self.lib.ef_cache_prefetch(self.h, visit_now, _hp(p), p.shape[0]))

    def ef_cache_evict(self, layer, experts):
        e = np.ascontiguousarray(experts, dtype=np.int32)
        self._chk(self.lib.ef_cache_evict(self.h, layer, _hp(e), len(e)))

    # -- f1: token scheduler
    def ef_token_schedule(self, paths, c0, c1, max_iter, batch_of, perm, info, batch_paths=None):
        """paths: uint8 device tensor [N, L, E] or [N, L*E]; outputs: int32 device tensors [N], [N], [8] and
        optionally uint8 [2, L*E]."""
        N = paths.shape[0]
        LE = paths.numel() // max(1, N)
        self._chk(self.lib.ef_token_schedule(self.h, _stream(), _dp(paths), N, LE, c0, c1, max_iter, _dp(batch_of),
                                             _dp(perm), _dp(info), _dp(batch_paths)))

    def ef_reindex_rows(self, src, perm, dst):
        n = perm.shape[0]
        row_bytes = src.element_size() * (src.numel() // max(1, src.shape[0]))
        self._chk(self.lib.ef_reindex_rows(self.h, _stream(), _dp(src), _dp(perm), n, row_bytes, _dp(dst)))

    def ef_path_hamming(self, paths, dist_out):
        N = paths.shape[0]
        LE = paths.numel() // max(1, N)
        self._chk(self.lib.ef_path_hamming(self.h, _stream(), _dp(paths), N, LE, _dp(dist_out)))

    def ef_path_hamming_static(self, paths, dist_out):
        N = paths.shape[0]
        LE = paths.numel() // max(1, N)
        self._chk(self.lib.ef_path_hamming_static(self.h, _stream(), _dp(paths), N, LE, _dp(dist_out)))

    def ef_cache_get_stats(self) -> dict:
        st = CacheStats()
        self._chk(self.lib.ef_cache_get_stats(self.h, ctypes.byref(st)))
        return st.as_dict()

    def ef_cache_reset_stats(self):
        self._chk(self.lib.ef_cache_reset_stats(self.h))

    def ef_cache_snapshot(self) -> list[int]:
        a = np.empty(self.cfg.n_slots, dtype=np.int32)
        self._chk(self.lib.ef_cache_snapshot(self.h, _hp(a)))
        return a.tolist()

    def ef_cache_clear(self):
        self._chk(self.lib.ef_cache_clear(self.h))

    def ef_copy_busy_ms(self) -> float:
        ms = ctypes.c_float()
        self._chk(self.lib.ef_copy_busy_ms(self.h, ctypes.byref(ms)))
        return float(ms.value)

    def ef_sync(self):
        self._chk(self.lib.ef_sync(self.h))

    def ef_launch_count(self) -> int:
        return int(self.lib.ef_launch_count(self.h))

    def ef_set_option(self, key: int, value: int):
        self._chk(self.lib.ef_set_option(self.h, int(key), int(value)))

    POLICIES = {"plec": 0, "lru": 1, "layer_lru": 2}

    def ef_set_cache_policy(self, policy):
        self._chk(self.lib.ef_set_cache_policy(self.h, self.POLICIES.get(policy, policy)))

    # -- include/ef_diag.h (diag=True contexts only)
    def ef_diag_set_simt_ffn(self, on: bool):
        self._chk(self.lib.ef_diag_set_simt_ffn(self.h, 1 if on else 0))

    def ef_diag_tma_fill_gbs(self, region_bytes: int, iters: int = 2000) -> float:
        out = ctypes.c_double()
        self._chk(self.lib.ef_diag_tma_fill_gbs(self.h, int(region_bytes), int(iters), ctypes.byref(out)))
        return float(out.value)

    def ef_diag_pair_handoff_gbs(self, region_bytes: int, iters: int, n_ctas: int, mode: int) -> float:
        out = ctypes.c_double()
        self._chk(self.lib.ef_diag_pair_handoff_gbs(self.h, int(region_bytes), int(iters), int(n_ctas), int(mode), ctypes.byref(out)))
        return float(out.value)

    def ef_diag_kprof(self, which: int, n_sms: int = 148):
        out = np.zeros((n_sms, 5), np.int64)
        self._chk(self.lib.ef_diag_kprof(self.h, int(which), out.ctypes.data_as(ctypes.c_void_p)))
        return out

    def ef_set_kernel_timing(self, on: bool):
        self._chk(self.lib.ef_set_kernel_timing(self.h, 1 if on else 0))

    def ef_get_kernel_times(self, reset: bool = True) -> dict:
        kt = KernelTimes()
        self._chk(self.lib.ef_get_kernel_times(self.h, ctypes.byref(kt), 1 if reset else 0))
        return kt.as_dict()

    def ef_get_launch_log(self, reset: bool = True, max_records: int = 65536) -> list[dict]:
        buf = (LaunchRecord * max_records)()
        n = ctypes.c_int32()
        self._chk(self.lib.ef_get_launch_log(self.h, buf, max_records, ctypes.byref(n), 1 if reset else 0))
        return [{"which": int(r.which), "groups": int(r.groups), "rows": int(r.rows), "ms": float(r.ms)} for r in buf[:n.value]]
