"""CPU ORACLE for the ExpertFlow MoE expert layer -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA path and
never imports ``paper_2410_17954_b200``.

* ``moe_oracle.c``  -- layer math, the plain definition (Eq. 1-2).
* ``token_sched.py`` -- the Token Scheduler of PAPER.md §3.3, step by step (integers only).
* ``cache_sim.py``  -- the expert-cache policy, step by step, integers only (§8(c) O2;
  PAPER.md §3.2.1, §3.2.2, §4.1).
* this file        -- builds the C file with gcc for the host it runs on and wraps it with ctypes;
  ``layer_forward`` strings the stages together in the paper's order.

Pinned by tests/test_oracle_layer.py and tests/test_oracle_cache.py (``-m "not gpu"``).
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "moe_oracle.c")
_LIBS: dict[str, ctypes.CDLL] = {}


def _host_tag() -> str:
    """Key the build by source text + CPU flags: -march=native objects must not travel between hosts."""
    h = hashlib.sha1()
    with open(_SRC, "rb") as f:
        h.update(f.read())
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    h.update(line.encode())
                    break
    except OSError:
        pass
    return h.hexdigest()[:12]


def build(real: str = "double") -> str:
    """Compile moe_oracle.c (gcc -O3 -march=native -fopenmp) for this host; returns the .so path."""
    out_dir = os.path.join(_HERE, "_build")
    os.makedirs(out_dir, exist_ok=True)
    so = os.path.join(out_dir, f"libmoe_oracle_{real}_{_host_tag()}.so")
    if not os.path.exists(so):
        tmp = so + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=c11",
               f"-DORC_REAL={real}", _SRC, "-o", tmp, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, so)
    return so


def _lib(real: str = "double") -> ctypes.CDLL:
    if real not in _LIBS:
        lib = ctypes.CDLL(build(real))
        lib.orc_real_bytes.restype = ctypes.c_int
        lib.orc_num_threads.restype = ctypes.c_int
        assert lib.orc_real_bytes() == (8 if real == "double" else 4)
        _LIBS[real] = lib
    return _LIBS[real]


def num_threads() -> int:
    return int(_lib().orc_num_threads())


def _p(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _rdt(real):
    return np.float64 if real == "double" else np.float32


def _c(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


# ---------------------------------------------------------------------------------------------
# stage wrappers (argument marshalling only)
# ---------------------------------------------------------------------------------------------
def router_logits(x, wr, bias=None, real="double"):
    """l[t,e] = w_e.x_t + b_e  (Eq. 1).  x:[T,d] bf16 bits, wr:[E,d] bf16 bits,
    bias: None | fp32 [E] | fp32 [T,E]."""
    x = _c(x, np.uint16); wr = _c(wr, np.uint16)
    T, d = x.shape; E = wr.shape[0]
    stride = 0
    if bias is not None:
        bias = _c(bias, np.float32)
        stride = 0 if bias.ndim == 1 else E
        assert bias.shape[-1] == E
    out = np.empty((T, E), dtype=_rdt(real))
    _lib(real).orc_router_logits(_p(x), _p(wr), _p(bias), ctypes.c_int64(stride), T, d, E, _p(out))
    return out


def topk_gate(logits, k, renorm=1, real="double"):
    """Top-k (ties -> lower index, pick order) + gate weights (Eq. 1-2)."""
    logits = _c(logits, _rdt(real))
    T, E = logits.shape
    idx = np.empty((T, k), dtype=np.int32)
    w = np.empty((T, k), dtype=_rdt(real))
    _lib(real).orc_topk_gate(_p(logits), T, E, k, int(renorm), _p(idx), _p(w))
    return idx, w


def permute(idx, E):
    idx = _c(idx, np.int32)
    T, k = idx.shape
    counts = np.empty(E, dtype=np.int32); offsets = np.empty(E + 1, dtype=np.int32)
    src = np.empty(T * k, dtype=np.int32); inv = np.empty(T * k, dtype=np.int32)
    _lib().orc_permute(_p(idx), T, k, E, _p(counts), _p(offsets), _p(src), _p(inv))
    return counts, offsets, src, inv


def gather_rows(x, src, k):
    x = _c(x, np.uint16); src = _c(src, np.int32)
    R = src.shape[0]; d = x.shape[1]
    out = np.empty((R, d), dtype=np.uint16)
    _lib().orc_gather_rows(_p(x), _p(src), ctypes.c_int64(R), k, d, _p(out))
    return out


def expert_ffn(xrows, wg, wu, wd, want_h=False, real="double"):
    """One expert on M rows.  wu given: SwiGLU (wg, wu, wd).  wu None: the Switch-style non-gated ReLU FFN with
    W1 = wg, W2 = wd (R30).  Returns y [M,d] (and h [M,f] if want_h)."""
    xrows = _c(xrows, np.uint16); wg = _c(wg, np.uint16); wd = _c(wd, np.uint16)
    M, d = xrows.shape; f = wg.shape[0]
    assert wg.shape == (f, d) and wd.shape == (d, f)
    y = np.empty((M, d), dtype=_rdt(real))
    h = np.empty((M, f), dtype=_rdt(real)) if want_h else None
    if wu is None:
        _lib(real).orc_expert_ffn_relu(_p(xrows), ctypes.c_int64(M), d, f, _p(wg), _p(wd), _p(y), _p(h))
    else:
        wu = _c(wu, np.uint16)
        assert wu.shape == (f, d)
        _lib(real).orc_expert_ffn(_p(xrows), ctypes.c_int64(M), d, f, _p(wg), _p(wu), _p(wd), _p(y), _p(h))
    return (y, h) if want_h else y


def combine(y_perm, inv, w, k, res=None, y_shared=None, real="double"):
    y_perm = _c(y_perm, _rdt(real)); inv = _c(inv, np.int32); w = _c(w, _rdt(real))
    T = w.shape[0]; d = y_perm.shape[1]
    if res is not None:
        res = _c(res, np.uint16)
    if y_shared is not None:
        y_shared = _c(y_shared, _rdt(real))
    out = np.empty((T, d), dtype=_rdt(real))
    _lib(real).orc_combine(_p(y_perm), _p(inv), _p(w), T, k, d, _p(res), _p(y_shared), _p(out))
    return out


def rmsnorm(x, eps=1e-5, real="double"):
    x = _c(x, np.uint16)
    T, d = x.shape
    out = np.empty((T, d), dtype=_rdt(real))
    _lib(real).orc_rmsnorm(_p(x), T, d, ctypes.c_double(eps), _p(out))
    return out


def round_bf16(a, real="double"):
    a = _c(a, _rdt(real))
    out = np.empty(a.shape, dtype=np.uint16)
    _lib(real).orc_round_bf16(_p(a), ctypes.c_int64(a.size), _p(out))
    return out


# ---------------------------------------------------------------------------------------------
# the layer, in the paper's order
# ---------------------------------------------------------------------------------------------
@dataclass
class LayerResult:
    logits: np.ndarray
    idx: np.ndarray
    w: np.ndarray
    counts: np.ndarray
    offsets: np.ndarray
    src: np.ndarray
    inv: np.ndarray
    x_perm: np.ndarray | None
    y_perm: np.ndarray | None
    out: np.ndarray | None


def layer_forward(x, wr, bias, experts, k, renorm=1, shared=(), res=None, rows=None, real="double"):
    """One MoE layer visit.

    experts: callable e -> (wg, wu, wd) or a sequence; shared: sequence of (wg, wu, wd).
    rows: optional array of token ids -- compute the FFN / combine only for those tokens
    (sampled parity at full size); out then has len(rows) rows in that order.
    """
    get = experts if callable(experts) else (lambda e: experts[e])
    E = wr.shape[0]
    logits = router_logits(x, wr, bias, real)
    idx, w = topk_gate(logits, k, renorm, real)
    counts, offsets, src, inv = permute(idx, E)
    x_perm = gather_rows(x, src, k)
    d = x.shape[1]
    if rows is None:
        y_perm = np.zeros((x_perm.shape[0], d), dtype=_rdt(real))
        for e in range(E):
            if counts[e] == 0:
                continue
            wg, wu, wd = get(e)
            y_perm[offsets[e]:offsets[e + 1]] = expert_ffn(x_perm[offsets[e]:offsets[e + 1]], wg, wu, wd, real=real)
        y_shared = None
        for (wg, wu, wd) in shared:
            ys = expert_ffn(x, wg, wu, wd, real=real)
            y_shared = ys if y_shared is None else y_shared + ys
        out = combine(y_perm, inv, w, k, res, y_shared, real)
        return LayerResult(logits, idx, w, counts, offsets, src, inv, x_perm, y_perm, out)
    # sampled tokens: each (token, choice) pair is one FFN row
    rows = np.asarray(rows, dtype=np.int64)
    out = np.zeros((rows.shape[0], d), dtype=_rdt(real))
    by_expert: dict[int, list[tuple[int, int]]] = {}
    for i, t in enumerate(rows):
        for j in range(k):
            by_expert.setdefault(int(idx[t, j]), []).append((i, j))
    for e, lst in sorted(by_expert.items()):
        wg, wu, wd = get(e)
        xs = np.stack([x[rows[i]] for i, _ in lst])
        ys = expert_ffn(xs, wg, wu, wd, real=real)
        for (i, j), yrow in zip(lst, ys):
            out[i] += w[rows[i], j] * yrow
    for (wg, wu, wd) in shared:
        out += expert_ffn(x[rows], wg, wu, wd, real=real)
    if res is not None:
        from_res = (np.ascontiguousarray(res[rows], dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)
        out += from_res.astype(_rdt(real))
    return LayerResult(logits, idx, w, counts, offsets, src, inv, x_perm, None, out)
