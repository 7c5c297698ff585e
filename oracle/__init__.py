"""fp64 CPU oracle for the HYPIC linear-attention hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin numpy/ctypes front end of ``oracle/hypic_oracle.c`` (plain C, fp64, token by token; see that file's
header for the passages of PAPER.md each function follows).  Only ``tests/``, ``__graft_entry__.smoke()``
and the ``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.  It imports
nothing from ``paper_2607_01299_b200`` and the CUDA path imports nothing from here.

Conventions (reading A1, row convention): state ``S`` is ``dv x dk``, ``T`` is ``dk x dk``,
token step ``S <- S diag(alpha_t); S += beta_t (v_t - S k_t) k_t^T`` with ``alpha_t = exp(g_t)``;
``compose``: ``S <- S T_i + E_i``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

GATE_SCALAR = 0
GATE_CHANNEL = 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hypic_oracle.c")
_LIB = os.path.join(_HERE, "libhypic_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O3 -march=native -fopenmp).  Returns the path of the shared object."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-shared", "-fPIC", "-std=c99", _SRC, "-o", tmp, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        path = build()
        lib = ctypes.CDLL(path)
        i32, vp = ctypes.c_int, ctypes.c_void_p
        lib.hypic_oracle_num_threads.restype = i32
        lib.hypic_oracle_set_num_threads.argtypes = [i32]
        lib.hypic_oracle_segment_encode.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]
        lib.hypic_oracle_segment_encode.restype = i32
        lib.hypic_oracle_sequential.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp]
        lib.hypic_oracle_sequential.restype = i32
        lib.hypic_oracle_seam_window.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]
        lib.hypic_oracle_seam_window.restype = i32
        lib.hypic_oracle_diag_encode.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]
        lib.hypic_oracle_diag_encode.restype = i32
        lib.hypic_oracle_diag_sequential.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp]
        lib.hypic_oracle_diag_sequential.restype = i32
        lib.hypic_oracle_diag_compose.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp]
        lib.hypic_oracle_diag_compose.restype = i32
        lib.hypic_oracle_rope_compose.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, vp]
        lib.hypic_oracle_rope_compose.restype = i32
        lib.hypic_oracle_compose.argtypes = [vp, vp, vp, i32, vp, vp, i32, i32, i32, i32, i32, vp]
        lib.hypic_oracle_compose.restype = i32
        _lib = lib
    return _lib


def num_threads() -> int:
    """OpenMP threads the oracle uses (reported as ``cores`` by bench.py)."""
    return int(_load().hypic_oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().hypic_oracle_set_num_threads(int(n))


def _f32(x, shape=None):
    """Widen an input (numpy array, or anything with .float().numpy(), e.g. a CPU torch tensor holding bf16)
    to a C-contiguous float32 array.  bf16 -> fp32 and fp32 -> fp32 are exact."""
    if not isinstance(x, np.ndarray):
        x = x.detach().cpu().float().numpy()
    x = np.ascontiguousarray(x, dtype=np.float32)
    if shape is not None:
        assert x.shape == tuple(shape), (x.shape, shape)
    return x


def _i32(x):
    if not isinstance(x, np.ndarray):
        x = np.asarray(x.detach().cpu().numpy() if hasattr(x, "detach") else x)
    return np.ascontiguousarray(x, dtype=np.int32)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _check_inputs(k, v, g, beta, gate):
    k, v, g, beta = _f32(k), _f32(v), _f32(g), _f32(beta)
    ttot, H, dk = k.shape
    dv = v.shape[2]
    assert v.shape[:2] == (ttot, H)
    assert beta.shape == (ttot, H)
    assert g.shape == ((ttot, H) if gate == GATE_SCALAR else (ttot, H, dk)), (g.shape, gate)
    return k, v, g, beta, ttot, H, dk, dv


def segment_encode(k, v, g, beta, cu_seqlens, gate: int = GATE_SCALAR):
    """(E, T) per segment and head: E:[n_seg,H,dv,dk], T:[n_seg,H,dk,dk], float64.

    k:[Ttot,H,dk], v:[Ttot,H,dv], g:[Ttot,H] or [Ttot,H,dk] (log-decay, alpha=exp(g)), beta:[Ttot,H];
    cu_seqlens:int32[n_seg+1].  PAPER.md:120 (T_C), PAPER.md:126 (S_{C|0})."""
    k, v, g, beta, ttot, H, dk, dv = _check_inputs(k, v, g, beta, gate)
    cu = _i32(cu_seqlens)
    n_seg = cu.shape[0] - 1
    assert cu[0] == 0 and cu[-1] == ttot and np.all(np.diff(cu) >= 0)
    E = np.empty((n_seg, H, dv, dk), dtype=np.float64)
    T = np.empty((n_seg, H, dk, dk), dtype=np.float64)
    rc = _load().hypic_oracle_segment_encode(_ptr(k), _ptr(v), _ptr(g), _ptr(beta), _ptr(cu), n_seg, H, dk, dv,
                                             gate, _ptr(E), _ptr(T))
    if rc != 0:
        raise ValueError(f"hypic_oracle_segment_encode failed with code {rc}")
    return E, T


def sequential(S_in, k, v, g, beta, cu_tokens, gate: int = GATE_SCALAR):
    """Plain token recurrence from S_in over each request's tokens [cu_tokens[r], cu_tokens[r+1]).

    S_in:[R,H,dv,dk] float64 or None (zeros).  Returns S_out:[R,H,dv,dk] float64.  PAPER.md:84 (Eq. 2)."""
    k, v, g, beta, ttot, H, dk, dv = _check_inputs(k, v, g, beta, gate)
    cu = _i32(cu_tokens)
    R = cu.shape[0] - 1
    assert np.all(np.diff(cu) >= 0) and cu[0] >= 0 and cu[-1] <= ttot
    if S_in is not None:
        S_in = np.ascontiguousarray(S_in, dtype=np.float64)
        assert S_in.shape == (R, H, dv, dk)
    S_out = np.empty((R, H, dv, dk), dtype=np.float64)
    rc = _load().hypic_oracle_sequential(_ptr(S_in), _ptr(k), _ptr(v), _ptr(g), _ptr(beta), _ptr(cu), R, H, dk, dv,
                                         gate, _ptr(S_out))
    if rc != 0:
        raise ValueError(f"hypic_oracle_sequential failed with code {rc}")
    return S_out


def seam_window(S_in, q, k, v, g, beta, cu_tokens, gate: int = GATE_SCALAR):
    """Seam-window step: token recurrence from S_in over each request's window tokens with the
    per-token read-out o_t = S_t q_t (row convention).  q:[Ttot,H,dk].  Returns (S_out:[R,H,dv,dk],
    o:[Ttot,H,dv]) float64; rows of o for tokens outside every request are NaN."""
    k, v, g, beta, ttot, H, dk, dv = _check_inputs(k, v, g, beta, gate)
    q = _f32(q)
    assert q.shape == (ttot, H, dk)
    cu = _i32(cu_tokens)
    R = cu.shape[0] - 1
    assert np.all(np.diff(cu) >= 0) and cu[0] >= 0 and cu[-1] <= ttot
    if S_in is not None:
        S_in = np.ascontiguousarray(S_in, dtype=np.float64)
        assert S_in.shape == (R, H, dv, dk)
    S_out = np.empty((R, H, dv, dk), dtype=np.float64)
    o = np.full((ttot, H, dv), np.nan, dtype=np.float64)
    rc = _load().hypic_oracle_seam_window(_ptr(S_in), _ptr(q), _ptr(k), _ptr(v), _ptr(g), _ptr(beta), _ptr(cu), R, H,
                                          dk, dv, gate, _ptr(S_out), _ptr(o))
    if rc != 0:
        raise ValueError(f"hypic_oracle_seam_window failed with code {rc}")
    return S_out, o


def _check_diag_inputs(k, v, g, gate):
    k, v, g = _f32(k), _f32(v), _f32(g)
    ttot, H, dk = k.shape
    dv = v.shape[2]
    assert v.shape[:2] == (ttot, H)
    assert g.shape == ((ttot, H) if gate == GATE_SCALAR else (ttot, H, dk)), (g.shape, gate)
    return k, v, g, ttot, H, dk, dv


def diag_encode(k, v, g, cu_seqlens, gate: int = GATE_SCALAR):
    """Scalar / diagonal families: (E:[n_seg,H,dv,dk], tvec:[n_seg,H] or [n_seg,H,dk])
    float64 for the recurrence S <- S diag(exp(g_t)) + v_t k_t^T from S = 0; tvec = prod_t exp(g_t)."""
    k, v, g, ttot, H, dk, dv = _check_diag_inputs(k, v, g, gate)
    cu = _i32(cu_seqlens)
    n_seg = cu.shape[0] - 1
    assert cu[0] == 0 and cu[-1] == ttot and np.all(np.diff(cu) >= 0)
    E = np.empty((n_seg, H, dv, dk), dtype=np.float64)
    tvec = np.empty((n_seg, H) if gate == GATE_SCALAR else (n_seg, H, dk), dtype=np.float64)
    rc = _load().hypic_oracle_diag_encode(_ptr(k), _ptr(v), _ptr(g), _ptr(cu), n_seg, H, dk, dv, gate, _ptr(E),
                                          _ptr(tvec))
    if rc != 0:
        raise ValueError(f"hypic_oracle_diag_encode failed with code {rc}")
    return E, tvec


def diag_sequential(S_in, k, v, g, cu_tokens, gate: int = GATE_SCALAR):
    """The same recurrence from S_in (None = zeros) over each request's tokens: S_out:[R,H,dv,dk] float64."""
    k, v, g, ttot, H, dk, dv = _check_diag_inputs(k, v, g, gate)
    cu = _i32(cu_tokens)
    R = cu.shape[0] - 1
    assert np.all(np.diff(cu) >= 0) and cu[0] >= 0 and cu[-1] <= ttot
    if S_in is not None:
        S_in = np.ascontiguousarray(S_in, dtype=np.float64)
        assert S_in.shape == (R, H, dv, dk)
    S_out = np.empty((R, H, dv, dk), dtype=np.float64)
    rc = _load().hypic_oracle_diag_sequential(_ptr(S_in), _ptr(k), _ptr(v), _ptr(g), _ptr(cu), R, H, dk, dv, gate,
                                              _ptr(S_out))
    if rc != 0:
        raise ValueError(f"hypic_oracle_diag_sequential failed with code {rc}")
    return S_out


def diag_compose(S_in, E_pool, t_pool, seg_ids, cu_segs):
    """S <- S diag(t_i) + E_i over each request's ordered ids (Eq. 6 with Table 3's compressed T_C).
    t_pool:[P,H] (scalar) or [P,H,dk]."""
    E_pool = np.ascontiguousarray(E_pool, dtype=np.float64)
    t_pool = np.ascontiguousarray(t_pool, dtype=np.float64)
    P, H, dv, dk = E_pool.shape
    gate = GATE_SCALAR if t_pool.ndim == 2 else GATE_CHANNEL
    assert t_pool.shape == ((P, H) if gate == GATE_SCALAR else (P, H, dk))
    ids, cu = _i32(seg_ids), _i32(cu_segs)
    R = cu.shape[0] - 1
    assert cu[0] == 0 and cu[-1] == ids.shape[0] and np.all(np.diff(cu) >= 0)
    assert ids.size == 0 or (ids.min() >= 0 and ids.max() < P)
    if S_in is not None:
        S_in = np.ascontiguousarray(S_in, dtype=np.float64)
        assert S_in.shape == (R, H, dv, dk)
    S_out = np.empty((R, H, dv, dk), dtype=np.float64)
    rc = _load().hypic_oracle_diag_compose(_ptr(S_in), _ptr(E_pool), _ptr(t_pool), _ptr(ids), _ptr(cu), R, H, dk, dv,
                                           gate, _ptr(S_out))
    if rc != 0:
        raise ValueError(f"hypic_oracle_diag_compose failed with code {rc}")
    return S_out


def rope_compose(S_in, E_pool, t_pool, seg_ids, cu_segs, pos, inv_freq):
    """Scalar family with RoPE inside the layer: S <- t_i S + E_i R(p_i)^T, every row of the zero-start end-state
    re-rotated like a key to the segment's global start position p_i (Eq. 7).
    t_pool:[P,H]; pos:int32[len(seg_ids)]; inv_freq:[dk/2] (pair = columns c, c + dk/2)."""
    E_pool = np.ascontiguousarray(E_pool, dtype=np.float64)
    t_pool = np.ascontiguousarray(t_pool, dtype=np.float64)
    inv_freq = np.ascontiguousarray(inv_freq, dtype=np.float64)
    P, H, dv, dk = E_pool.shape
    assert t_pool.shape == (P, H) and dk % 2 == 0 and inv_freq.shape == (dk // 2,)
    ids, cu, pos = _i32(seg_ids), _i32(cu_segs), _i32(pos)
    R = cu.shape[0] - 1
    assert cu[0] == 0 and cu[-1] == ids.shape[0] and np.all(np.diff(cu) >= 0) and pos.shape == ids.shape
    assert ids.size == 0 or (ids.min() >= 0 and ids.max() < P)
    if S_in is not None:
        S_in = np.ascontiguousarray(S_in, dtype=np.float64)
        assert S_in.shape == (R, H, dv, dk)
    S_out = np.empty((R, H, dv, dk), dtype=np.float64)
    rc = _load().hypic_oracle_rope_compose(_ptr(S_in), _ptr(E_pool), _ptr(t_pool), _ptr(ids), _ptr(cu), _ptr(pos),
                                           _ptr(inv_freq), R, H, dk, dv, _ptr(S_out))
    if rc != 0:
        raise ValueError(f"hypic_oracle_rope_compose failed with code {rc}")
    return S_out


def compose(S_in, E_pool, T_pool, seg_ids, cu_segs):
    """S_out[r,h] = fold of ``S <- S T_i + E_i`` over the request's ordered ids.  PAPER.md:182 (Eq. 6).

    E_pool:[P,H,dv,dk], T_pool:[P,H,dk,dk] -- float32 pools are read as float32 (exactly widened), anything
    else as float64.  S_in:[R,H,dv,dk] or None.  Returns float64 [R,H,dv,dk]."""
    if not isinstance(E_pool, np.ndarray):
        E_pool = E_pool.detach().cpu().numpy()
    if not isinstance(T_pool, np.ndarray):
        T_pool = T_pool.detach().cpu().numpy()
    f32 = E_pool.dtype == np.float32 and T_pool.dtype == np.float32
    dt = np.float32 if f32 else np.float64
    E_pool = np.ascontiguousarray(E_pool, dtype=dt)
    T_pool = np.ascontiguousarray(T_pool, dtype=dt)
    P, H, dv, dk = E_pool.shape
    assert T_pool.shape == (P, H, dk, dk)
    ids, cu = _i32(seg_ids), _i32(cu_segs)
    R = cu.shape[0] - 1
    assert cu[0] == 0 and cu[-1] == ids.shape[0] and np.all(np.diff(cu) >= 0)
    if S_in is not None:
        if not isinstance(S_in, np.ndarray):
            S_in = S_in.detach().cpu().numpy()
        S_in = np.ascontiguousarray(S_in, dtype=np.float64)
        assert S_in.shape == (R, H, dv, dk)
    S_out = np.empty((R, H, dv, dk), dtype=np.float64)
    rc = _load().hypic_oracle_compose(_ptr(S_in), _ptr(E_pool), _ptr(T_pool), int(f32), _ptr(ids), _ptr(cu), R, P, H,
                                      dk, dv, _ptr(S_out))
    if rc != 0:
        raise ValueError(f"hypic_oracle_compose failed with code {rc}")
    return S_out


def rel_fro(x, ref) -> float:
    """||x - ref||_F / ||ref||_F over the whole array (the error metric of BASELINE.json:north_star)."""
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.linalg.norm(ref.ravel())
    num = np.linalg.norm((x - ref).ravel())
    return float(num / den) if den > 0 else float(num)
