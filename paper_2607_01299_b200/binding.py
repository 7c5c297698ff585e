"""Thin Python binding of libhypic.so (include/hypic.h): argument marshalling only.

Same names as the C ABI.  Every step of the path runs in the CUDA kernels behind the library; torch is used
for device memory and streams.  There is NO CPU fallback: if the shared library is missing or a tensor is not
on a CUDA device, the call raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import torch

HYPIC_OK = 0
HYPIC_ERR_INVALID_ARG = 1
HYPIC_ERR_UNSUPPORTED = 2
HYPIC_ERR_WORKSPACE = 3
HYPIC_ERR_CUDA = 4
HYPIC_ERR_STATIC_SCRATCH = 5
HYPIC_DT_F32 = 0
HYPIC_DT_BF16 = 1
HYPIC_GATE_SCALAR = 0
HYPIC_GATE_CHANNEL = 1
HYPIC_IMPL_AUTO = 0
HYPIC_IMPL_SIMT = 1
HYPIC_IMPL_TENSOR = 2

EXPORTS = (
    "hypic_set_impl", "hypic_get_impl", "hypic_segment_encode_workspace", "hypic_segment_encode", "hypic_compose",
    "hypic_status_string", "hypic_version", "hypic_last_launch_count", "hypic_last_cuda_error", "hypic_encode_impl_for",
    "hypic_compose_impl_for", "hypic_debug_timeout_count", "hypic_envelope_violation_count", "hypic_compose_f16",
    "hypic_tuple_pack_f16", "hypic_seam_window", "hypic_diag_encode", "hypic_diag_compose",
    "hypic_diag_encode_impl_for", "hypic_diag_compose_f16", "hypic_forward_encode", "hypic_rope_compose_workspace",
    "hypic_rope_compose", "hypic_rope_compose_f16", "hypic_static_scratch_bytes", "hypic_segment_encode_static",
)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhypic.so")
_lib = None


class HypicError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        extra = ""
        if self.status == HYPIC_ERR_CUDA and _lib is not None:
            extra = f", cudaError {int(_lib.hypic_last_cuda_error())}"
        super().__init__(f"{where} failed: status {status} ({hypic_status_string(status)}{extra})")


def load_library() -> ctypes.CDLL:
    """dlopen libhypic.so (built by ``python -m paper_2607_01299_b200.build``) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2607_01299_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    i32, vp, sz = ctypes.c_int32, ctypes.c_void_p, ctypes.c_size_t
    lib.hypic_set_impl.argtypes = [ctypes.c_int]
    lib.hypic_set_impl.restype = ctypes.c_int
    lib.hypic_get_impl.argtypes = []
    lib.hypic_get_impl.restype = ctypes.c_int
    lib.hypic_segment_encode_workspace.argtypes = [i32, i32, i32, i32, i32, ctypes.c_int, ctypes.c_int]
    lib.hypic_segment_encode_workspace.restype = sz
    lib.hypic_segment_encode.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, ctypes.c_int, ctypes.c_int, vp,
                                         vp, vp, sz, vp]
    lib.hypic_segment_encode.restype = ctypes.c_int
    lib.hypic_static_scratch_bytes.argtypes = []
    lib.hypic_static_scratch_bytes.restype = sz
    lib.hypic_segment_encode_static.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, ctypes.c_int, ctypes.c_int,
                                                vp, vp, vp]
    lib.hypic_segment_encode_static.restype = ctypes.c_int
    lib.hypic_compose.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp, vp]
    lib.hypic_compose.restype = ctypes.c_int
    lib.hypic_compose_f16.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp, vp]
    lib.hypic_compose_f16.restype = ctypes.c_int
    lib.hypic_tuple_pack_f16.argtypes = [vp, vp, sz, vp]
    lib.hypic_tuple_pack_f16.restype = ctypes.c_int
    lib.hypic_seam_window.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, ctypes.c_int, ctypes.c_int, vp,
                                      vp, vp, vp]
    lib.hypic_seam_window.restype = ctypes.c_int
    lib.hypic_diag_encode.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, ctypes.c_int, ctypes.c_int, vp, vp, vp]
    lib.hypic_diag_encode.restype = ctypes.c_int
    lib.hypic_diag_compose.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, ctypes.c_int, vp, vp]
    lib.hypic_diag_compose.restype = ctypes.c_int
    lib.hypic_forward_encode.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, ctypes.c_int, ctypes.c_int, vp,
                                         vp, vp, vp]
    lib.hypic_forward_encode.restype = ctypes.c_int
    lib.hypic_diag_compose_f16.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, ctypes.c_int, vp, vp]
    lib.hypic_diag_compose_f16.restype = ctypes.c_int
    lib.hypic_rope_compose_workspace.argtypes = [i32, i32]
    lib.hypic_rope_compose_workspace.restype = sz
    lib.hypic_rope_compose.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp, vp, sz, vp]
    lib.hypic_rope_compose.restype = ctypes.c_int
    lib.hypic_rope_compose_f16.argtypes = list(lib.hypic_rope_compose.argtypes)
    lib.hypic_rope_compose_f16.restype = ctypes.c_int
    lib.hypic_diag_encode_impl_for.argtypes = [i32, i32, i32, ctypes.c_int, ctypes.c_int]
    lib.hypic_diag_encode_impl_for.restype = ctypes.c_int
    lib.hypic_status_string.argtypes = [ctypes.c_int]
    lib.hypic_status_string.restype = ctypes.c_char_p
    lib.hypic_version.argtypes = []
    lib.hypic_version.restype = ctypes.c_int
    lib.hypic_last_launch_count.argtypes = []
    lib.hypic_last_launch_count.restype = ctypes.c_int
    lib.hypic_last_cuda_error.argtypes = []
    lib.hypic_last_cuda_error.restype = ctypes.c_int
    lib.hypic_encode_impl_for.argtypes = [i32, i32, i32, ctypes.c_int, ctypes.c_int]
    lib.hypic_encode_impl_for.restype = ctypes.c_int
    lib.hypic_compose_impl_for.argtypes = [i32, i32, i32]
    lib.hypic_compose_impl_for.restype = ctypes.c_int
    lib.hypic_debug_timeout_count.argtypes = []
    lib.hypic_debug_timeout_count.restype = ctypes.c_uint
    lib.hypic_envelope_violation_count.argtypes = []
    lib.hypic_envelope_violation_count.restype = ctypes.c_uint
    _lib = lib
    return lib


def hypic_status_string(status: int) -> str:
    return load_library().hypic_status_string(int(status)).decode()


def hypic_version() -> int:
    return int(load_library().hypic_version())


def hypic_set_impl(impl: int) -> None:
    rc = load_library().hypic_set_impl(int(impl))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_set_impl")


def hypic_get_impl() -> int:
    return int(load_library().hypic_get_impl())


def hypic_encode_impl_for(H: int, dk: int, dv: int, kv_dtype: int, gate: int) -> int:
    return int(load_library().hypic_encode_impl_for(H, dk, dv, kv_dtype, gate))


def hypic_diag_encode_impl_for(H: int, dk: int, dv: int, kv_dtype: int, gate: int) -> int:
    return int(load_library().hypic_diag_encode_impl_for(H, dk, dv, kv_dtype, gate))


def hypic_compose_impl_for(H: int, dk: int, dv: int) -> int:
    return int(load_library().hypic_compose_impl_for(H, dk, dv))


def hypic_envelope_violation_count() -> int:
    return int(load_library().hypic_envelope_violation_count())


def hypic_debug_timeout_count() -> int:
    return int(load_library().hypic_debug_timeout_count())


def hypic_last_launch_count() -> int:
    return int(load_library().hypic_last_launch_count())


def _dev_ptr(t: Optional[torch.Tensor], name: str, dtype=None) -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"{name} must be {dtype}, got {t.dtype}")
    return t.data_ptr() if t.numel() > 0 else None


def _stream_handle(stream: Optional[torch.cuda.Stream]) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def hypic_segment_encode_workspace(n_seg: int, t_total: int, H: int, dk: int, dv: int, kv_dtype: int,
                                   gate: int) -> int:
    return int(load_library().hypic_segment_encode_workspace(n_seg, t_total, H, dk, dv, kv_dtype, gate))


def hypic_segment_encode(k: torch.Tensor, v: torch.Tensor, g: torch.Tensor, beta: torch.Tensor,
                         cu_seqlens: torch.Tensor, gate: int = HYPIC_GATE_SCALAR, *,
                         E: Optional[torch.Tensor] = None, T: Optional[torch.Tensor] = None,
                         workspace: Optional[torch.Tensor] = None,
                         stream: Optional[torch.cuda.Stream] = None) -> Tuple[torch.Tensor, torch.Tensor]:
    """E:[n_seg,H,dv,dk], T:[n_seg,H,dk,dk] fp32 for packed k:[Ttot,H,dk], v:[Ttot,H,dv] (bf16 or fp32),
    g:[Ttot,H] or [Ttot,H,dk] fp32, beta:[Ttot,H] fp32, cu_seqlens:int32[n_seg+1] (device)."""
    lib = load_library()
    for name, t in (("k", k), ("v", v), ("g", g), ("beta", beta), ("cu_seqlens", cu_seqlens)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if k.dim() != 3 or v.dim() != 3 or k.shape[:2] != v.shape[:2] or k.dtype != v.dtype:
        raise ValueError("k:[Ttot,H,dk] and v:[Ttot,H,dv] must agree in Ttot, H and dtype")
    t_total, H, dk = (int(x) for x in k.shape)
    dv = int(v.shape[2])
    if k.dtype == torch.bfloat16:
        kv_dtype = HYPIC_DT_BF16
    elif k.dtype == torch.float32:
        kv_dtype = HYPIC_DT_F32
    else:
        raise ValueError(f"k/v must be bf16 or fp32, got {k.dtype}")
    want_g = (t_total, H) if gate == HYPIC_GATE_SCALAR else (t_total, H, dk)
    if tuple(g.shape) != want_g or tuple(beta.shape) != (t_total, H):
        raise ValueError(f"g must be {want_g} and beta {(t_total, H)}; got {tuple(g.shape)}, {tuple(beta.shape)}")
    n_seg = int(cu_seqlens.numel()) - 1
    if n_seg < 0:
        raise ValueError("cu_seqlens must have n_seg+1 >= 1 entries")
    dev = k.device
    if E is None:
        E = torch.empty((n_seg, H, dv, dk), dtype=torch.float32, device=dev)
    if T is None:
        T = torch.empty((n_seg, H, dk, dk), dtype=torch.float32, device=dev)
    if tuple(E.shape) != (n_seg, H, dv, dk) or tuple(T.shape) != (n_seg, H, dk, dk):
        raise ValueError("E / T have the wrong shape")
    need = int(lib.hypic_segment_encode_workspace(n_seg, t_total, H, dk, dv, kv_dtype, gate))
    if need > 0 and (workspace is None or workspace.numel() * workspace.element_size() < need):
        workspace = torch.empty(need, dtype=torch.uint8, device=dev)
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    with torch.cuda.device(dev):
        rc = lib.hypic_segment_encode(
            _dev_ptr(k, "k"), _dev_ptr(v, "v"), _dev_ptr(g, "g", torch.float32), _dev_ptr(beta, "beta", torch.float32),
            _dev_ptr(cu_seqlens, "cu_seqlens", torch.int32), n_seg, t_total, H, dk, dv, kv_dtype, int(gate),
            _dev_ptr(E, "E", torch.float32), _dev_ptr(T, "T", torch.float32), _dev_ptr(workspace, "workspace"),
            ws_bytes, _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_segment_encode")
    return E, T


def hypic_static_scratch_bytes() -> int:
    return int(load_library().hypic_static_scratch_bytes())


def hypic_segment_encode_static(k: torch.Tensor, v: torch.Tensor, g: torch.Tensor, beta: torch.Tensor,
                                cu_seqlens: torch.Tensor, gate: int, E: torch.Tensor, T: torch.Tensor, *,
                                stream: Optional[torch.cuda.Stream] = None) -> Tuple[torch.Tensor, torch.Tensor]:
    """hypic_segment_encode without a workspace and without any allocation: the scratch is a 4 MiB static device array
    inside the library (include/hypic.h).  E:[n_seg,H,dv,dk] and T:[n_seg,H,dk,dk] fp32 are the CALLER's (this wrapper
    allocates nothing either); raises HypicError(HYPIC_ERR_STATIC_SCRATCH) when the problem does not fit.  Calls that
    overlap on the GPU race on the array."""
    lib = load_library()
    for name, t in (("k", k), ("v", v), ("g", g), ("beta", beta), ("cu_seqlens", cu_seqlens), ("E", E), ("T", T)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if k.dim() != 3 or v.dim() != 3 or k.shape[:2] != v.shape[:2] or k.dtype != v.dtype:
        raise ValueError("k:[Ttot,H,dk] and v:[Ttot,H,dv] must agree in Ttot, H and dtype")
    t_total, H, dk = (int(x) for x in k.shape)
    dv = int(v.shape[2])
    if k.dtype not in (torch.bfloat16, torch.float32):
        raise ValueError(f"k/v must be bf16 or fp32, got {k.dtype}")
    kv_dtype = HYPIC_DT_BF16 if k.dtype == torch.bfloat16 else HYPIC_DT_F32
    want_g = (t_total, H) if gate == HYPIC_GATE_SCALAR else (t_total, H, dk)
    if tuple(g.shape) != want_g or tuple(beta.shape) != (t_total, H):
        raise ValueError(f"g must be {want_g} and beta {(t_total, H)}; got {tuple(g.shape)}, {tuple(beta.shape)}")
    n_seg = int(cu_seqlens.numel()) - 1
    if n_seg < 0 or tuple(E.shape) != (n_seg, H, dv, dk) or tuple(T.shape) != (n_seg, H, dk, dk):
        raise ValueError("cu_seqlens / E / T have the wrong shape")
    with torch.cuda.device(k.device):
        rc = lib.hypic_segment_encode_static(
            _dev_ptr(k, "k"), _dev_ptr(v, "v"), _dev_ptr(g, "g", torch.float32), _dev_ptr(beta, "beta", torch.float32),
            _dev_ptr(cu_seqlens, "cu_seqlens", torch.int32), n_seg, t_total, H, dk, dv, kv_dtype, int(gate),
            _dev_ptr(E, "E", torch.float32), _dev_ptr(T, "T", torch.float32), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_segment_encode_static")
    return E, T


def hypic_compose(S_in: Optional[torch.Tensor], E_pool: torch.Tensor, T_pool: torch.Tensor, seg_ids: torch.Tensor,
                  cu_segs: torch.Tensor, *, total_steps: Optional[int] = None, S_out: Optional[torch.Tensor] = None,
                  stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """S_out[r,h] = fold of S <- S T_i + E_i over seg_ids[cu_segs[r]:cu_segs[r+1]] from S_in[r,h] (None = 0)."""
    lib = load_library()
    for name, t in (("E_pool", E_pool), ("T_pool", T_pool), ("seg_ids", seg_ids), ("cu_segs", cu_segs)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if E_pool.dim() != 4 or T_pool.dim() != 4:
        raise ValueError("E_pool:[P,H,dv,dk], T_pool:[P,H,dk,dk]")
    P, H, dv, dk = (int(x) for x in E_pool.shape)
    if tuple(T_pool.shape) != (P, H, dk, dk):
        raise ValueError("T_pool must be [P,H,dk,dk]")
    R = int(cu_segs.numel()) - 1
    if R < 0:
        raise ValueError("cu_segs must have R+1 >= 1 entries")
    if total_steps is None:
        total_steps = int(seg_ids.numel())  # shape metadata, no device sync
    if S_in is not None and tuple(S_in.shape) != (R, H, dv, dk):
        raise ValueError("S_in must be [R,H,dv,dk]")
    if S_out is None:
        S_out = torch.empty((R, H, dv, dk), dtype=torch.float32, device=E_pool.device)
    if tuple(S_out.shape) != (R, H, dv, dk):
        raise ValueError("S_out must be [R,H,dv,dk]")
    with torch.cuda.device(E_pool.device):
        rc = lib.hypic_compose(
            _dev_ptr(S_in, "S_in", torch.float32), _dev_ptr(E_pool, "E_pool", torch.float32),
            _dev_ptr(T_pool, "T_pool", torch.float32), _dev_ptr(seg_ids, "seg_ids", torch.int32),
            _dev_ptr(cu_segs, "cu_segs", torch.int32), R, P, int(total_steps), H, dk, dv,
            _dev_ptr(S_out, "S_out", torch.float32), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_compose")
    return S_out


def hypic_compose_f16(S_in: Optional[torch.Tensor], E_pool: torch.Tensor, T_pool: torch.Tensor, seg_ids: torch.Tensor,
                      cu_segs: torch.Tensor, *, total_steps: Optional[int] = None,
                      S_out: Optional[torch.Tensor] = None,
                      stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """hypic_compose over fp16-stored pools (E_pool, T_pool: torch.float16); S_in / S_out stay fp32."""
    lib = load_library()
    for name, t in (("E_pool", E_pool), ("T_pool", T_pool), ("seg_ids", seg_ids), ("cu_segs", cu_segs)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if E_pool.dim() != 4 or T_pool.dim() != 4:
        raise ValueError("E_pool:[P,H,dv,dk], T_pool:[P,H,dk,dk]")
    P, H, dv, dk = (int(x) for x in E_pool.shape)
    if tuple(T_pool.shape) != (P, H, dk, dk):
        raise ValueError("T_pool must be [P,H,dk,dk]")
    R = int(cu_segs.numel()) - 1
    if R < 0:
        raise ValueError("cu_segs must have R+1 >= 1 entries")
    if total_steps is None:
        total_steps = int(seg_ids.numel())  # shape metadata, no device sync
    if S_in is not None and tuple(S_in.shape) != (R, H, dv, dk):
        raise ValueError("S_in must be [R,H,dv,dk]")
    if S_out is None:
        S_out = torch.empty((R, H, dv, dk), dtype=torch.float32, device=E_pool.device)
    if tuple(S_out.shape) != (R, H, dv, dk):
        raise ValueError("S_out must be [R,H,dv,dk]")
    with torch.cuda.device(E_pool.device):
        rc = lib.hypic_compose_f16(
            _dev_ptr(S_in, "S_in", torch.float32), _dev_ptr(E_pool, "E_pool", torch.float16),
            _dev_ptr(T_pool, "T_pool", torch.float16), _dev_ptr(seg_ids, "seg_ids", torch.int32),
            _dev_ptr(cu_segs, "cu_segs", torch.int32), R, P, int(total_steps), H, dk, dv,
            _dev_ptr(S_out, "S_out", torch.float32), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_compose_f16")
    return S_out


def hypic_tuple_pack_f16(src: torch.Tensor, dst: Optional[torch.Tensor] = None,
                         stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """dst = fp16(src), round to nearest even: packs fp32 E / T tensors into the fp16 pools of hypic_compose_f16."""
    lib = load_library()
    if not src.is_cuda:
        raise ValueError("src must be a CUDA tensor (no CPU fallback)")
    if dst is None:
        dst = torch.empty(src.shape, dtype=torch.float16, device=src.device)
    if dst.numel() != src.numel():
        raise ValueError("dst must have as many elements as src")
    with torch.cuda.device(src.device):
        rc = lib.hypic_tuple_pack_f16(_dev_ptr(src, "src", torch.float32), _dev_ptr(dst, "dst", torch.float16),
                                      int(src.numel()), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_tuple_pack_f16")
    return dst


def hypic_seam_window(S_in: Optional[torch.Tensor], q: torch.Tensor, k: torch.Tensor, v: torch.Tensor, g: torch.Tensor,
                      beta: torch.Tensor, cu_tokens: torch.Tensor, gate: int = HYPIC_GATE_SCALAR, *,
                      S_out: Optional[torch.Tensor] = None, o: Optional[torch.Tensor] = None,
                      stream: Optional[torch.cuda.Stream] = None) -> Tuple[torch.Tensor, torch.Tensor]:
    """Seam-window step: token recurrence over each request's window [cu_tokens[r], cu_tokens[r+1]) from S_in[r]
    (None = 0) with per-token read-out o[t,h] = S_t q_t.  Returns (S_out:[R,H,dv,dk], o:[Ttot,H,dv]) fp32; rows of o
    for tokens outside every window are left as they were (zeros when o is allocated here)."""
    lib = load_library()
    for name, t in (("q", q), ("k", k), ("v", v), ("g", g), ("beta", beta), ("cu_tokens", cu_tokens)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if k.dim() != 3 or v.dim() != 3 or k.shape[:2] != v.shape[:2] or k.dtype != v.dtype:
        raise ValueError("k:[Ttot,H,dk] and v:[Ttot,H,dv] must agree in Ttot, H and dtype")
    if q.shape != k.shape or q.dtype != k.dtype:
        raise ValueError("q must have k's shape and dtype")
    t_total, H, dk = (int(x) for x in k.shape)
    dv = int(v.shape[2])
    if k.dtype == torch.bfloat16:
        kv_dtype = HYPIC_DT_BF16
    elif k.dtype == torch.float32:
        kv_dtype = HYPIC_DT_F32
    else:
        raise ValueError(f"q/k/v must be bf16 or fp32, got {k.dtype}")
    want_g = (t_total, H) if gate == HYPIC_GATE_SCALAR else (t_total, H, dk)
    if tuple(g.shape) != want_g or tuple(beta.shape) != (t_total, H):
        raise ValueError(f"g must be {want_g} and beta {(t_total, H)}; got {tuple(g.shape)}, {tuple(beta.shape)}")
    R = int(cu_tokens.numel()) - 1
    if R < 0:
        raise ValueError("cu_tokens must have R+1 >= 1 entries")
    dev = k.device
    if S_in is not None and tuple(S_in.shape) != (R, H, dv, dk):
        raise ValueError("S_in must be [R,H,dv,dk]")
    if S_out is None:
        S_out = torch.empty((R, H, dv, dk), dtype=torch.float32, device=dev)
    if o is None:
        o = torch.zeros((t_total, H, dv), dtype=torch.float32, device=dev)
    if tuple(S_out.shape) != (R, H, dv, dk) or tuple(o.shape) != (t_total, H, dv):
        raise ValueError("S_out / o have the wrong shape")
    with torch.cuda.device(dev):
        rc = lib.hypic_seam_window(
            _dev_ptr(q, "q"), _dev_ptr(k, "k"), _dev_ptr(v, "v"), _dev_ptr(g, "g", torch.float32),
            _dev_ptr(beta, "beta", torch.float32), _dev_ptr(cu_tokens, "cu_tokens", torch.int32), R, t_total, H, dk,
            dv, kv_dtype, int(gate), _dev_ptr(S_in, "S_in", torch.float32), _dev_ptr(S_out, "S_out", torch.float32),
            _dev_ptr(o, "o", torch.float32), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_seam_window")
    return S_out, o


def hypic_diag_encode(k: torch.Tensor, v: torch.Tensor, g: torch.Tensor, cu_seqlens: torch.Tensor,
                      gate: int = HYPIC_GATE_SCALAR, *, E: Optional[torch.Tensor] = None,
                      tvec: Optional[torch.Tensor] = None,
                      stream: Optional[torch.cuda.Stream] = None) -> Tuple[torch.Tensor, torch.Tensor]:
    """Scalar / diagonal families: E:[n_seg,H,dv,dk] fp32 and tvec:[n_seg,H] (scalar gate) or [n_seg,H,dk] fp32 for
    the recurrence S <- S diag(exp(g_t)) + v_t k_t^T over each segment from S = 0."""
    lib = load_library()
    for name, t in (("k", k), ("v", v), ("g", g), ("cu_seqlens", cu_seqlens)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if k.dim() != 3 or v.dim() != 3 or k.shape[:2] != v.shape[:2] or k.dtype != v.dtype:
        raise ValueError("k:[Ttot,H,dk] and v:[Ttot,H,dv] must agree in Ttot, H and dtype")
    t_total, H, dk = (int(x) for x in k.shape)
    dv = int(v.shape[2])
    if k.dtype == torch.bfloat16:
        kv_dtype = HYPIC_DT_BF16
    elif k.dtype == torch.float32:
        kv_dtype = HYPIC_DT_F32
    else:
        raise ValueError(f"k/v must be bf16 or fp32, got {k.dtype}")
    want_g = (t_total, H) if gate == HYPIC_GATE_SCALAR else (t_total, H, dk)
    if tuple(g.shape) != want_g:
        raise ValueError(f"g must be {want_g}; got {tuple(g.shape)}")
    n_seg = int(cu_seqlens.numel()) - 1
    if n_seg < 0:
        raise ValueError("cu_seqlens must have n_seg+1 >= 1 entries")
    dev = k.device
    t_shape = (n_seg, H) if gate == HYPIC_GATE_SCALAR else (n_seg, H, dk)
    if E is None:
        E = torch.empty((n_seg, H, dv, dk), dtype=torch.float32, device=dev)
    if tvec is None:
        tvec = torch.empty(t_shape, dtype=torch.float32, device=dev)
    if tuple(E.shape) != (n_seg, H, dv, dk) or tuple(tvec.shape) != t_shape:
        raise ValueError("E / tvec have the wrong shape")
    with torch.cuda.device(dev):
        rc = lib.hypic_diag_encode(_dev_ptr(k, "k"), _dev_ptr(v, "v"), _dev_ptr(g, "g", torch.float32),
                                   _dev_ptr(cu_seqlens, "cu_seqlens", torch.int32), n_seg, t_total, H, dk, dv,
                                   kv_dtype, int(gate), _dev_ptr(E, "E", torch.float32),
                                   _dev_ptr(tvec, "tvec", torch.float32), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_diag_encode")
    return E, tvec


def hypic_diag_compose(S_in: Optional[torch.Tensor], E_pool: torch.Tensor, t_pool: torch.Tensor,
                       seg_ids: torch.Tensor, cu_segs: torch.Tensor, *, total_steps: Optional[int] = None,
                       S_out: Optional[torch.Tensor] = None,
                       stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """S_out[r,h] = fold of S <- S diag(t_i) + E_i over seg_ids[cu_segs[r]:cu_segs[r+1]] from S_in[r,h] (None = 0);
    t_pool:[P,H] (scalar family) or [P,H,dk] (diagonal family), fp32.  E_pool fp32, or fp16 (hypic_diag_compose_f16)."""
    lib = load_library()
    for name, t in (("E_pool", E_pool), ("t_pool", t_pool), ("seg_ids", seg_ids), ("cu_segs", cu_segs)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if E_pool.dim() != 4:
        raise ValueError("E_pool:[P,H,dv,dk]")
    P, H, dv, dk = (int(x) for x in E_pool.shape)
    if tuple(t_pool.shape) == (P, H):
        gate = HYPIC_GATE_SCALAR
    elif tuple(t_pool.shape) == (P, H, dk):
        gate = HYPIC_GATE_CHANNEL
    else:
        raise ValueError("t_pool must be [P,H] or [P,H,dk]")
    R = int(cu_segs.numel()) - 1
    if R < 0:
        raise ValueError("cu_segs must have R+1 >= 1 entries")
    if total_steps is None:
        total_steps = int(seg_ids.numel())
    if S_in is not None and tuple(S_in.shape) != (R, H, dv, dk):
        raise ValueError("S_in must be [R,H,dv,dk]")
    if S_out is None:
        S_out = torch.empty((R, H, dv, dk), dtype=torch.float32, device=E_pool.device)
    if tuple(S_out.shape) != (R, H, dv, dk):
        raise ValueError("S_out must be [R,H,dv,dk]")
    f16 = E_pool.dtype == torch.float16
    fn = lib.hypic_diag_compose_f16 if f16 else lib.hypic_diag_compose
    with torch.cuda.device(E_pool.device):
        rc = fn(
            _dev_ptr(S_in, "S_in", torch.float32), _dev_ptr(E_pool, "E_pool", torch.float16 if f16 else torch.float32),
            _dev_ptr(t_pool, "t_pool", torch.float32), _dev_ptr(seg_ids, "seg_ids", torch.int32),
            _dev_ptr(cu_segs, "cu_segs", torch.int32), R, P, int(total_steps), H, dk, dv, gate,
            _dev_ptr(S_out, "S_out", torch.float32), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_diag_compose")
    return S_out


def hypic_rope_compose_workspace(total_steps: int, dk: int) -> int:
    return int(load_library().hypic_rope_compose_workspace(int(total_steps), int(dk)))


def hypic_rope_compose(S_in: Optional[torch.Tensor], E_pool: torch.Tensor, t_pool: torch.Tensor,
                       seg_ids: torch.Tensor, cu_segs: torch.Tensor, pos: torch.Tensor, inv_freq: torch.Tensor, *,
                       total_steps: Optional[int] = None, S_out: Optional[torch.Tensor] = None,
                       workspace: Optional[torch.Tensor] = None,
                       stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """Scalar family with RoPE inside the layer (Eq. 7): S <- t_i S + E_i R(pos_i)^T over
    seg_ids[cu_segs[r]:cu_segs[r+1]] from S_in[r,h] (None = 0).  E_pool:[P,H,dv,dk] fp32 (or fp16:
    hypic_rope_compose_f16), t_pool:[P,H] fp32,
    pos:int32[len(seg_ids)], inv_freq:fp32[dk/2].  A workspace is allocated when none is given."""
    lib = load_library()
    for name, t in (("E_pool", E_pool), ("t_pool", t_pool), ("seg_ids", seg_ids), ("cu_segs", cu_segs), ("pos", pos),
                    ("inv_freq", inv_freq)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if E_pool.dim() != 4:
        raise ValueError("E_pool:[P,H,dv,dk]")
    P, H, dv, dk = (int(x) for x in E_pool.shape)
    if tuple(t_pool.shape) != (P, H):
        raise ValueError("t_pool must be [P,H] (scalar family only: a diagonal T does not commute with rotations)")
    if tuple(inv_freq.shape) != (dk // 2,):
        raise ValueError("inv_freq must be [dk/2]")
    if pos.numel() != seg_ids.numel():
        raise ValueError("pos must have one entry per seg_ids entry")
    R = int(cu_segs.numel()) - 1
    if R < 0:
        raise ValueError("cu_segs must have R+1 >= 1 entries")
    if total_steps is None:
        total_steps = int(seg_ids.numel())
    if S_in is not None and tuple(S_in.shape) != (R, H, dv, dk):
        raise ValueError("S_in must be [R,H,dv,dk]")
    if S_out is None:
        S_out = torch.empty((R, H, dv, dk), dtype=torch.float32, device=E_pool.device)
    if tuple(S_out.shape) != (R, H, dv, dk):
        raise ValueError("S_out must be [R,H,dv,dk]")
    need = hypic_rope_compose_workspace(total_steps, dk)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=E_pool.device)
    f16 = E_pool.dtype == torch.float16
    fn = lib.hypic_rope_compose_f16 if f16 else lib.hypic_rope_compose
    with torch.cuda.device(E_pool.device):
        rc = fn(
            _dev_ptr(S_in, "S_in", torch.float32), _dev_ptr(E_pool, "E_pool", torch.float16 if f16 else torch.float32),
            _dev_ptr(t_pool, "t_pool", torch.float32), _dev_ptr(seg_ids, "seg_ids", torch.int32),
            _dev_ptr(cu_segs, "cu_segs", torch.int32), _dev_ptr(pos, "pos", torch.int32),
            _dev_ptr(inv_freq, "inv_freq", torch.float32), R, P, int(total_steps), H, dk, dv,
            _dev_ptr(S_out, "S_out", torch.float32), _dev_ptr(workspace, "workspace", torch.uint8),
            int(workspace.numel()), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_rope_compose")
    return S_out


def hypic_forward_encode(q: torch.Tensor, k: torch.Tensor, v: torch.Tensor, g: torch.Tensor, beta: torch.Tensor,
                         cu_seqlens: torch.Tensor, gate: int = HYPIC_GATE_SCALAR, *,
                         stream: Optional[torch.cuda.Stream] = None) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """One pass per segment from the zero state: per-token outputs o:[Ttot,H,dv] and the tuple (E:[n_seg,H,dv,dk],
    T:[n_seg,H,dk,dk]) of hypic_segment_encode, all fp32."""
    lib = load_library()
    for name, t in (("q", q), ("k", k), ("v", v), ("g", g), ("beta", beta), ("cu_seqlens", cu_seqlens)):
        if not t.is_cuda:
            raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if k.dim() != 3 or v.dim() != 3 or k.shape[:2] != v.shape[:2] or k.dtype != v.dtype or q.shape != k.shape \
            or q.dtype != k.dtype:
        raise ValueError("q, k:[Ttot,H,dk] and v:[Ttot,H,dv] must agree in Ttot, H and dtype")
    t_total, H, dk = (int(x) for x in k.shape)
    dv = int(v.shape[2])
    if k.dtype == torch.bfloat16:
        kv_dtype = HYPIC_DT_BF16
    elif k.dtype == torch.float32:
        kv_dtype = HYPIC_DT_F32
    else:
        raise ValueError(f"q/k/v must be bf16 or fp32, got {k.dtype}")
    want_g = (t_total, H) if gate == HYPIC_GATE_SCALAR else (t_total, H, dk)
    if tuple(g.shape) != want_g or tuple(beta.shape) != (t_total, H):
        raise ValueError(f"g must be {want_g} and beta {(t_total, H)}")
    n_seg = int(cu_seqlens.numel()) - 1
    if n_seg < 0:
        raise ValueError("cu_seqlens must have n_seg+1 >= 1 entries")
    dev = k.device
    o = torch.empty((t_total, H, dv), dtype=torch.float32, device=dev)
    E = torch.empty((n_seg, H, dv, dk), dtype=torch.float32, device=dev)
    T = torch.empty((n_seg, H, dk, dk), dtype=torch.float32, device=dev)
    with torch.cuda.device(dev):
        rc = lib.hypic_forward_encode(
            _dev_ptr(q, "q"), _dev_ptr(k, "k"), _dev_ptr(v, "v"), _dev_ptr(g, "g", torch.float32),
            _dev_ptr(beta, "beta", torch.float32), _dev_ptr(cu_seqlens, "cu_seqlens", torch.int32), n_seg, t_total, H,
            dk, dv, kv_dtype, int(gate), _dev_ptr(o, "o", torch.float32), _dev_ptr(E, "E", torch.float32),
            _dev_ptr(T, "T", torch.float32), _stream_handle(stream))
    if rc != HYPIC_OK:
        raise HypicError(rc, "hypic_forward_encode")
    return o, E, T
