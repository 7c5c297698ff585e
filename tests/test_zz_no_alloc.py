"""hypic_segment_encode_static (include/hypic.h): the allocation-free entry point, whose scratch is a 4 MiB static device
array inside the library, against the existing path hypic_segment_encode (caller-owned workspace) on the same inputs,
within the tolerance of the parity tests (parity_util.TOL_*), on two calls in a row.  Named to be collected last."""
import numpy as np
import pytest
import torch

from paper_2607_01299_b200 import binding as hb
from paper_2607_01299_b200 import workloads as wl
from parity_util import TOL_BF16, TOL_F32, check_E, check_T

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    hb.load_library()  # fail loudly if the extension is missing
    hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)
    yield
    hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)
    assert hb.hypic_debug_timeout_count() == 0, "a tensor-family kernel hit a bounded-wait timeout"


def _existing(inp):
    E, T = hb.hypic_segment_encode(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, inp.gate)
    torch.cuda.synchronize()
    return E, T


def _static(inp, fill):
    n_seg, (_, H, dk), dv = len(inp.seg_lens), inp.k.shape, inp.v.shape[2]
    E = torch.full((n_seg, H, dv, dk), fill, dtype=torch.float32, device=inp.k.device)  # outputs are the caller's,
    T = torch.full((n_seg, H, dk, dk), fill, dtype=torch.float32, device=inp.k.device)  # pre-filled with garbage
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    hb.hypic_segment_encode_static(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, inp.gate, E, T)
    torch.cuda.synchronize()
    return E, T, free0 - torch.cuda.mem_get_info()[0]


def _same(a, b, tol):
    E, T = a
    Er, Tr = (x.detach().cpu().numpy().astype(np.float64) for x in b)
    check_E(E, Er, tol)
    check_T(T, Tr, tol)


def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row():
    """Tensor family (bf16, d = 128, scalar gate), ragged segments over several chunks, an empty one included.  The first
    call's inputs push units onto the in-call fallback list (|v| ~ 1e4 leaves fp16's range), so the shared array is left
    holding a non-empty list; the second call, on ordinary inputs of another shape, must not see any of it."""
    assert hb.hypic_static_scratch_bytes() == 4 << 20
    a = wl.make_encode_inputs([300, 64, 1000, 0, 37], 8, 128, 128, kv_dtype=torch.bfloat16, seed=wl.seed_for(1, 71),
                              device="cuda")
    a.v.mul_(1.0e4)
    b = wl.make_encode_inputs([129, 700, 64, 5], 4, 128, 128, kv_dtype=torch.bfloat16, seed=wl.seed_for(1, 72),
                              device="cuda")
    ref_a, ref_b = _existing(a), _existing(b)  # also loads every kernel the static calls will launch
    Ea, Ta, _ = _static(a, 7.0)
    Eb, Tb, grew = _static(b, float("nan"))
    _same((Ea, Ta), ref_a, TOL_BF16)
    _same((Eb, Tb), ref_b, TOL_BF16)
    assert grew == 0, f"device memory in use grew by {grew} bytes across an allocation-free call"
    # and again in the other order: every call leaves the array usable for the next
    Ea2, Ta2, _ = _static(a, -1.0)
    _same((Ea2, Ta2), ref_a, TOL_BF16)


def test_static_entry_covers_the_fp32_family_too():
    """cfg0 (fp32, d = 64) runs on the family that needs no scratch at all: same entry point, same results."""
    inp = wl.cfg0(device="cuda")
    ref = _existing(inp)
    for fill in (0.0, 3.0):
        E, T, _ = _static(inp, fill)
        _same((E, T), ref, TOL_F32)


def test_static_entry_per_channel_gate_that_fits():
    """Per-channel gate (prep records in the scratch): 3 chunks x 2 heads fit; twice in a row, second time on other data."""
    for seed in (74, 75):
        inp = wl.make_encode_inputs([100, 64], 2, 128, 128, kv_dtype=torch.bfloat16, gate=wl.GATE_CHANNEL, g_lo=-0.02,
                                    seed=wl.seed_for(3, seed), device="cuda")
        ref = _existing(inp)
        E, T, _ = _static(inp, float("nan"))
        _same((E, T), ref, TOL_BF16)


def test_static_entry_rejects_what_does_not_fit():
    """Per-channel gate at d = 128: 40 KB of prep record per chunk and head; 64 chunks x 8 heads is far beyond 4 MiB.
    The call must return HYPIC_ERR_STATIC_SCRATCH without launching anything (the outputs keep their fill)."""
    inp = wl.make_encode_inputs([4096], 8, 128, 128, kv_dtype=torch.bfloat16, gate=wl.GATE_CHANNEL, g_lo=-0.01,
                                seed=wl.seed_for(3, 73), device="cuda")
    need = hb.hypic_segment_encode_workspace(1, 4096, 8, 128, 128, hb.HYPIC_DT_BF16, hb.HYPIC_GATE_CHANNEL)
    assert need > hb.hypic_static_scratch_bytes()
    E = torch.full((1, 8, 128, 128), 5.0, dtype=torch.float32, device="cuda")
    T = torch.full((1, 8, 128, 128), 5.0, dtype=torch.float32, device="cuda")
    with pytest.raises(hb.HypicError) as ei:
        hb.hypic_segment_encode_static(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, inp.gate, E, T)
    torch.cuda.synchronize()
    assert ei.value.status == hb.HYPIC_ERR_STATIC_SCRATCH
    assert "static" in hb.hypic_status_string(hb.HYPIC_ERR_STATIC_SCRATCH)
    assert bool((E == 5.0).all()) and bool((T == 5.0).all())
