"""GPU parity: libhypic (through the C ABI via the thin binding) vs the fp64 oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json:north_star's (parity_util.TOL_*).  Every kernel family is
checked (AUTO = what bench.py times, SIMT, TENSOR); a family that does not cover a shape is skipped."""
import contextlib

import numpy as np
import pytest
import torch

import oracle
from paper_2607_01299_b200 import binding as hb
from paper_2607_01299_b200 import workloads as wl
from parity_util import (per_unit_rel, TOL_BF16, TOL_F32, check_E, check_T, oracle_compose_units, oracle_encode,
                         oracle_encode_units, oracle_encode_units_batched)

pytestmark = pytest.mark.gpu
T_FLOOR_TEST = 1e-30  # reading S6: below this norm T is compared absolutely

IMPLS = [("auto", hb.HYPIC_IMPL_AUTO), ("simt", hb.HYPIC_IMPL_SIMT), ("tensor", hb.HYPIC_IMPL_TENSOR)]


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    hb.load_library()  # fail loudly if the extension is missing
    yield
    hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)
    assert hb.hypic_debug_timeout_count() == 0, "a tensor-family kernel hit a bounded-wait timeout"


@contextlib.contextmanager
def impl_family(impl):
    hb.hypic_set_impl(impl)
    try:
        yield
    except hb.HypicError as e:
        if e.status == hb.HYPIC_ERR_UNSUPPORTED and impl == hb.HYPIC_IMPL_TENSOR:
            pytest.skip("tensor family does not cover this shape")
        raise
    finally:
        hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)


def gpu_encode(inp, impl):
    with impl_family(impl):
        E, T = hb.hypic_segment_encode(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, inp.gate)
        torch.cuda.synchronize()
    return E, T


def gpu_compose(S_in, E, T, ids, cu, impl, **kw):
    with impl_family(impl):
        out = hb.hypic_compose(S_in, E, T, ids, cu, **kw)
        torch.cuda.synchronize()
    return out


# ------------------------------------------------------------------------------------------------ cfg0
@pytest.mark.parametrize("name,impl", IMPLS)
def test_cfg0_fp32_encode_and_compose_vs_sequential(name, impl):
    """cfg0: 1 head, d=64, fp32, 2 x 128 tokens; E,T per segment; compose from 0 and from N(0,0.1) must equal
    the sequential recurrence over all 256 tokens (Eq. 4)."""
    inp = wl.cfg0("cuda")
    E, T = gpu_encode(inp, impl)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_F32)
    check_T(T, T_ref, TOL_F32)
    s_in = wl.cfg0_s_in("cuda")
    ids = torch.tensor([0, 1, 0, 1], dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, 2, 4], dtype=torch.int32, device="cuda")
    S_in = torch.cat([torch.zeros_like(s_in), s_in], 0)
    S = gpu_compose(S_in, E, T, ids, cu, impl)
    c = inp.cpu()
    seq = oracle.sequential(S_in.cpu().numpy().astype(np.float64), torch.cat([c.k, c.k]), torch.cat([c.v, c.v]),
                            torch.cat([c.g, c.g]), torch.cat([c.beta, c.beta]),
                            np.array([0, 256, 512], dtype=np.int32), gate=c.gate)
    check_E(S, seq, TOL_F32, "S_out vs sequential")
    # S_in = NULL is the same as zeros
    S0 = gpu_compose(None, E, T, ids[:2].contiguous(), cu[:2].contiguous(), impl)
    check_E(S0, seq[:1], TOL_F32, "S_out (S_in=NULL) vs sequential")


# ------------------------------------------------------------------------- ragged / edge-case encodes
RAGGED = [200, 64, 65, 1, 0, 63, 333, 128, 0, 2]


@pytest.mark.parametrize("name,impl", IMPLS)
@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
@pytest.mark.parametrize("kv,d,tol", [(torch.bfloat16, 128, TOL_BF16), (torch.float32, 128, TOL_F32),
                                      (torch.float32, 64, TOL_F32), (torch.bfloat16, 64, TOL_BF16)])
def test_encode_ragged_segments(name, impl, gate, kv, d, tol):
    """Lengths spanning several 64-token chunks with ragged tails, plus length 0 / 1 / 63 / 64 / 65."""
    inp = wl.make_encode_inputs(RAGGED, 3, d, d, kv_dtype=kv, gate=gate, g_lo=-0.05, seed=wl.seed_for(1, 11),
                                device="cuda")
    E, T = gpu_encode(inp, impl)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, tol)
    check_T(T, T_ref, tol)
    # empty segments: E = 0, T = I exactly
    for s, L in enumerate(RAGGED):
        if L == 0:
            assert torch.count_nonzero(E[s]) == 0
            assert torch.equal(T[s], torch.eye(d, device="cuda").expand_as(T[s]))


@pytest.mark.parametrize("name,impl", IMPLS)
def test_encode_dv_not_equal_dk(name, impl):
    inp = wl.make_encode_inputs([70, 129], 2, 64, 96, kv_dtype=torch.float32, seed=wl.seed_for(0, 3), device="cuda")
    E, T = gpu_encode(inp, impl)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_F32)
    check_T(T, T_ref, TOL_F32)


@pytest.mark.parametrize("name,impl", IMPLS)
def test_encode_degenerate_inputs(name, impl):
    """beta = 0 => T = (prod alpha) I, E = 0; n_seg = 0; all segments empty."""
    inp = wl.make_encode_inputs([130, 64], 2, 128, 128, kv_dtype=torch.bfloat16, seed=5, device="cuda")
    inp.beta.zero_()
    E, T = gpu_encode(inp, impl)
    assert torch.count_nonzero(E) == 0
    g = inp.g.double().cpu()
    for s, (a, b) in enumerate([(0, 130), (130, 194)]):
        for h in range(2):
            want = torch.exp(g[a:b, h].sum()) * torch.eye(128, dtype=torch.float64)
            assert torch.allclose(T[s, h].double().cpu(), want, rtol=2e-5, atol=0)
    empty = wl.make_encode_inputs([], 2, 128, 128, kv_dtype=torch.bfloat16, seed=5, device="cuda")
    E0, T0 = gpu_encode(empty, impl)
    assert E0.shape == (0, 2, 128, 128) and T0.shape == (0, 2, 128, 128)
    zeros = wl.make_encode_inputs([0, 0], 2, 128, 128, kv_dtype=torch.bfloat16, seed=5, device="cuda")
    E1, T1 = gpu_encode(zeros, impl)
    assert torch.count_nonzero(E1) == 0 and torch.equal(T1, torch.eye(128, device="cuda").expand_as(T1))


# ------------------------------------------------------------------------------------------ compose
@pytest.mark.parametrize("name,impl", IMPLS)
@pytest.mark.parametrize("H", [3, 4])
@pytest.mark.parametrize("d", [128, 64])
def test_compose_near_unit_pool(name, impl, d, H):
    """Reading S9: pool with ||T||_F = O(1..10) (short segments, weak decay), so S.T is not negligible; fp32
    pools vs fp64 compose of the same pools -> 1e-5.  Lists of length 0, 1 and up to 40; unsorted ids."""
    P = 24  # H = 3: one chain per CTA in the tensor family; H = 4: heads h, h + 1 interleaved in one CTA
    pin = wl.near_unit_pool_inputs(P, H, device="cuda", d=d, kv_dtype=torch.float32)
    hb.hypic_set_impl(hb.HYPIC_IMPL_SIMT)
    E, T = hb.hypic_segment_encode(pin.k, pin.v, pin.g, pin.beta, pin.cu_seqlens, pin.gate)
    hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)
    assert float(T.norm(dim=(-1, -2)).min()) > 0.5
    req = wl.make_compose_requests(9, P, H, d, d, n_lo=0, n_hi=24, seed=77, device="cuda", s_in_std=1.0)
    # force an empty list and a singleton
    cu = req.cu_segs.cpu().clone()
    S = gpu_compose(req.S_in, E, T, req.seg_ids, req.cu_segs, impl)
    ref = oracle.compose(req.S_in.cpu().numpy(), E.cpu().numpy(), T.cpu().numpy(), req.seg_ids.cpu().numpy(),
                         cu.numpy())
    check_E(S, ref, TOL_F32, "S_out")
    # long chain that repeats ids (40 steps)
    gen = torch.Generator().manual_seed(123)
    ids = torch.randint(0, P, (40,), generator=gen, dtype=torch.int32).cuda()
    cu2 = torch.tensor([0, 0, 1, 40], dtype=torch.int32, device="cuda")  # empty, singleton, 39-long
    S_in2 = torch.randn(3, H, d, d, device="cuda")
    S2 = gpu_compose(S_in2, E, T, ids, cu2, impl)
    ref2 = oracle.compose(S_in2.cpu().numpy(), E.cpu().numpy(), T.cpu().numpy(), ids.cpu().numpy(),
                          cu2.cpu().numpy())
    check_E(S2, ref2, TOL_F32, "S_out (chain)")
    assert torch.equal(S2[0], S_in2[0])  # empty list copies S_in
    # in-place: S_out aliases S_in
    S3 = S_in2.clone()
    gpu_compose(S3, E, T, ids, cu2, impl, S_out=S3)
    assert torch.equal(S3, S2)
    # S_in = NULL
    S4 = gpu_compose(None, E, T, ids, cu2, impl)
    ref4 = oracle.compose(None, E.cpu().numpy(), T.cpu().numpy(), ids.cpu().numpy(), cu2.cpu().numpy())
    check_E(S4, ref4, TOL_F32, "S_out (NULL S_in)")
    assert torch.count_nonzero(S4[0]) == 0


@pytest.mark.parametrize("name,impl", IMPLS)
def test_compose_order_matters(name, impl):
    pin = wl.near_unit_pool_inputs(4, 1, device="cuda", d=128, kv_dtype=torch.float32, seed_off=3)
    hb.hypic_set_impl(hb.HYPIC_IMPL_SIMT)
    E, T = hb.hypic_segment_encode(pin.k, pin.v, pin.g, pin.beta, pin.cu_seqlens, pin.gate)
    hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)
    ids = torch.tensor([0, 1, 2, 3, 3, 2, 1, 0], dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, 4, 8], dtype=torch.int32, device="cuda")
    S = gpu_compose(None, E, T, ids, cu, impl)
    ref = oracle.compose(None, E.cpu().numpy(), T.cpu().numpy(), ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S, ref, TOL_F32)
    assert oracle.rel_fro(S[0].cpu().numpy(), ref[1]) > 1e-2  # the two orders really differ


# ------------------------------------------------------------- end to end at bf16: encode -> compose
@pytest.mark.parametrize("name,impl", IMPLS)
def test_cfg1_small_end_to_end_vs_sequential(name, impl):
    """cfg1 scaled down (H=4, 4 x 320 tokens): GPU encode (bf16) -> GPU compose vs the fp64 sequential
    recurrence over the concatenation -> 3e-3 (reading S8)."""
    inp = wl.cfg1("cuda", seg_len=320, n_seg=4, H=4)
    E, T = gpu_encode(inp, impl)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)
    ids = torch.arange(4, dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, 4], dtype=torch.int32, device="cuda")
    S = gpu_compose(None, E, T, ids, cu, impl)
    c = inp.cpu()
    seq = oracle.sequential(None, c.k, c.v, c.g, c.beta, np.array([0, 1280], dtype=np.int32), gate=c.gate)
    check_E(S, seq, TOL_BF16, "S_out vs sequential")


# ------------------------------------------- full sizes, bench.py's launch configuration (AUTO family)
def _sample_units(n_a, n_b, n, seed):
    gen = np.random.default_rng(seed)
    return sorted({(int(gen.integers(n_a)), int(gen.integers(n_b))) for _ in range(n)})


def test_cfg1_full_size():
    """cfg1 as written (H=16, 4 x 2048, bf16): every unit against the oracle, then compose the 4 in order."""
    inp = wl.cfg1("cuda")
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)
    ids = torch.arange(4, dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, 4], dtype=torch.int32, device="cuda")
    S = gpu_compose(None, E, T, ids, cu, hb.HYPIC_IMPL_AUTO)
    ref = oracle.compose(None, E.cpu().numpy(), T.cpu().numpy(), ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S, ref, TOL_F32, "S_out vs fp64 compose of the same pools")
    ref_e2e = oracle.compose(None, E_ref, T_ref, ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S, ref_e2e, TOL_BF16, "S_out end to end")


def _compose_all_heads_ref(S_in, E, T, ids, cu):
    """fp64 compose of the same fp32 pools, every (request, head) chain, in one oracle call."""
    return oracle.compose(None if S_in is None else S_in.cpu().numpy(), E.cpu().numpy(), T.cpu().numpy(),
                          ids.cpu().numpy(), cu.cpu().numpy())


def test_cfg2_one_layer_every_unit():
    """cfg2, one of the 36 layers at full size (20 x 4096, H=32): EVERY one of the 640 (segment, head) units against the
    oracle (a tail-wave or head-boundary bug that hits one unit in fifty cannot hide behind a sample), then the
    composition of the 20 segments for every head."""
    inp = wl.cfg2_layer(0, "cuda")
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)  # 4096 tokens: T underflows -> absolute criterion
    ids = torch.arange(20, dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, 20], dtype=torch.int32, device="cuda")
    S = gpu_compose(None, E, T, ids, cu, hb.HYPIC_IMPL_AUTO)
    check_E(S, _compose_all_heads_ref(None, E, T, ids, cu), TOL_F32, "S_out")
    check_E(S, oracle.compose(None, E_ref, T_ref, ids.cpu().numpy(), cu.cpu().numpy()), TOL_BF16, "S_out end to end")


def test_cfg2_folded_layers_launch_configuration_every_unit():
    """cfg2 in the launch configuration bench.py times: 6 independent layers folded into the head axis (H = 192,
    SURVEY.md 8(b); bench.py's --fold default: 3,840 units = 25.9 waves on 148 SMs), full size (20 x 4096).  The folded
    call must reproduce the per-layer calls bit for bit (units are independent), ALL 3,840 units are checked against the
    oracle, and so is the folded composition of every head."""
    layers = [wl.cfg2_layer(l, "cuda") for l in range(6)]
    inp = wl.fold_layers(layers)
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    for l in (0, 5):
        E1, T1 = gpu_encode(layers[l], hb.HYPIC_IMPL_AUTO)
        assert torch.equal(E[:, 32 * l:32 * l + 32], E1) and torch.equal(T[:, 32 * l:32 * l + 32], T1)
        del E1, T1
    del layers
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)
    del E_ref, T_ref
    ids = torch.arange(20, dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, 20], dtype=torch.int32, device="cuda")
    S = gpu_compose(None, E, T, ids, cu, hb.HYPIC_IMPL_AUTO)
    check_E(S, _compose_all_heads_ref(None, E, T, ids, cu), TOL_F32, "S_out (folded)")


def test_cfg3_varlen_channel_gate_full_head_count():
    """cfg3 exactly as bench.py times it (64 varlen segments, per-channel gate, H = 32): the shortest and the longest
    segment plus 34 sampled (segment, head) units, one oracle call over all of them."""
    inp = wl.cfg3("cuda")
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    assert torch.isfinite(E).all() and torch.isfinite(T).all()
    lens = inp.seg_lens
    units = [(int(np.argmin(lens)), 1), (int(np.argmin(lens)), 31), (int(np.argmax(lens)), 2), (int(np.argmax(lens)), 30)]
    units += [u for u in _sample_units(64, 32, 34, 3) if u not in units]
    E_ref, T_ref = oracle_encode_units_batched(inp, units)
    si, hi = torch.tensor([u[0] for u in units]), torch.tensor([u[1] for u in units])
    check_E(E[si, hi][:, None], E_ref, TOL_BF16)
    check_T(T[si, hi][:, None], T_ref, TOL_BF16)


def test_cfg4_compose_stress_every_chain():
    """cfg4 at full size for one layer-iteration (P=1024, H=32, R=128, n_r ~ U{16..64}): ALL 4,096 (request, head)
    chains against the fp64 compose of the same fp32 pools."""
    pin = wl.cfg4_pool_inputs(device="cuda")
    _, T = gpu_encode(pin, hb.HYPIC_IMPL_AUTO)
    del pin
    E = wl.cfg4_pool_E(device="cuda")
    req = wl.cfg4_requests(device="cuda")
    S = gpu_compose(req.S_in, E, T, req.seg_ids, req.cu_segs, hb.HYPIC_IMPL_AUTO)
    check_E(S, _compose_all_heads_ref(req.S_in, E, T, req.seg_ids, req.cu_segs), TOL_F32, "S_out")


# ------------------------------------------------- tensor family: range handling of the fp16 operands
@pytest.mark.parametrize("case", ["strong_erasure", "no_gate_long", "v_x100", "v_x0.01", "gate_x2"])
def test_tensor_family_operand_range(case):
    """The tensor family feeds fp16 operands to tcgen05.mma; T rows are held row-normalised in TMEM.
    Cases that move T, E or the gate far from the benchmark distributions must still meet the bf16 tolerance:
    beta = 1 (every key is fully erased, T decays by projections alone), g = 0 over 1536 tokens (no gate decay at
    all, T shrinks only through the delta rule), v scaled by 100 and by 0.01, and g ~ U(-1, 0) (T underflows fp32
    within a few hundred tokens: absolute criterion of reading S6)."""
    lens = [1536, 200] if case == "no_gate_long" else [384, 130, 64]
    inp = wl.make_encode_inputs(lens, 2, 128, 128, kv_dtype=torch.bfloat16, g_lo=-0.05, seed=wl.seed_for(1, 31),
                                device="cuda")
    if case == "strong_erasure":
        inp.beta.fill_(1.0)
    elif case == "no_gate_long":
        inp.g.zero_()
    elif case == "v_x100":
        inp.v.mul_(100.0)
    elif case == "v_x0.01":
        inp.v.mul_(0.01)
    elif case == "gate_x2":
        inp.g.mul_(2.0)
    before = hb.hypic_envelope_violation_count()
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_TENSOR)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)
    assert hb.hypic_envelope_violation_count() == before


def test_tensor_encode_is_deterministic_and_order_independent():
    """The fused encode kernel pipelines producer warps, two chains and TMA rings through a dozen barriers; a missing
    hand-over shows up as run-to-run differences long before it breaks the tolerance (a race between two producer
    warps did exactly that during development: errors of 2e-4 .. 3e-2 depending on timing, on short ragged segments
    only).  Same inputs twice -> bit-identical outputs; and every unit equals its own single-unit call (units are
    independent whatever their neighbours and the launch shape are)."""
    lens = [200, 64, 130, 1000, 1, 4096, 0, 63]
    inp = wl.make_encode_inputs(lens, 3, 128, 128, kv_dtype=torch.bfloat16, seed=wl.seed_for(1, 36), device="cuda")
    E0, T0 = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    for _ in range(4):
        E1, T1 = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
        assert torch.equal(E0, E1) and torch.equal(T0, T1)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E0, E_ref, TOL_BF16)
    check_T(T0, T_ref, TOL_BF16)
    cu = np.concatenate([[0], np.cumsum(lens)])
    for s, h in [(0, 0), (2, 1), (3, 2), (7, 0)]:
        sl = slice(int(cu[s]), int(cu[s + 1]))
        one = wl.EncodeInputs(k=inp.k[sl, h:h + 1].contiguous(), v=inp.v[sl, h:h + 1].contiguous(),
                              g=inp.g[sl, h:h + 1].contiguous(), beta=inp.beta[sl, h:h + 1].contiguous(),
                              cu_seqlens=torch.tensor([0, lens[s]], dtype=torch.int32, device="cuda"), gate=inp.gate,
                              seg_lens=[lens[s]])
        E1, T1 = gpu_encode(one, hb.HYPIC_IMPL_AUTO)
        assert torch.equal(E1[0, 0], E0[s, h]) and torch.equal(T1[0, 0], T0[s, h])


@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
@pytest.mark.parametrize("g_lo", [-1.0, -0.3])
def test_auto_meets_tolerance_for_any_gate_strength(gate, g_lo):
    """Table 1's gates are data-dependent with no range given.  g ~ U(-1, 0) puts the log-decay of a
    64-token chunk near -32, g ~ U(-0.3, 0) near -10.  AUTO (what a caller gets by default) must meet the bf16
    tolerance with no caller action: the scalar gate never enters the fp16 algebra, a per-channel
    chunk below e^-9 sends its unit to the fp32 family inside the same call (device-side fallback list)."""
    inp = wl.make_encode_inputs([700, 130, 64, 1], 3, 128, 128, kv_dtype=torch.bfloat16, gate=gate, g_lo=g_lo,
                                seed=wl.seed_for(1, 32), device="cuda")
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)


def test_fallback_list_takes_only_the_units_that_need_it():
    """Per-channel gate, one (segment, head) with one strongly decaying channel range: that unit alone leaves the fp16
    envelope.  Every unit must match the oracle, and the units inside the envelope must be bit-identical to a call
    without the outlier (they stay on the tcgen05 path)."""
    inp = wl.make_encode_inputs([256, 300, 128], 4, 128, 128, kv_dtype=torch.bfloat16, gate=wl.GATE_CHANNEL,
                                seed=wl.seed_for(3, 33), device="cuda")
    E0, T0 = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    before = hb.hypic_envelope_violation_count()
    inp.g[256 + 70:256 + 200, 2, 5:9] = -0.4  # segment 1, head 2: chunks 1 and 2 decay to e^-25 in four channels
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    assert hb.hypic_envelope_violation_count() > before
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)
    keep = torch.ones(3, 4, dtype=torch.bool)
    keep[1, 2] = False
    assert torch.equal(E[keep], E0[keep]) and torch.equal(T[keep], T0[keep])
    assert not torch.equal(E[1, 2], E0[1, 2])


def test_tensor_encode_random_ragged_mixes_are_reproducible_and_match_the_fp32_family():
    """24 random mixes of segment counts, head counts, lengths (empty, shorter than a chunk, ragged, up to 2,100 tokens)
    and gate strengths through the fused tensor kernel: every call reproduces itself bit for bit (the kernel pipelines
    six warp roles through some forty barriers), and matches the fp32 SIMT family -- itself checked against the oracle
    above -- within the bf16 tolerance on every unit."""
    rng = np.random.default_rng(123)

    def rel(a, b):
        num = (a.double() - b.double()).flatten(2).norm(dim=-1)
        den = b.double().flatten(2).norm(dim=-1)
        return float(torch.where(den > T_FLOOR_TEST, num / den.clamp_min(1e-300), num).max())

    for trial in range(24):
        n_seg, H, mode = int(rng.integers(1, 40)), int(rng.integers(1, 9)), trial % 4
        lens = [int(x) for x in rng.integers(0, [700, 130, 2100, 66][mode], n_seg)]
        if sum(lens) == 0:
            lens[0] = 5
        inp = wl.make_encode_inputs(lens, H, 128, 128, kv_dtype=torch.bfloat16, g_lo=[-0.05, -0.5, -0.01, -0.1][mode],
                                    seed=wl.seed_for(1, 100 + trial), device="cuda")
        E1, T1 = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
        E2, T2 = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
        assert torch.equal(E1, E2) and torch.equal(T1, T2), f"trial {trial}: two runs differ"
        Es, Ts = gpu_encode(inp, hb.HYPIC_IMPL_SIMT)
        eE, eT = rel(E1, Es), rel(T1, Ts)
        assert eE <= TOL_BF16 and eT <= TOL_BF16, f"trial {trial}: E {eE:.2e} T {eT:.2e} (H={H}, lens={lens[:8]}...)"
    assert hb.hypic_debug_timeout_count() == 0


def test_long_weakly_gated_segments_stay_within_tolerance():
    """The fp16 operands' rounding is a random walk over the chunks (T: ~1.4e-3 at 4,096 tokens, ~2.2e-3 at 8,192, ~3e-3 at
    16,384), which only shows where T is still representable, i.e. for very weak gates.  AUTO must meet the tolerance
    there too: units beyond 8,192 tokens whose T stays above the 1e-30 floor are recomputed by the fp32 family inside the
    call; shorter ones and strongly decaying ones stay on the tensor kernel."""
    inp = wl.make_encode_inputs([16384, 8192, 4096], 2, 128, 128, kv_dtype=torch.bfloat16, g_lo=-0.002, seed=wl.seed_for(1, 41),
                                device="cuda")
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)
    # the 16,384-token units came from the fp32 family (a few 1e-4 after that many fp32 steps), the 8,192-token ones from the
    # tensor kernel (~2e-3)
    err = per_unit_rel(T.cpu().numpy(), T_ref)
    assert err[0].max() < 6e-4 and err[1].min() > 1e-3, err


@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
def test_fp16_operand_overflow_falls_back_in_call(gate):
    """|v| up to ~5e4: the weighted values leave fp16's range inside the tensor family, the result would hold Inf / NaN;
    the unit must come back from the fp32 family instead, within tolerance."""
    inp = wl.make_encode_inputs([200, 64], 2, 128, 128, kv_dtype=torch.bfloat16, gate=gate, seed=wl.seed_for(1, 34),
                                device="cuda")
    inp.v.mul_(1.0e4)
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    E_ref, T_ref = oracle_encode(inp)
    check_E(E, E_ref, TOL_BF16)
    check_T(T, T_ref, TOL_BF16)


@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
def test_neighbour_segment_cannot_poison_a_ragged_tail(gate):
    """The TMA boxes of a segment's last chunk also hold the first tokens of the next segment.  Inf / NaN planted
    there must not reach this segment (0 x Inf = NaN): its E and T still match the oracle."""
    inp = wl.make_encode_inputs([100, 64, 30], 2, 128, 128, kv_dtype=torch.bfloat16, gate=gate, seed=wl.seed_for(1, 35),
                                device="cuda")
    ref = wl.make_encode_inputs([100, 64, 30], 2, 128, 128, kv_dtype=torch.bfloat16, gate=gate, seed=wl.seed_for(1, 35),
                                device="cuda")
    inp.k[100:164] = float("inf")
    inp.v[100:164] = float("nan")
    E, T = gpu_encode(inp, hb.HYPIC_IMPL_AUTO)
    E_ref, T_ref = oracle_encode(ref)
    for s in (0, 2):
        check_E(E[s:s + 1], E_ref[s:s + 1], TOL_BF16)
        check_T(T[s:s + 1], T_ref[s:s + 1], TOL_BF16)
    assert not torch.isfinite(E[1]).all()  # the poisoned segment itself is non-finite on both sides


# ------------------------------------------------------------- fp16-stored tuples
def test_tuple_pack_f16_is_ieee_rne():
    """hypic_tuple_pack_f16 = IEEE fp32 -> fp16 conversion, bit for bit (numpy's astype is the definition): normal
    values, fp16 subnormals, overflow to inf, signed zeros, a ragged tail."""
    gen = torch.Generator().manual_seed(5)
    x = torch.randn(4099, generator=gen) * torch.pow(10.0, torch.randint(-9, 6, (4099,), generator=gen).float())
    x[:6] = torch.tensor([0.0, -0.0, 65504.0, 65520.0, -1e-8, 6.0e-8])
    got = hb.hypic_tuple_pack_f16(x.cuda()).cpu().numpy()
    with np.errstate(over="ignore"):
        want = x.numpy().astype(np.float16)
    assert np.array_equal(got.view(np.uint16), want.view(np.uint16))
    assert hb.hypic_tuple_pack_f16(torch.empty(0, device="cuda")).numel() == 0


@pytest.mark.parametrize("H", [3, 4])
def test_compose_f16_pools_vs_oracle(H):
    """hypic_compose_f16: pools stored in fp16 (as the paper caches them) are exact inputs; the fold
    must match the fp64 compose of the same stored values to the fp32-input tolerance.  Near-unit pool (reading S9),
    lists of length 0, 1 and 39, repeated and unsorted ids, NULL and in-place S."""
    P, d = 24, 128  # H = 3: one chain per CTA; H = 4: heads h, h + 1 interleaved in one CTA
    pin = wl.near_unit_pool_inputs(P, H, device="cuda", d=d, kv_dtype=torch.float32)
    hb.hypic_set_impl(hb.HYPIC_IMPL_SIMT)
    E, T = hb.hypic_segment_encode(pin.k, pin.v, pin.g, pin.beta, pin.cu_seqlens, pin.gate)
    hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)
    Eh, Th = hb.hypic_tuple_pack_f16(E), hb.hypic_tuple_pack_f16(T)
    E64, T64 = Eh.cpu().numpy().astype(np.float32), Th.cpu().numpy().astype(np.float32)
    gen = torch.Generator().manual_seed(321)
    ids = torch.randint(0, P, (40,), generator=gen, dtype=torch.int32).cuda()
    cu = torch.tensor([0, 0, 1, 40], dtype=torch.int32, device="cuda")
    S_in = torch.randn(3, H, d, d, device="cuda")
    S = hb.hypic_compose_f16(S_in, Eh, Th, ids, cu)
    torch.cuda.synchronize()
    ref = oracle.compose(S_in.cpu().numpy(), E64, T64, ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S, ref, TOL_F32, "S_out (fp16 pools)")
    assert torch.equal(S[0], S_in[0])  # empty list copies S_in
    S0 = hb.hypic_compose_f16(None, Eh, Th, ids, cu)
    ref0 = oracle.compose(None, E64, T64, ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S0, ref0, TOL_F32, "S_out (fp16 pools, NULL S_in)")
    S3 = S_in.clone()
    hb.hypic_compose_f16(S3, Eh, Th, ids, cu, S_out=S3)
    assert torch.equal(S3, S)
    # what fp16 storage costs against the fp32 tuples (context: the paper reports 6e-5 at layer 0)
    ref32 = oracle.compose(S_in.cpu().numpy(), E.cpu().numpy(), T.cpu().numpy(), ids.cpu().numpy(), cu.cpu().numpy())
    assert oracle.rel_fro(S.cpu().numpy()[2], ref32[2]) < 2e-3
    with pytest.raises(hb.HypicError):
        hb.hypic_compose_f16(None, Eh[..., :64, :64].contiguous(), Th[..., :64, :64].contiguous(), ids, cu)


def test_cfg4_compose_f16_sampled_requests():
    """cfg4 at full size for one layer-iteration with fp16-stored pools: sampled chains against the fp64 compose of
    the stored values."""
    pin = wl.cfg4_pool_inputs(device="cuda")
    _, T = gpu_encode(pin, hb.HYPIC_IMPL_AUTO)
    del pin
    Th = hb.hypic_tuple_pack_f16(T)
    del T
    Eh = hb.hypic_tuple_pack_f16(wl.cfg4_pool_E(device="cuda"))
    req = wl.cfg4_requests(device="cuda")
    S = hb.hypic_compose_f16(req.S_in, Eh, Th, req.seg_ids, req.cu_segs)
    assert torch.isfinite(S).all()
    units = _sample_units(128, 32, 6, 5)
    ref = oracle_compose_units(req.S_in, Eh.float(), Th.float(), req.seg_ids, req.cu_segs, units)
    ri, hi = torch.tensor([u[0] for u in units]), torch.tensor([u[1] for u in units])
    check_E(S[ri, hi][:, None], ref, TOL_F32, "S_out")


# ------------------------------------------------------------------------------------------------ seam window
def _oracle_seam(si):
    c = si.enc.cpu()
    return oracle.seam_window(si.S_in.cpu().numpy(), si.q.float().cpu().numpy(), c.k, c.v, c.g, c.beta, c.cu_seqlens,
                              gate=c.gate)


def _typical_readout(S_in, q, k, v, g, beta, cu, gate):
    """||S_t||_F ||q_t||_2 / sqrt(dk) per (token, head): the size a read-out of the state S_t has for a query in general
    position.  S_t comes from the oracle, one token at a time.  numpy inputs; S_in may be None."""
    ttot, H, dk = q.shape
    out = np.zeros((ttot, H))
    for r in range(len(cu) - 1):
        S = None if S_in is None else S_in[r:r + 1]
        for t in range(int(cu[r]), int(cu[r + 1])):
            sl = slice(t, t + 1)
            S, _ = oracle.seam_window(S, q[sl], k[sl], v[sl], g[sl], beta[sl], np.array([0, 1], dtype=np.int32), gate=gate)
            out[t] = np.sqrt((S[0] ** 2).sum(axis=(-1, -2))) * np.sqrt((q[t].astype(np.float64) ** 2).sum(-1)) / np.sqrt(dk)
    return out


def _check_o(o_gpu, o_ref, cu, tol, typical=None):
    """DESIGN.md reading W2: per (token, head), ||o - o_ref||_2 <= tol * max(||o_ref||_2, ||S_t||_F ||q_t||_2 / sqrt(dk)).
    The first term is the plain relative error; the second keeps the bound meaningful where q_t is nearly orthogonal to
    the state (o_t = S_t q_t cancels and no fp32 evaluation can be relatively accurate).  Rows outside every window must
    be left untouched."""
    o_gpu = o_gpu.cpu().numpy().astype(np.float64)
    inside = np.zeros(o_ref.shape[0], dtype=bool)
    for r in range(len(cu) - 1):
        inside[cu[r]:cu[r + 1]] = True
    assert np.isfinite(o_gpu).all()
    num = np.sqrt(((o_gpu[inside] - o_ref[inside]) ** 2).sum(-1))
    den = np.sqrt((o_ref[inside] ** 2).sum(-1))
    if typical is not None:
        den = np.maximum(den, typical[inside])
    worst = float((num / np.maximum(den, 1e-300)).max()) if inside.any() else 0.0
    assert worst <= tol, f"o: max per-token rel. L2 error {worst:.3e} > {tol:.1e}"
    if typical is not None and inside.any():
        # rows whose read-out is not a cancellation (||o_ref|| at least the general-position size) must also meet the
        # PLAIN relative bound, so that a regression in well-conditioned rows cannot hide behind the W2 denominator
        plain = np.sqrt((o_ref[inside] ** 2).sum(-1))
        good = plain >= typical[inside]
        if good.any():
            worst_plain = float((num[good] / np.maximum(plain[good], 1e-300)).max())
            assert worst_plain <= tol, f"o: max plain rel. L2 error on well-conditioned rows {worst_plain:.3e} > {tol:.1e}"
    assert np.all(o_gpu[~inside] == 0.0), "o rows outside every window must be left untouched"
    return worst


@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
@pytest.mark.parametrize("kv,d,dv", [(torch.bfloat16, 128, 128), (torch.float32, 128, 128), (torch.float32, 64, 64),
                                     (torch.bfloat16, 128, 72), (torch.float32, 64, 33)])
def test_seam_window_vs_oracle(gate, kv, d, dv):
    """hypic_seam_window: windows of w = 8 (the default), 0, 1, 7, 9 (a ragged second tile), 16 and
    37 tokens, from a non-zero running state, both gates, dv off the 32-row CTA tile."""
    lens = [8, 0, 1, 7, 9, 16, 37, 8]
    si = wl.make_seam_inputs(lens, 3, d, dv, kv_dtype=kv, gate=gate, g_lo=-0.3, seed=wl.seed_for(5, 1), device="cuda")
    S_ref, o_ref = _oracle_seam(si)
    e = si.enc
    host = [t.float().cpu().numpy() for t in (si.q, e.k, e.v, e.g, e.beta)]
    cu_h = e.cu_seqlens.cpu().numpy()
    S, o = hb.hypic_seam_window(si.S_in, si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)
    torch.cuda.synchronize()
    assert hb.hypic_last_launch_count() == 1
    check_E(S, S_ref, TOL_F32, "S_out")
    _check_o(o, o_ref, cu_h, TOL_F32, _typical_readout(si.S_in.cpu().numpy(), *host, cu_h, e.gate))
    assert torch.equal(S[1], si.S_in[1])  # empty window hands the state on unchanged
    # NULL S_in = zero state; in-place S; windows that skip tokens (cu_tokens[0] > 0, cu_tokens[R] < t_total)
    S0, o0 = hb.hypic_seam_window(None, si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)
    S0_ref, o0_ref = oracle.seam_window(None, *host, cu_h, gate=e.gate)
    check_E(S0, S0_ref, TOL_F32, "S_out (NULL S_in)")
    _check_o(o0, o0_ref, cu_h, TOL_F32, _typical_readout(None, *host, cu_h, e.gate))
    S2 = si.S_in.clone()
    hb.hypic_seam_window(S2, si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate, S_out=S2)
    assert torch.equal(S2, S)
    cu_in = torch.tensor([3, 11, 11, 30], dtype=torch.int32, device="cuda")
    S3, o3 = hb.hypic_seam_window(si.S_in[:3].contiguous(), si.q, e.k, e.v, e.g, e.beta, cu_in, e.gate)
    S3_ref, o3_ref = oracle.seam_window(si.S_in[:3].cpu().numpy(), *host, cu_in.cpu().numpy(), gate=e.gate)
    check_E(S3, S3_ref, TOL_F32, "S_out (inner windows)")
    _check_o(o3, o3_ref, cu_in.cpu().numpy(), TOL_F32,
             _typical_readout(si.S_in[:3].cpu().numpy(), *host, cu_in.cpu().numpy(), e.gate))


@pytest.mark.parametrize("g_lo", [-12.0, -40.0])
def test_seam_window_strong_decay(g_lo):
    """Scalar gate with a log-decay far below the benchmark's: some (g_lo = -12) or all (g_lo = -40) staged tiles
    fall outside the range in which the kernel runs its decay-folded form, so both forms and the switch between them
    are checked; the state in front of the window is forgotten almost completely."""
    lens = [8, 24, 5, 64]
    si = wl.make_seam_inputs(lens, 2, 128, 128, kv_dtype=torch.float32, g_lo=g_lo, seed=wl.seed_for(5, 3),
                             device="cuda")
    e = si.enc
    S_ref, o_ref = _oracle_seam(si)
    host = [t.float().cpu().numpy() for t in (si.q, e.k, e.v, e.g, e.beta)]
    cu_h = e.cu_seqlens.cpu().numpy()
    S, o = hb.hypic_seam_window(si.S_in, si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)
    torch.cuda.synchronize()
    check_E(S, S_ref, TOL_F32, "S_out")
    _check_o(o, o_ref, cu_h, TOL_F32, _typical_readout(si.S_in.cpu().numpy(), *host, cu_h, e.gate))


def test_seam_then_compose_equals_sequential_over_the_whole_segment():
    """PAPER.md:234 end to end: a segment whose first w tokens are left out of the cached tuple.  Seam step from the
    running state, then hypic_compose with the tuple of the remaining tokens, equals the token recurrence over the whole
    segment (oracle.sequential), and the seam outputs equal the recurrence's read-outs."""
    w, L, H, d = 8, 200, 2, 128
    full = wl.make_seam_inputs([L, L], H, d, d, kv_dtype=torch.float32, seed=wl.seed_for(5, 2), device="cuda")
    e = full.enc
    cu_seam = torch.tensor([0, w], dtype=torch.int32, device="cuda")
    # request 0 only: seam = tokens [0, w), cached rest = tokens [w, L)
    S_in = full.S_in[:1].contiguous()
    S_mid, o = hb.hypic_seam_window(S_in, full.q, e.k, e.v, e.g, e.beta, cu_seam, e.gate)
    cu_rest = torch.tensor([0, w, L], dtype=torch.int32, device="cuda")  # segment 0 = the seam (unused), 1 = the rest
    with impl_family(hb.HYPIC_IMPL_SIMT):
        E, T = hb.hypic_segment_encode(e.k[:L].contiguous(), e.v[:L].contiguous(), e.g[:L].contiguous(),
                                       e.beta[:L].contiguous(), cu_rest, e.gate)
        S = hb.hypic_compose(S_mid, E, T, torch.tensor([1], dtype=torch.int32, device="cuda"),
                             torch.tensor([0, 1], dtype=torch.int32, device="cuda"))
    torch.cuda.synchronize()
    c = e.cpu()
    S_ref = oracle.sequential(S_in.cpu().numpy(), c.k[:L], c.v[:L], c.g[:L], c.beta[:L],
                              np.array([0, L], dtype=np.int32), gate=c.gate)
    check_E(S, S_ref, TOL_F32, "S after seam + compose")
    _, o_ref = oracle.seam_window(S_in.cpu().numpy(), full.q.float().cpu().numpy(), c.k, c.v, c.g, c.beta,
                                  np.array([0, w], dtype=np.int32), gate=c.gate)
    _check_o(o, o_ref, np.array([0, w]), TOL_F32)


def test_seam_window_cfg_full_size_sampled_units():
    """The launch bench.py times (128 windows of 8 tokens, 32 heads, bf16): sampled (request, head) units."""
    si = wl.seam_cfg(device="cuda")
    e = si.enc
    S, o = hb.hypic_seam_window(si.S_in, si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)
    torch.cuda.synchronize()
    assert torch.isfinite(S).all() and torch.isfinite(o).all()
    cu = e.cu_seqlens.cpu().numpy()
    for r, h in _sample_units(128, 32, 8, 9):
        sl = slice(int(cu[r]), int(cu[r + 1]))
        f = lambda t: t[sl, h:h + 1].float().cpu().numpy()
        S_ref, o_ref = oracle.seam_window(si.S_in[r:r + 1, h:h + 1].cpu().numpy(), f(si.q), f(e.k), f(e.v), f(e.g),
                                          f(e.beta), np.array([0, sl.stop - sl.start], dtype=np.int32), gate=e.gate)
        check_E(S[r:r + 1, h:h + 1], S_ref, TOL_F32, "S_out")
        _check_o(o[sl, h:h + 1], o_ref, np.array([0, sl.stop - sl.start]), TOL_F32)


# ------------------------------------------------------------------------------------------------ scalar / diagonal families
def _check_tvec(t_gpu, t_ref, tol):
    t_gpu = t_gpu.cpu().numpy().astype(np.float64)
    assert np.isfinite(t_gpu).all()
    big = np.abs(t_ref) >= T_FLOOR_DIAG
    err = np.abs(t_gpu - t_ref)[big] / np.abs(t_ref)[big]
    worst = float(err.max()) if big.any() else 0.0
    assert worst <= tol, f"tvec: max rel. error {worst:.3e} > {tol:.1e}"
    if (~big).any():
        assert np.abs(t_gpu[~big]).max() <= 2 * T_FLOOR_DIAG
    return worst


T_FLOOR_DIAG = 1e-30  # reading S6 carried over: below this the fp32 tvec may flush; absolute check


def _diag_tol(inp, impl):
    """fp32 CUDA-core kernel: 1e-5 whatever the input dtype (inputs are exact); tcgen05 kernel (fp16 operands): 3e-3."""
    kv = hb.HYPIC_DT_BF16 if inp.k.dtype == torch.bfloat16 else hb.HYPIC_DT_F32
    hb.hypic_set_impl(impl)
    fam = hb.hypic_diag_encode_impl_for(inp.H, inp.dk, inp.dv, kv, inp.gate)
    hb.hypic_set_impl(hb.HYPIC_IMPL_AUTO)
    if fam < 0:
        pytest.skip("tensor family does not cover this shape")
    return TOL_BF16 if fam == hb.HYPIC_IMPL_TENSOR else TOL_F32


def gpu_diag_encode(inp, impl):
    with impl_family(impl):
        E, tv = hb.hypic_diag_encode(inp.k, inp.v, inp.g, inp.cu_seqlens, inp.gate)
        torch.cuda.synchronize()
    return E, tv


@pytest.mark.parametrize("name,impl", IMPLS)
@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
@pytest.mark.parametrize("kv,d,dv", [(torch.float32, 128, 128), (torch.bfloat16, 128, 128), (torch.float32, 64, 64),
                                     (torch.float32, 128, 40), (torch.bfloat16, 64, 100)])
def test_diag_encode_ragged_segments(name, impl, gate, kv, d, dv):
    """hypic_diag_encode (Table 1 scalar / diagonal families): ragged segments incl. empty, 1 token, chunk tails, for
    every kernel family that covers the shape."""
    lens = [70, 0, 1, 129, 16, 333, 15, 64, 200]
    inp = wl.make_encode_inputs(lens, 3, d, dv, kv_dtype=kv, gate=gate, g_lo=-0.2, seed=wl.seed_for(6, 1), device="cuda")
    tol = _diag_tol(inp, impl)
    E, tv = gpu_diag_encode(inp, impl)
    assert hb.hypic_last_launch_count() == 1
    c = inp.cpu()
    E_ref, t_ref = oracle.diag_encode(c.k, c.v, c.g, c.cu_seqlens, gate=c.gate)
    check_E(E, E_ref, tol, "E (diag family)")
    _check_tvec(tv, t_ref, TOL_F32)
    assert torch.all(E[1] == 0) and torch.all(tv[1] == 1)  # empty segment: E = 0, tvec = 1


def test_diag_encode_tensor_unsplit_schedule():
    """n_seg x H = 444 units: more than half a wave of 3 CTAs per SM, so the scalar-family kernel keeps one CTA per
    unit (the ragged-segment tests, 27 units, take its cluster-pair split): all units against the oracle."""
    lens = [70, 64, 1, 129, 130, 200, 63, 65, 0, 128, 192, 5]
    inp = wl.make_encode_inputs(lens, 37, 128, 128, kv_dtype=torch.bfloat16, g_lo=-0.2, seed=wl.seed_for(6, 6), device="cuda")
    E, tv = gpu_diag_encode(inp, hb.HYPIC_IMPL_TENSOR)
    c = inp.cpu()
    E_ref, t_ref = oracle.diag_encode(c.k, c.v, c.g, c.cu_seqlens, gate=c.gate)
    check_E(E, E_ref, TOL_BF16, "E (scalar family, unsplit)")
    _check_tvec(tv, t_ref, TOL_F32)


@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
def test_diag_encode_tensor_envelope_guard(gate):
    """The tcgen05 kernels of the scalar / diagonal families assume log-decays <= 0; a call that breaks this is counted
    (and the fp32 kernel handles it)."""
    inp = wl.make_encode_inputs([200, 64], 2, 128, 128, kv_dtype=torch.bfloat16, gate=gate, g_lo=-0.1,
                                seed=wl.seed_for(6, 7), device="cuda")
    before = hb.hypic_envelope_violation_count()
    gpu_diag_encode(inp, hb.HYPIC_IMPL_TENSOR)
    assert hb.hypic_envelope_violation_count() == before  # inside the envelope: nothing counted
    g_bad = inp.g.clone()
    g_bad[70] = 0.5  # growth instead of decay on one token
    bad = wl.EncodeInputs(k=inp.k, v=inp.v, g=g_bad, beta=inp.beta, cu_seqlens=inp.cu_seqlens, gate=inp.gate,
                          seg_lens=inp.seg_lens)
    gpu_diag_encode(bad, hb.HYPIC_IMPL_TENSOR)
    assert hb.hypic_envelope_violation_count() > before
    E, tv = gpu_diag_encode(bad, hb.HYPIC_IMPL_SIMT)  # the fp32 kernel has no such limit
    c = bad.cpu()
    E_ref, t_ref = oracle.diag_encode(c.k, c.v, c.g, c.cu_seqlens, gate=c.gate)
    check_E(E, E_ref, TOL_F32, "E (fp32 kernel, growing gate)")
    _check_tvec(tv, t_ref, TOL_F32)


def test_diag_encode_tensor_channel_gate_full_size_sampled_units():
    """Diagonal family (GLA) on the tcgen05 kernel at the bench shape (20 x 4096 tokens, H = 32, per-channel gate with a
    milder decay so that tvec stays representable): sampled units against the oracle, tvec of those units included."""
    inp = wl.make_encode_inputs([4096] * 20, 32, 128, 128, kv_dtype=torch.bfloat16, gate=wl.GATE_CHANNEL, g_lo=-0.01,
                                seed=wl.seed_for(6, 4), device="cuda")
    assert hb.hypic_diag_encode_impl_for(32, 128, 128, hb.HYPIC_DT_BF16, wl.GATE_CHANNEL) == hb.HYPIC_IMPL_TENSOR
    E, tv = gpu_diag_encode(inp, hb.HYPIC_IMPL_AUTO)
    assert torch.isfinite(E).all() and torch.isfinite(tv).all()
    for s, h in _sample_units(inp.n_seg, inp.H, 4, 12):
        u = inp.unit(s, h)
        E_ref, t_ref = oracle.diag_encode(u.k, u.v, u.g, u.cu_seqlens, gate=u.gate)
        check_E(E[s:s + 1, h:h + 1], E_ref, TOL_BF16, "E (diagonal family, tensor)")
        _check_tvec(tv[s:s + 1, h:h + 1], t_ref, TOL_F32)
    assert hb.hypic_debug_timeout_count() == 0


def test_diag_encode_tensor_cfg2_layer_sampled_units():
    """The launch bench.py times for the scalar family (one cfg2-shaped layer: 20 x 4096 tokens, H = 32, bf16) on the
    tcgen05 kernel: sampled (segment, head) units against the oracle, every tvec against the fp64 sum."""
    inp = wl.cfg2_layer(3, device="cuda")
    assert hb.hypic_diag_encode_impl_for(inp.H, 128, 128, hb.HYPIC_DT_BF16, wl.GATE_SCALAR) == hb.HYPIC_IMPL_TENSOR
    E, tv = gpu_diag_encode(inp, hb.HYPIC_IMPL_AUTO)
    assert torch.isfinite(E).all()
    cu = inp.cu_seqlens.cpu().numpy()
    t_ref = np.stack([np.exp(inp.g[cu[s]:cu[s + 1]].double().sum(0).cpu().numpy()) for s in range(inp.n_seg)])
    _check_tvec(tv, t_ref, TOL_F32)
    for s, h in _sample_units(inp.n_seg, inp.H, 5, 11):
        u = inp.unit(s, h)
        E_ref, _ = oracle.diag_encode(u.k, u.v, u.g, u.cu_seqlens, gate=u.gate)
        check_E(E[s:s + 1, h:h + 1], E_ref, TOL_BF16, "E (scalar family, tensor)")
    assert hb.hypic_debug_timeout_count() == 0


@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
def test_diag_encode_long_and_strong_decay(gate):
    """A 5,000-token segment at the benchmark's decay (tvec ~ e^-125: far below 1 but representable) and a segment with
    g ~ U(-30, 0): tvec underflows fp32 and E is set by the last few tokens only."""
    for lens, g_lo in (([5000, 300], -0.05), ([200, 64], -30.0)):
        inp = wl.make_encode_inputs(lens, 2, 128, 128, kv_dtype=torch.float32, gate=gate, g_lo=g_lo,
                                    seed=wl.seed_for(6, 2), device="cuda")
        E, tv = hb.hypic_diag_encode(inp.k, inp.v, inp.g, inp.cu_seqlens, inp.gate)
        c = inp.cpu()
        E_ref, t_ref = oracle.diag_encode(c.k, c.v, c.g, c.cu_seqlens, gate=c.gate)
        check_E(E, E_ref, TOL_F32, f"E (g_lo={g_lo})")
        _check_tvec(tv, t_ref, TOL_F32)


@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
@pytest.mark.parametrize("d", [128, 64])
def test_diag_compose_vs_oracle_and_sequential(gate, d):
    """hypic_diag_compose: lists of length 0, 1 and 40 with repeated, unsorted ids; NULL and in-place S; and
    encode -> compose in order equals the recurrence over the concatenation (oracle.diag_sequential)."""
    P, H = 24, 3
    lens = [int(x) for x in np.random.default_rng(61).integers(16, 65, P)]
    pin = wl.make_encode_inputs(lens, H, d, d, kv_dtype=torch.float32, gate=gate, g_lo=-0.01, seed=wl.seed_for(6, 3),
                                device="cuda")
    E, tv = hb.hypic_diag_encode(pin.k, pin.v, pin.g, pin.cu_seqlens, pin.gate)
    gen = torch.Generator().manual_seed(322)
    ids = torch.randint(0, P, (41,), generator=gen, dtype=torch.int32).cuda()
    cu = torch.tensor([0, 0, 1, 41], dtype=torch.int32, device="cuda")
    S_in = torch.randn(3, H, d, d, device="cuda")
    S = hb.hypic_diag_compose(S_in, E, tv, ids, cu)
    torch.cuda.synchronize()
    assert hb.hypic_last_launch_count() == 1
    ref = oracle.diag_compose(S_in.cpu().numpy(), E.cpu().numpy(), tv.cpu().numpy(), ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S, ref, TOL_F32, "S_out (diag compose)")
    assert torch.equal(S[0], S_in[0])
    S0 = hb.hypic_diag_compose(None, E, tv, ids, cu)
    ref0 = oracle.diag_compose(None, E.cpu().numpy(), tv.cpu().numpy(), ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S0, ref0, TOL_F32, "S_out (NULL S_in)")
    S3 = S_in.clone()
    hb.hypic_diag_compose(S3, E, tv, ids, cu, S_out=S3)
    assert torch.equal(S3, S)
    # fp16-stored end-states are exact inputs: fold of the stored values to the fp32-input tolerance
    Eh = hb.hypic_tuple_pack_f16(E)
    Sh = hb.hypic_diag_compose(S_in, Eh, tv, ids, cu)
    refh = oracle.diag_compose(S_in.cpu().numpy(), Eh.float().cpu().numpy(), tv.cpu().numpy(), ids.cpu().numpy(),
                               cu.cpu().numpy())
    check_E(Sh, refh, TOL_F32, "S_out (diag compose, fp16 end-states)")
    # all P segments in order from S_in[2] == the token recurrence over the concatenation
    all_ids = torch.arange(P, dtype=torch.int32, device="cuda")
    S_all = hb.hypic_diag_compose(S_in[2:3].contiguous(), E, tv, all_ids, torch.tensor([0, P], dtype=torch.int32,
                                                                                       device="cuda"))
    c = pin.cpu()
    seq = oracle.diag_sequential(S_in[2:3].cpu().numpy(), c.k, c.v, c.g, np.array([0, sum(lens)], dtype=np.int32),
                                 gate=c.gate)
    check_E(S_all, seq, TOL_F32, "encode -> compose vs sequential")


@pytest.mark.parametrize("dk,dv", [(24, 5), (40, 64), (256, 3), (1024, 2)])
@pytest.mark.parametrize("channel", [False, True])
def test_diag_compose_general_widths(dk, dv, channel):
    """hypic_diag_compose outside dk in {64, 128}: widths whose float4 count does not divide the CTA width take the
    kernel's general decay-vector path (one float4 of tvec per owned float4), the others the shared one."""
    P, H = 9, 2
    gen = torch.Generator().manual_seed(5100 + dk + dv)
    E = torch.randn((P, H, dv, dk), generator=gen).cuda()
    tv = (torch.rand((P, H, dk) if channel else (P, H), generator=gen) * 0.5 + 0.5).cuda()
    ids = torch.randint(0, P, (23,), generator=gen, dtype=torch.int32).cuda()
    cu = torch.tensor([0, 3, 3, 23], dtype=torch.int32, device="cuda")
    S_in = torch.randn((3, H, dv, dk), generator=gen).cuda()
    S = hb.hypic_diag_compose(S_in, E, tv, ids, cu)
    ref = oracle.diag_compose(S_in.cpu().numpy(), E.cpu().numpy(), tv.cpu().numpy(), ids.cpu().numpy(), cu.cpu().numpy())
    check_E(S, ref, TOL_F32, "S_out (diag compose, general width)")
    Eh = hb.hypic_tuple_pack_f16(E)
    Sh = hb.hypic_diag_compose(S_in, Eh, tv, ids, cu)
    refh = oracle.diag_compose(S_in.cpu().numpy(), Eh.float().cpu().numpy(), tv.cpu().numpy(), ids.cpu().numpy(),
                               cu.cpu().numpy())
    check_E(Sh, refh, TOL_F32, "S_out (diag compose, general width, fp16 end-states)")


def test_diag_compose_cfg4_lists_sampled_requests():
    """The launch bench.py times for the scalar family's compose (cfg4's request lists over a pool of 1,024 end-states,
    one scalar each), fp32 and fp16-stored end-states: sampled (request, head) chains against the oracle."""
    E = wl.cfg4_pool_E(device="cuda")
    gen = torch.Generator(device="cuda").manual_seed(wl.seed_for(6, 5))
    t_pool = torch.rand((E.shape[0], 32), device="cuda", generator=gen) * 0.5 + 0.5
    req = wl.cfg4_requests(device="cuda")
    S = hb.hypic_diag_compose(req.S_in, E, t_pool, req.seg_ids, req.cu_segs)
    Eh = hb.hypic_tuple_pack_f16(E)
    Sh = hb.hypic_diag_compose(req.S_in, Eh, t_pool, req.seg_ids, req.cu_segs)
    torch.cuda.synchronize()
    assert torch.isfinite(S).all() and torch.isfinite(Sh).all()
    ids_all, cu = req.seg_ids.cpu().numpy(), req.cu_segs.cpu().numpy()
    for r, h in _sample_units(128, 32, 6, 13):
        ids = torch.as_tensor(ids_all[cu[r]:cu[r + 1]], dtype=torch.long, device="cuda")
        n = len(ids)
        args = (np.arange(n, dtype=np.int32), np.array([0, n], dtype=np.int32))
        s0 = req.S_in[r:r + 1, h:h + 1].cpu().numpy()
        tp = t_pool[ids, h:h + 1].cpu().numpy()
        ref = oracle.diag_compose(s0, E[ids, h:h + 1].cpu().numpy(), tp, *args)
        check_E(S[r:r + 1, h:h + 1], ref, TOL_F32, "S_out (scalar family, cfg4 lists)")
        refh = oracle.diag_compose(s0, Eh[ids, h:h + 1].float().cpu().numpy(), tp, *args)
        check_E(Sh[r:r + 1, h:h + 1], refh, TOL_F32, "S_out (scalar family, fp16 end-states)")


# ------------------------------------------------------------------------------------------------ state RoPE re-rotation
def _inv_freq(dk, device="cuda"):
    return (10000.0 ** (-torch.arange(dk // 2, dtype=torch.float64) / (dk // 2))).float().to(device)


@pytest.mark.parametrize("dk,dv", [(128, 128), (64, 64), (128, 33), (8, 5), (32, 1024)])
def test_rope_compose_vs_oracle(dk, dv):
    """hypic_rope_compose (Eq. 7): lists of length 0, 1 and 40 with repeated, unsorted ids and start
    positions up to 2^20 (an fp32 angle would be off by 6e-2 rad there); NULL and in-place S; p = 0 equals
    hypic_diag_compose bit for bit up to the rotation's own rounding (cos = 1, sin = 0: exactly)."""
    P, H = 24, 3
    gen = torch.Generator().manual_seed(4100 + dk + dv)
    E = torch.randn((P, H, dv, dk), generator=gen).cuda()
    t_pool = (torch.rand((P, H), generator=gen) * 0.5 + 0.5).cuda()
    ids = torch.randint(0, P, (41,), generator=gen, dtype=torch.int32).cuda()
    pos = torch.randint(0, 1 << 20, (41,), generator=gen, dtype=torch.int32).cuda()
    cu = torch.tensor([0, 0, 1, 41], dtype=torch.int32, device="cuda")
    w = _inv_freq(dk)
    S_in = torch.randn((3, H, dv, dk), generator=gen).cuda()
    S = hb.hypic_rope_compose(S_in, E, t_pool, ids, cu, pos, w)
    torch.cuda.synchronize()
    assert hb.hypic_last_launch_count() == 2
    args = (E.cpu().numpy(), t_pool.cpu().numpy(), ids.cpu().numpy(), cu.cpu().numpy(), pos.cpu().numpy(),
            w.cpu().numpy())
    ref = oracle.rope_compose(S_in.cpu().numpy(), *args)
    check_E(S, ref, TOL_F32, "S_out (rope compose)")
    assert torch.equal(S[0], S_in[0])  # empty list: S_in is copied
    S0 = hb.hypic_rope_compose(None, E, t_pool, ids, cu, pos, w)
    check_E(S0, oracle.rope_compose(None, *args), TOL_F32, "S_out (NULL S_in)")
    S3 = S_in.clone()
    hb.hypic_rope_compose(S3, E, t_pool, ids, cu, pos, w, S_out=S3)
    assert torch.equal(S3, S)
    Sz = hb.hypic_rope_compose(S_in, E, t_pool, ids, cu, torch.zeros_like(pos), w)
    assert torch.equal(Sz, hb.hypic_diag_compose(S_in, E, t_pool, ids, cu))
    # fp16-stored end-states are exact inputs: the fold of the stored values, to the fp32-input tolerance
    Eh = hb.hypic_tuple_pack_f16(E)
    Sh = hb.hypic_rope_compose(S_in, Eh, t_pool, ids, cu, pos, w)
    refh = oracle.rope_compose(S_in.cpu().numpy(), Eh.float().cpu().numpy(), *args[1:])
    check_E(Sh, refh, TOL_F32, "S_out (rope compose, fp16 end-states)")
    # the rotation matters: without it the result is far from the reference
    assert oracle.rel_fro(hb.hypic_diag_compose(S_in, E, t_pool, ids, cu)[2].cpu().numpy(), ref[2]) > 1e-2


def test_rope_compose_end_to_end_equals_spliced_sequence():
    """Cache time: hypic_diag_encode of segments whose keys carry RoPE from position 0.  Reuse time: hypic_rope_compose
    with the global start positions.  Must equal the oracle's token recurrence over the spliced sequence whose keys carry
    RoPE at their global positions; bf16 k/v, so the bf16 tolerance."""
    H, d = 2, 128
    lens = [300, 64, 1000, 17, 555]
    gen = torch.Generator().manual_seed(4200)
    Ttot = sum(lens)
    k = torch.nn.functional.normalize(torch.randn((Ttot, H, d), generator=gen, dtype=torch.float64), dim=-1)
    v = torch.randn((Ttot, H, d), generator=gen).to(torch.bfloat16)
    g = -0.05 * torch.rand((Ttot, H), generator=gen)
    w = _inv_freq(d, "cpu")
    starts = np.concatenate([[0], np.cumsum(lens)[:-1]])

    def rope(kk, p0):  # keys at positions p0, p0 + 1, ...: pairs (c, c + d/2), angles in fp64
        ang = (torch.arange(kk.shape[0], dtype=torch.float64) + p0)[:, None] * w.double()[None, :]
        co, si = ang.cos()[:, None, :], ang.sin()[:, None, :]
        a, b = kk[..., :d // 2], kk[..., d // 2:]
        return torch.cat([a * co - b * si, a * si + b * co], dim=-1)

    k_local = torch.cat([rope(k[s:s + n], 0) for s, n in zip(starts, lens)]).to(torch.bfloat16)
    cu_tok = torch.tensor(np.concatenate([[0], np.cumsum(lens)]), dtype=torch.int32)
    E, tv = hb.hypic_diag_encode(k_local.cuda(), v.cuda(), g.cuda(), cu_tok.cuda(), wl.GATE_SCALAR)
    ids = torch.arange(len(lens), dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, len(lens)], dtype=torch.int32, device="cuda")
    S_in = torch.randn((1, H, d, d), generator=gen).cuda()
    S = hb.hypic_rope_compose(S_in, E, tv, ids, cu, torch.tensor(starts, dtype=torch.int32).cuda(), w.cuda())
    # reference: the global keys are the rotation of the SAME bf16-rounded local keys (rotation and rounding do not
    # commute, and the cached tuples were built from the rounded ones)
    k_ref = torch.cat([_rerotate(k_local[s:s + n].double(), int(s), w) for s, n in zip(starts, lens)])
    seq = oracle.diag_sequential(S_in.cpu().numpy(), k_ref.float().numpy(), v.float().numpy(), g.numpy(),
                                 np.array([0, Ttot], dtype=np.int32), wl.GATE_SCALAR)
    check_E(S, seq, TOL_BF16, "rope compose vs spliced sequence")


def _rerotate(k_rot0, shift, w):
    """Keys already rotated from position 0, moved to start position `shift` (R(a + t) = R(a) R(t)), fp64."""
    d = k_rot0.shape[-1]
    ang = shift * w.double()
    co, si = ang.cos()[None, None, :], ang.sin()[None, None, :]
    a, b = k_rot0[..., :d // 2], k_rot0[..., d // 2:]
    return torch.cat([a * co - b * si, a * si + b * co], dim=-1)


def test_rope_compose_cfg4_lists_sampled_requests():
    """cfg4's request lists over a pool of 1,024 end-states (one scalar each) with start positions up to 131,072: sampled
    (request, head) chains against the oracle."""
    E = wl.cfg4_pool_E(device="cuda")
    gen = torch.Generator(device="cuda").manual_seed(wl.seed_for(6, 7))
    t_pool = torch.rand((E.shape[0], 32), device="cuda", generator=gen) * 0.5 + 0.5
    req = wl.cfg4_requests(device="cuda")
    pos = torch.randint(0, 131072, (req.n_steps,), device="cuda", generator=gen, dtype=torch.int32)
    w = _inv_freq(128)
    S = hb.hypic_rope_compose(req.S_in, E, t_pool, req.seg_ids, req.cu_segs, pos, w)
    torch.cuda.synchronize()
    assert torch.isfinite(S).all()
    ids_all, cu, pos_all = req.seg_ids.cpu().numpy(), req.cu_segs.cpu().numpy(), pos.cpu().numpy()
    for r, h in _sample_units(128, 32, 6, 17):
        ids = torch.as_tensor(ids_all[cu[r]:cu[r + 1]], dtype=torch.long, device="cuda")
        n = len(ids)
        ref = oracle.rope_compose(req.S_in[r:r + 1, h:h + 1].cpu().numpy(), E[ids, h:h + 1].cpu().numpy(),
                                  t_pool[ids, h:h + 1].cpu().numpy(), np.arange(n, dtype=np.int32),
                                  np.array([0, n], dtype=np.int32), pos_all[cu[r]:cu[r + 1]], w.cpu().numpy())
        check_E(S[r:r + 1, h:h + 1], ref, TOL_F32, "S_out (rope compose, cfg4 lists)")


# ------------------------------------------------------------------------------------------------ forward + encode in one pass
@pytest.mark.parametrize("gate", [wl.GATE_SCALAR, wl.GATE_CHANNEL])
@pytest.mark.parametrize("kv,d,dv", [(torch.float32, 128, 128), (torch.bfloat16, 128, 128), (torch.float32, 64, 64),
                                     (torch.bfloat16, 128, 72), (torch.float32, 64, 33)])
def test_forward_encode_vs_oracle(gate, kv, d, dv):
    """hypic_forward_encode: one pass emits o, E and T.  o against the oracle's token recurrence with
    read-outs from the zero state (oracle.seam_window, pins W1-W4), (E, T) against oracle.segment_encode (pins P1-P10);
    ragged segments incl. empty and 1-token ones, dv off the 64-row tile so that a CTA straddles the E / T boundary."""
    lens = [70, 0, 1, 129, 16, 200]
    si = wl.make_seam_inputs(lens, 3, d, dv, kv_dtype=kv, gate=gate, g_lo=-0.1, seed=wl.seed_for(7, 1), device="cuda")
    e = si.enc
    o, E, T = hb.hypic_forward_encode(si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)
    torch.cuda.synchronize()
    assert hb.hypic_last_launch_count() == 1
    c = e.cpu()
    E_ref, T_ref = oracle.segment_encode(c.k, c.v, c.g, c.beta, c.cu_seqlens, gate=c.gate)
    check_E(E, E_ref, TOL_F32, "E (forward-encode)")
    check_T(T, T_ref, TOL_F32, "T (forward-encode)")
    host = [t.float().cpu().numpy() for t in (si.q, e.k, e.v, e.g, e.beta)]
    cu_h = e.cu_seqlens.cpu().numpy()
    S_ref, o_ref = oracle.seam_window(None, *host, cu_h, gate=e.gate)
    assert np.array_equal(S_ref, E_ref)  # the two oracle routes agree bit for bit on the end-state
    _check_o(o, o_ref, cu_h, TOL_F32, _typical_readout(None, *host, cu_h, e.gate))
    # and the tensor-family encode of the same inputs returns the same tuple within its own tolerance
    if kv == torch.bfloat16 and d == 128 and dv == 128:
        E2, T2 = hb.hypic_segment_encode(e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)
        check_E(E2, E.cpu().numpy(), TOL_BF16, "E (tensor family vs forward-encode)")
        check_T(T2, T.cpu().numpy(), TOL_BF16, "T (tensor family vs forward-encode)")


def test_forward_encode_bench_size_sampled_units():
    """hypic_forward_encode in the launch bench.py times (20 x 4096 tokens, H = 32, bf16 q/k/v): sampled (segment, head)
    units, o against oracle.seam_window from the zero state, (E, T) against oracle.segment_encode."""
    si = wl.make_seam_inputs([4096] * 20, 32, 128, 128, kv_dtype=torch.bfloat16, seed=wl.seed_for(7, 0), device="cuda")
    e = si.enc
    o, E, T = hb.hypic_forward_encode(si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)
    torch.cuda.synchronize()
    assert torch.isfinite(o).all() and torch.isfinite(E).all() and torch.isfinite(T).all()
    tol = TOL_F32  # fp32 arithmetic on both q/k/v dtypes
    for s, h in [(0, 0), (19, 31)] + _sample_units(20, 32, 6, 11):
        sl = slice(4096 * s, 4096 * (s + 1))
        f = lambda t: t[sl, h:h + 1].float().cpu().numpy()
        cu1 = np.array([0, 4096], dtype=np.int32)
        S_ref, o_ref = oracle.seam_window(None, f(si.q), f(e.k), f(e.v), f(e.g), f(e.beta), cu1, gate=e.gate)
        u = e.unit(s, h)
        E_ref, T_ref = oracle.segment_encode(u.k, u.v, u.g, u.beta, u.cu_seqlens, gate=u.gate)
        check_E(E[s:s + 1, h:h + 1], E_ref, tol, "E (forward-encode)")
        check_T(T[s:s + 1, h:h + 1], T_ref, tol, "T (forward-encode)")
        _check_o(o[sl, h:h + 1], o_ref, cu1, tol, _typical_readout(None, f(si.q), f(e.k), f(e.v), f(e.g), f(e.beta), cu1, e.gate))


def test_compose_interleaved_heads_every_unit():
    """R x H = 40 x 8 = 320 chains: enough for the tensor-family compose kernels to fold heads h, h + 1 of a request as
    two interleaved chains of one CTA (below 2 x 148 units they run one chain per CTA).  Every unit against the oracle,
    fp32 pools and fp16-stored pools; lists of length 0..12 with repeated, unsorted ids; NULL S_in as well."""
    P, H, d, R = 16, 8, 128, 40
    pin = wl.near_unit_pool_inputs(P, H, device="cuda", d=d, kv_dtype=torch.float32)
    with impl_family(hb.HYPIC_IMPL_SIMT):
        E, T = hb.hypic_segment_encode(pin.k, pin.v, pin.g, pin.beta, pin.cu_seqlens, pin.gate)
    req = wl.make_compose_requests(R, P, H, d, d, n_lo=0, n_hi=12, seed=78, device="cuda", s_in_std=1.0)
    ids, cu = req.seg_ids.cpu().numpy(), req.cu_segs.cpu().numpy()
    for S_in in (req.S_in, None):
        s_host = None if S_in is None else S_in.cpu().numpy()
        S = gpu_compose(S_in, E, T, req.seg_ids, req.cu_segs, hb.HYPIC_IMPL_TENSOR)
        check_E(S, oracle.compose(s_host, E.cpu().numpy(), T.cpu().numpy(), ids, cu), TOL_F32, "S_out (fp32 pools)")
        Eh, Th = hb.hypic_tuple_pack_f16(E), hb.hypic_tuple_pack_f16(T)
        Sh = hb.hypic_compose_f16(S_in, Eh, Th, req.seg_ids, req.cu_segs)
        torch.cuda.synchronize()
        check_E(Sh, oracle.compose(s_host, Eh.float().cpu().numpy(), Th.float().cpu().numpy(), ids, cu), TOL_F32,
                "S_out (fp16 pools)")
    assert hb.hypic_debug_timeout_count() == 0
