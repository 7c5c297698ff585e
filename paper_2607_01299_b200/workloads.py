"""Seeded synthetic inputs for the HYPIC hot path (segment encode + composition).

This module holds NONE of the method's arithmetic: it only draws random tensors with the shapes, sizes and
value distributions of ``BASELINE.json:configs`` (cfg0..cfg4, 0-indexed; recipe in DESIGN.md "Input recipe").
Both sides of every parity test consume the same bits: tensors are generated once (on whatever device is
asked for) and the oracle is handed a host copy.  Neither ``oracle/`` nor the CUDA path is imported here.

Stand-in statement: the paper measures on Qwen3.5/Ring hybrid models over RAG/agent traces;
neither weights nor traces are available, so these inputs take only their shapes (segments of 256-4k tokens,
PAPER.md:321; dk=dv=128, 32 heads) and the distributions BASELINE.json fixes.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence

import torch

GATE_SCALAR = 0
GATE_CHANNEL = 1

BASE_SEED = 20260701  # DESIGN.md reading S4: seed = BASE_SEED + 1000*cfg + layer


def seed_for(cfg: int, layer: int = 0) -> int:
    return BASE_SEED + 1000 * cfg + layer


@dataclasses.dataclass
class EncodeInputs:
    """Packed inputs of hypic_segment_encode (layouts of include/hypic.h)."""

    k: torch.Tensor  # [Ttot,H,dk]  bf16 or fp32
    v: torch.Tensor  # [Ttot,H,dv]  same dtype as k
    g: torch.Tensor  # [Ttot,H] (scalar gate) or [Ttot,H,dk] (per-channel gate), fp32 log-decay
    beta: torch.Tensor  # [Ttot,H] fp32
    cu_seqlens: torch.Tensor  # int32 [n_seg+1]
    gate: int
    seg_lens: List[int]

    @property
    def n_seg(self) -> int:
        return len(self.seg_lens)

    @property
    def t_total(self) -> int:
        return int(self.k.shape[0])

    @property
    def H(self) -> int:
        return int(self.k.shape[1])

    @property
    def dk(self) -> int:
        return int(self.k.shape[2])

    @property
    def dv(self) -> int:
        return int(self.v.shape[2])

    def unit(self, seg: int, head: int) -> "EncodeInputs":
        """The single (segment, head) unit as a 1-segment, 1-head problem on the CPU (for sampled oracle checks)."""
        t0 = sum(self.seg_lens[:seg])
        t1 = t0 + self.seg_lens[seg]
        sl = slice(t0, t1)
        hs = slice(head, head + 1)
        return EncodeInputs(
            k=self.k[sl, hs].cpu().contiguous(), v=self.v[sl, hs].cpu().contiguous(),
            g=self.g[sl, hs].cpu().contiguous(), beta=self.beta[sl, hs].cpu().contiguous(),
            cu_seqlens=torch.tensor([0, t1 - t0], dtype=torch.int32), gate=self.gate, seg_lens=[t1 - t0])

    def cpu(self) -> "EncodeInputs":
        return EncodeInputs(self.k.cpu(), self.v.cpu(), self.g.cpu(), self.beta.cpu(), self.cu_seqlens.cpu(),
                            self.gate, list(self.seg_lens))


def make_encode_inputs(seg_lens: Sequence[int], H: int, dk: int, dv: int, *, kv_dtype: torch.dtype,
                       gate: int = GATE_SCALAR, g_lo: float = -0.05, beta_kind: str = "sigmoid",
                       seed: int = BASE_SEED, device: str = "cpu") -> EncodeInputs:
    """k ~ N(0,1) L2-normalised per (token, head) in fp32 then cast (reading S1); v ~ N(0,1);
    g ~ U(g_lo, 0) fp32; beta = sigmoid(N(0,1)) or U(0,1) fp32."""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    ttot = int(sum(seg_lens))
    k = torch.randn((ttot, H, dk), generator=gen, device=device, dtype=torch.float32)
    k = k / k.norm(dim=-1, keepdim=True).clamp_min(1e-20)
    k = k.to(kv_dtype)
    v = torch.randn((ttot, H, dv), generator=gen, device=device, dtype=torch.float32).to(kv_dtype)
    gshape = (ttot, H) if gate == GATE_SCALAR else (ttot, H, dk)
    g = torch.rand(gshape, generator=gen, device=device, dtype=torch.float32) * float(g_lo)  # U(g_lo, 0]
    if beta_kind == "sigmoid":
        beta = torch.sigmoid(torch.randn((ttot, H), generator=gen, device=device, dtype=torch.float32))
    elif beta_kind == "uniform":
        beta = torch.rand((ttot, H), generator=gen, device=device, dtype=torch.float32)
    else:
        raise ValueError(beta_kind)
    cu = torch.zeros(len(seg_lens) + 1, dtype=torch.int32)
    cu[1:] = torch.cumsum(torch.tensor(list(seg_lens), dtype=torch.int64), 0).to(torch.int32)
    return EncodeInputs(k=k, v=v, g=g, beta=beta, cu_seqlens=cu.to(device), gate=gate, seg_lens=list(seg_lens))


# ---------------------------------------------------------------------------------------------------------
# The five BASELINE.json configs (0-indexed).  ``scale`` shrinks token counts for quick tests; scale=1 is the
# configuration as written.
# ---------------------------------------------------------------------------------------------------------

def cfg0(device: str = "cpu") -> EncodeInputs:
    """cfg0: 1 head, dk=dv=64, fp32; two segments of 128 tokens; g ~ U(-0.1,0); beta ~ U(0,1)."""
    return make_encode_inputs([128, 128], 1, 64, 64, kv_dtype=torch.float32, g_lo=-0.1, beta_kind="uniform",
                              seed=seed_for(0), device=device)


def cfg0_s_in(device: str = "cpu") -> torch.Tensor:
    """cfg0's non-zero start state S_in ~ N(0, 0.1) (std 0.1, reading S2): [1 request, 1 head, 64, 64] fp32."""
    gen = torch.Generator(device=device)
    gen.manual_seed(seed_for(0, 500))
    return 0.1 * torch.randn((1, 1, 64, 64), generator=gen, device=device, dtype=torch.float32)


def cfg1(device: str = "cpu", seg_len: int = 2048, n_seg: int = 4, H: int = 16) -> EncodeInputs:
    """cfg1: H=16, dk=dv=128, 4 segments x 2048 tokens, bf16 k/v, g ~ U(-0.05,0), beta = sigmoid(N(0,1))."""
    return make_encode_inputs([seg_len] * n_seg, H, 128, 128, kv_dtype=torch.bfloat16, g_lo=-0.05,
                              beta_kind="sigmoid", seed=seed_for(1), device=device)


def cfg2_layer(layer: int, device: str = "cpu", seg_len: int = 4096, n_seg: int = 20, H: int = 32) -> EncodeInputs:
    """cfg2: one of 36 independent layers: 20 segments x 4096 tokens, H=32, dk=dv=128, cfg1's distributions
    (reading S3), seeded per layer."""
    return make_encode_inputs([seg_len] * n_seg, H, 128, 128, kv_dtype=torch.bfloat16, g_lo=-0.05,
                              beta_kind="sigmoid", seed=seed_for(2, layer), device=device)


def fold_layers(layers: List[EncodeInputs]) -> EncodeInputs:
    """Independent layers with the same packing, folded into the head axis ("fold layers into the
    head axis when the caller's layout is [Ttot, layers*H, d]"): head l*H + h of the result is head h of layers[l].
    Pure layout: values are copied, none is recomputed.  One call then covers all the folded layers."""
    first = layers[0]
    for x in layers[1:]:
        if x.seg_lens != first.seg_lens or x.gate != first.gate or x.k.dtype != first.k.dtype:
            raise ValueError("fold_layers: layers must share segment lengths, gate kind and dtype")
    cat = lambda ts: torch.cat(ts, dim=1).contiguous()
    return EncodeInputs(k=cat([x.k for x in layers]), v=cat([x.v for x in layers]), g=cat([x.g for x in layers]),
                        beta=cat([x.beta for x in layers]), cu_seqlens=first.cu_seqlens, gate=first.gate,
                        seg_lens=list(first.seg_lens))


def cfg3_seg_lens(n_seg: int = 64, lo: int = 512, hi: int = 16384) -> List[int]:
    gen = torch.Generator()
    gen.manual_seed(seed_for(3, 999))
    return [int(x) for x in torch.randint(lo, hi + 1, (n_seg,), generator=gen)]


def cfg3(device: str = "cpu", n_seg: int = 64, lo: int = 512, hi: int = 16384, H: int = 32) -> EncodeInputs:
    """cfg3: 64 varlen segments ~ U[512,16384], H=32, dk=dv=128, bf16 k/v, per-channel g ~ U(-0.05,0) fp32."""
    return make_encode_inputs(cfg3_seg_lens(n_seg, lo, hi), H, 128, 128, kv_dtype=torch.bfloat16,
                              gate=GATE_CHANNEL, g_lo=-0.05, beta_kind="sigmoid", seed=seed_for(3), device=device)


@dataclasses.dataclass
class ComposeRequests:
    """Request lists of hypic_compose: ids of request r are seg_ids[cu_segs[r]:cu_segs[r+1]], in order."""

    seg_ids: torch.Tensor  # int32 [sum n_r]
    cu_segs: torch.Tensor  # int32 [R+1]
    S_in: Optional[torch.Tensor]  # [R,H,dv,dk] fp32 or None

    @property
    def R(self) -> int:
        return int(self.cu_segs.shape[0]) - 1

    @property
    def n_steps(self) -> int:
        return int(self.seg_ids.shape[0])


def make_compose_requests(R: int, P: int, H: int, dk: int, dv: int, *, n_lo: int, n_hi: int, seed: int,
                          device: str = "cpu", s_in_std: Optional[float] = 1.0) -> ComposeRequests:
    """n_r ~ U{n_lo..n_hi}; ids = first n_r entries of a seeded random permutation of 0..P-1 (unsorted, so the
    order matters -- reading S5); S_in ~ N(0, s_in_std) fp32, or None."""
    gen = torch.Generator()
    gen.manual_seed(int(seed))
    ids, cu = [], [0]
    for _ in range(R):
        n = int(torch.randint(n_lo, n_hi + 1, (1,), generator=gen))
        n = min(n, P)
        ids.append(torch.randperm(P, generator=gen)[:n].to(torch.int32))
        cu.append(cu[-1] + n)
    seg_ids = torch.cat(ids) if ids else torch.zeros(0, dtype=torch.int32)
    S_in = None
    if s_in_std is not None:
        dgen = torch.Generator(device=device)
        dgen.manual_seed(int(seed) + 7)
        S_in = float(s_in_std) * torch.randn((R, H, dv, dk), generator=dgen, device=device, dtype=torch.float32)
    return ComposeRequests(seg_ids=seg_ids.to(device), cu_segs=torch.tensor(cu, dtype=torch.int32, device=device),
                           S_in=S_in)


def cfg4_pool_inputs(P: int = 1024, H: int = 32, seg_len: int = 256, device: str = "cpu", layer: int = 0) -> EncodeInputs:
    """Token inputs whose encoded T forms cfg4's pool: P random seg_len-token segments with cfg1's
    distributions ("T taken from encoding random 256-token segments")."""
    return make_encode_inputs([seg_len] * P, H, 128, 128, kv_dtype=torch.bfloat16, g_lo=-0.05, beta_kind="sigmoid",
                              seed=seed_for(4, layer), device=device)


def cfg4_pool_E(P: int = 1024, H: int = 32, device: str = "cpu", layer: int = 0) -> torch.Tensor:
    """cfg4's E pool: E ~ N(0,1) fp32 [P,H,128,128]."""
    gen = torch.Generator(device=device)
    gen.manual_seed(seed_for(4, layer) + 333)
    return torch.randn((P, H, 128, 128), generator=gen, device=device, dtype=torch.float32)


def cfg4_requests(R: int = 128, P: int = 1024, H: int = 32, device: str = "cpu", layer: int = 0) -> ComposeRequests:
    """cfg4: 128 requests, each a random ordered subset of 16..64 pool segments, S_in ~ N(0,1)."""
    return make_compose_requests(R, P, H, 128, 128, n_lo=16, n_hi=64, seed=seed_for(4, layer) + 555, device=device,
                                 s_in_std=1.0)


def near_unit_pool_inputs(P: int, H: int, device: str = "cpu", d: int = 128, kv_dtype: torch.dtype = torch.bfloat16,
                          seed_off: int = 0) -> EncodeInputs:
    """Parity-only compose case (reading S9): T from short segments (16..64 tokens, g ~ U(-0.01,0)) so that
    ||T||_F = O(1..10) and the S.T product is not negligible next to E."""
    gen = torch.Generator()
    gen.manual_seed(seed_for(4, 77) + seed_off)
    lens = [int(x) for x in torch.randint(16, 65, (P,), generator=gen)]
    return make_encode_inputs(lens, H, d, d, kv_dtype=kv_dtype, g_lo=-0.01, beta_kind="sigmoid",
                              seed=seed_for(4, 78) + seed_off, device=device)


# ---------------------------------------------------------------------------------------------------------
# Seam-window step: R windows of w tokens each (w = 8 default),
# one per request, with queries and a non-zero running state in front of every window.
# ---------------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class SeamInputs:
    enc: EncodeInputs        # k, v, g, beta of the window tokens; enc.cu_seqlens = cu_tokens of the R windows
    q: torch.Tensor          # [Ttot, H, dk], L2-normalised like k (the layers normalise q and k alike), kv dtype
    S_in: torch.Tensor       # [R, H, dv, dk] fp32 ~ N(0, 1): stands in for the composed state in front of the seam


def make_seam_inputs(win_lens: Sequence[int], H: int, dk: int, dv: int, *, kv_dtype: torch.dtype,
                     gate: int = GATE_SCALAR, g_lo: float = -0.05, seed: int = BASE_SEED,
                     device: str = "cpu") -> SeamInputs:
    enc = make_encode_inputs(win_lens, H, dk, dv, kv_dtype=kv_dtype, gate=gate, g_lo=g_lo, seed=seed, device=device)
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed) + 500_000)
    q = torch.randn((enc.t_total, H, dk), generator=gen, device=device, dtype=torch.float32)
    q = (q / q.norm(dim=-1, keepdim=True).clamp_min(1e-20)).to(kv_dtype)
    S_in = torch.randn((len(win_lens), H, dv, dk), generator=gen, device=device, dtype=torch.float32)
    return SeamInputs(enc=enc, q=q, S_in=S_in)


def seam_cfg(R: int = 128, H: int = 32, w: int = 8, device: str = "cpu", layer: int = 0) -> SeamInputs:
    """One seam per request of cfg4's batch (R = 128 requests, H = 32 heads, dk = dv = 128, bf16 q/k/v, w = 8)."""
    return make_seam_inputs([w] * R, H, 128, 128, kv_dtype=torch.bfloat16, seed=seed_for(5, layer), device=device)
