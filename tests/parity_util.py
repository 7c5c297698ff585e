"""Helpers shared by the GPU parity tests: error metric of BASELINE.json:north_star and sampled-unit oracles."""
from __future__ import annotations

import numpy as np
import torch

import oracle

TOL_F32 = 1e-5   # fp32 k/v, or compose fed fp32 pools (north_star)
TOL_BF16 = 3e-3  # bf16 k/v with fp32 accumulation (north_star)
T_FLOOR = 1e-30  # DESIGN.md reading S6: below this ||T_ref||_F the check on T is absolute


def per_unit_rel(x: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """Relative Frobenius error per leading-2-dims unit ([N,H,rows,cols] -> [N,H])."""
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    num = np.sqrt(((x - ref) ** 2).sum(axis=(-1, -2)))
    den = np.sqrt((ref ** 2).sum(axis=(-1, -2)))
    return np.where(den > 0, num / np.maximum(den, 1e-300), num)


def check_E(E_gpu, E_ref, tol, what="E"):
    E_gpu = E_gpu.detach().cpu().numpy() if isinstance(E_gpu, torch.Tensor) else E_gpu
    assert np.isfinite(E_gpu).all(), f"{what}: non-finite values"
    err = per_unit_rel(E_gpu, E_ref)
    den = np.sqrt((np.asarray(E_ref) ** 2).sum(axis=(-1, -2)))
    # units whose reference is exactly zero (empty segments) must be exactly zero
    zero = den == 0
    if zero.any():
        assert np.abs(E_gpu[zero]).max() == 0.0, f"{what}: expected exact zeros"
    worst = float(err[~zero].max()) if (~zero).any() else 0.0
    assert worst <= tol, f"{what}: max per-unit rel. Frobenius error {worst:.3e} > {tol:.1e}"
    return worst


def check_T(T_gpu, T_ref, tol, what="T"):
    """Reading S6: relative where ||T_ref||_F >= 1e-30, else ||T_gpu||_F <= 1e-30."""
    T_gpu = T_gpu.detach().cpu().numpy() if isinstance(T_gpu, torch.Tensor) else T_gpu
    assert np.isfinite(T_gpu).all(), f"{what}: non-finite values"
    den = np.sqrt((np.asarray(T_ref, dtype=np.float64) ** 2).sum(axis=(-1, -2)))
    err = per_unit_rel(T_gpu, T_ref)
    big = den >= T_FLOOR
    worst = float(err[big].max()) if big.any() else 0.0
    assert worst <= tol, f"{what}: max per-unit rel. Frobenius error {worst:.3e} > {tol:.1e}"
    if (~big).any():
        gn = np.sqrt((T_gpu.astype(np.float64) ** 2).sum(axis=(-1, -2)))[~big]
        assert gn.max() <= T_FLOOR, f"{what}: underflowed units must stay below {T_FLOOR}: {gn.max():.3e}"
    return worst


def oracle_encode(inp):
    """fp64 oracle (E, T) for an EncodeInputs (any device)."""
    c = inp.cpu()
    return oracle.segment_encode(c.k, c.v, c.g, c.beta, c.cu_seqlens, gate=c.gate)


def oracle_encode_units(inp, units):
    """Oracle (E, T) for sampled (segment, head) units of a large EncodeInputs: lists of [dv,dk], [dk,dk]."""
    Es, Ts = [], []
    for s, h in units:
        u = inp.unit(s, h)
        E, T = oracle.segment_encode(u.k, u.v, u.g, u.beta, u.cu_seqlens, gate=u.gate)
        Es.append(E[0, 0])
        Ts.append(T[0, 0])
    return np.stack(Es)[:, None], np.stack(Ts)[:, None]


def oracle_encode_units_batched(inp, units):
    """As oracle_encode_units, but the sampled units go to the oracle in ONE call (packed as len(units) one-head
    segments), so that its OpenMP loop over independent units uses every host core: [n,1,dv,dk], [n,1,dk,dk]."""
    cu = np.concatenate([[0], np.cumsum(inp.seg_lens)]).astype(np.int64)
    ks, vs, gs, bs, lens = [], [], [], [], []
    for s, h in units:
        sl = slice(int(cu[s]), int(cu[s + 1]))
        ks.append(inp.k[sl, h:h + 1].cpu())
        vs.append(inp.v[sl, h:h + 1].cpu())
        gs.append(inp.g[sl, h:h + 1].cpu())
        bs.append(inp.beta[sl, h:h + 1].cpu())
        lens.append(int(cu[s + 1] - cu[s]))
    cu_u = torch.tensor(np.concatenate([[0], np.cumsum(lens)]), dtype=torch.int32)
    E, T = oracle.segment_encode(torch.cat(ks), torch.cat(vs), torch.cat(gs), torch.cat(bs), cu_u, gate=inp.gate)
    return E, T


def oracle_compose_units(S_in, E_pool, T_pool, seg_ids, cu_segs, units):
    """Oracle composed state for sampled (request, head) units of a large compose problem: [n,1,dv,dk]."""
    ids_all = seg_ids.cpu().numpy()
    cu = cu_segs.cpu().numpy()
    outs = []
    for r, h in units:
        ids = ids_all[cu[r]:cu[r + 1]]
        idx = torch.as_tensor(ids, dtype=torch.long, device=E_pool.device)
        Ep = E_pool[idx, h].cpu().numpy()[:, None]
        Tp = T_pool[idx, h].cpu().numpy()[:, None]
        s0 = None if S_in is None else S_in[r, h].cpu().numpy().astype(np.float64)[None, None]
        out = oracle.compose(s0, Ep, Tp, np.arange(len(ids), dtype=np.int32), np.array([0, len(ids)], dtype=np.int32))
        outs.append(out[0, 0])
    return np.stack(outs)[:, None]
