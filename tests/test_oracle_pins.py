"""Pins for the fp64 oracle (CPU only).  Each test checks ``oracle/`` against something the paper or the
mathematics fixes -- a printed value, a closed form, an invariant, a brute force written along a DIFFERENT
route (explicit matrices in the PAPER's column convention) -- never against a retyped copy of its own loop.

P-numbers refer to DESIGN.md "Oracle pins".
"""
import os

import numpy as np
import pytest

import oracle
from oracle import GATE_CHANNEL, GATE_SCALAR

RNG = np.random.default_rng(20260701)


def _rand_inputs(L, H, dk, dv, gate, rng, g_lo=-0.1, normalise=True, beta_hi=1.0):
    k = rng.standard_normal((L, H, dk)).astype(np.float32)
    if normalise:
        k /= np.linalg.norm(k, axis=-1, keepdims=True)
    v = rng.standard_normal((L, H, dv)).astype(np.float32)
    gshape = (L, H) if gate == GATE_SCALAR else (L, H, dk)
    g = (rng.random(gshape) * g_lo).astype(np.float32)
    beta = (rng.random((L, H)) * beta_hi).astype(np.float32)
    return k, v, g, beta


def _cu(lens):
    return np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)


# ---------------------------------------------------------------------------------------------------------
# P4: brute force from explicitly built matrices, in the PAPER's convention (column vectors, left-multiplying;
# PAPER.md:84 Eq. 2, Table 1), then transposed.  Also pins reading A1 (row vs column convention),
# G1 (u_i = beta k v^T), G3 (ordered product, later tokens on the left) and A3 (decay-then-erase order).
# ---------------------------------------------------------------------------------------------------------
def _paper_convention_bruteforce(k, v, g, beta, gate, S0_paper=None):
    """k:[L,dk] v:[L,dv] float64.  Returns (S_L paper [dk,dv], T_C paper [dk,dk])."""
    L, dk = k.shape
    dv = v.shape[1]
    I = np.eye(dk)
    S = np.zeros((dk, dv)) if S0_paper is None else S0_paper.copy()
    Tc = np.eye(dk)
    for i in range(L):
        ki = k[i][:, None]
        if gate == GATE_SCALAR:  # GDN: T_i = g_i (I - beta_i k_i k_i^T)
            Ti = np.exp(g[i]) * (I - beta[i] * (ki @ ki.T))
        else:  # KDA: T_i = (I - beta_i k_i k_i^T) diag(g_i)
            Ti = (I - beta[i] * (ki @ ki.T)) @ np.diag(np.exp(g[i]))
        ui = beta[i] * (ki @ v[i][None, :])
        S = Ti @ S + ui
        Tc = Ti @ Tc  # prod_{i=n}^{1}: later tokens on the left
    return S, Tc


@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
@pytest.mark.parametrize("L,dk,dv", [(4, 4, 4), (4, 4, 3), (7, 5, 6)])
def test_P4_bruteforce_paper_convention(gate, L, dk, dv):
    rng = np.random.default_rng(100 + L + dk + 7 * gate)
    k, v, g, beta = _rand_inputs(L, 1, dk, dv, gate, rng, g_lo=-0.5, normalise=False)
    E, T = oracle.segment_encode(k, v, g, beta, _cu([L]), gate)
    S_p, T_p = _paper_convention_bruteforce(k[:, 0].astype(np.float64), v[:, 0].astype(np.float64),
                                            g[:, 0].astype(np.float64), beta[:, 0].astype(np.float64), gate)
    np.testing.assert_allclose(E[0, 0], S_p.T, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(T[0, 0], T_p.T, rtol=1e-12, atol=1e-14)


def test_P4_unrolled_sum_of_products():
    """E = sum_t beta_t v_t k_t^T A_{t+1}...A_L and T = A_1 A_2 A_3 A_4 with A_t = alpha_t (I - beta_t k_t k_t^T)
    (row convention, Eq. 2 unrolled): 4 tokens, dk = dv = 4, matrices built explicitly."""
    rng = np.random.default_rng(4)
    L, d = 4, 4
    k, v, g, beta = _rand_inputs(L, 1, d, d, GATE_SCALAR, rng, g_lo=-0.3, normalise=False)
    E, T = oracle.segment_encode(k, v, g, beta, _cu([L]))
    kk, vv = k[:, 0].astype(np.float64), v[:, 0].astype(np.float64)
    A = [np.exp(float(g[t, 0])) * (np.eye(d) - float(beta[t, 0]) * np.outer(kk[t], kk[t])) for t in range(L)]
    T_ref = A[0] @ A[1] @ A[2] @ A[3]
    E_ref = np.zeros((d, d))
    for t in range(L):
        # the write enters AFTER token t's own decay/erase: S_t = S_{t-1} A_t + beta_t v_t k_t^T
        tail = np.eye(d)
        for s in range(t + 1, L):
            tail = tail @ A[s]
        E_ref += float(beta[t, 0]) * np.outer(vv[t], kk[t]) @ tail
    np.testing.assert_allclose(T[0, 0], T_ref, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(E[0, 0], E_ref, rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------------------------------------------------
# P1: compose(encode(C_1..C_n); S_in) == sequential recurrence over the concatenation (Eq. 4/6, Insight 1)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
@pytest.mark.parametrize("lens", [[128, 128], [1, 63, 64, 65, 7], [50, 0, 33], [200]])
@pytest.mark.parametrize("zero_start", [True, False])
def test_P1_compose_equals_sequential(gate, lens, zero_start):
    rng = np.random.default_rng(sum(lens) + 13 * gate + zero_start)
    H, dk, dv = 2, 16, 12
    L = sum(lens)
    k, v, g, beta = _rand_inputs(L, H, dk, dv, gate, rng)
    E, T = oracle.segment_encode(k, v, g, beta, _cu(lens), gate)
    S_in = None if zero_start else 0.1 * rng.standard_normal((1, H, dv, dk))
    ids = np.arange(len(lens), dtype=np.int32)
    S_comp = oracle.compose(S_in, E, T, ids, np.array([0, len(lens)], dtype=np.int32))
    S_seq = oracle.sequential(S_in, k, v, g, beta, np.array([0, L], dtype=np.int32), gate)
    assert oracle.rel_fro(S_comp, S_seq) < 1e-12


def test_P1_compose_is_order_sensitive():
    """Non-commutativity (reading S10): swapping two segments changes the result, and the swapped composition
    equals the sequential recurrence over the swapped token order."""
    rng = np.random.default_rng(77)
    H, d = 1, 8
    lens = [20, 30]
    k, v, g, beta = _rand_inputs(50, H, d, d, GATE_SCALAR, rng)
    E, T = oracle.segment_encode(k, v, g, beta, _cu(lens))
    cu1 = np.array([0, 2], dtype=np.int32)
    S01 = oracle.compose(None, E, T, np.array([0, 1], dtype=np.int32), cu1)
    S10 = oracle.compose(None, E, T, np.array([1, 0], dtype=np.int32), cu1)
    assert oracle.rel_fro(S10, S01) > 1e-3
    perm = np.concatenate([np.arange(20, 50), np.arange(0, 20)])
    S_seq = oracle.sequential(None, k[perm], v[perm], g[perm], beta[perm], np.array([0, 50], dtype=np.int32))
    assert oracle.rel_fro(S10, S_seq) < 1e-12


# ---------------------------------------------------------------------------------------------------------
# P2: beta = 0  =>  T = (prod alpha) I  (scalar) / diag(prod_t alpha_{t,c}) (per-channel), E = 0  (Table 3)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
def test_P2_beta_zero_closed_form(gate):
    rng = np.random.default_rng(2 + gate)
    L, H, dk, dv = 90, 3, 8, 6
    k, v, g, beta = _rand_inputs(L, H, dk, dv, gate, rng)
    beta[:] = 0.0
    E, T = oracle.segment_encode(k, v, g, beta, _cu([L]), gate)
    assert np.all(E == 0.0)
    for h in range(H):
        if gate == GATE_SCALAR:
            ref = np.exp(g[:, h].astype(np.float64).sum()) * np.eye(dk)
        else:
            ref = np.diag(np.exp(g[:, h].astype(np.float64).sum(axis=0)))
        np.testing.assert_allclose(T[0, h], ref, rtol=1e-12, atol=1e-300)


# ---------------------------------------------------------------------------------------------------------
# P3: Table 2's nine printed values from the oracle's T with constant decay, beta = 0
# ---------------------------------------------------------------------------------------------------------
def test_P3_table2_printed_values(golden_dir):
    rows = []
    with open(os.path.join(golden_dir, "table2_naive_addition_error.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                e, n, val = line.split()
                rows.append((int(e), int(n), float(val)))
    assert len(rows) == 9
    rng = np.random.default_rng(3)
    dk, dv = 8, 5
    S1 = rng.standard_normal((dv, dk))  # stands for S_{C1|0}
    for e, n, printed in rows:
        gamma = 1.0 - 2.0 ** e
        k, v, _, beta = _rand_inputs(n, 1, dk, dv, GATE_SCALAR, rng)
        beta[:] = 0.0  # RetNet: T_i = gamma I, no delta-rule term
        g = np.full((n, 1), np.log(gamma), dtype=np.float32)
        gamma_eff = float(np.exp(np.float64(g[0, 0])))  # the fp32-rounded log-decay the oracle actually sees
        _, T = oracle.segment_encode(k, v, g, beta, _cu([n]))
        delta = S1 @ T[0, 0] - S1  # (T_{C2} - I) applied to S_{C1|0}, Eq. 5 (row convention)
        ratio = np.linalg.norm(delta) / np.linalg.norm(S1)
        assert abs(ratio - (1.0 - gamma_eff ** n)) < 1e-12
        assert abs(ratio - printed) <= 5.1e-4, (e, n, ratio, printed)  # printed to 3 decimals


# ---------------------------------------------------------------------------------------------------------
# P5: T(C1 C2) = T(C1) T(C2);  E(C1 C2) = E(C1) T(C2) + E(C2)     (Eq. 4; independence of prefix)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
def test_P5_concatenation_law(gate):
    rng = np.random.default_rng(5 + gate)
    H, dk, dv = 2, 10, 7
    l1, l2 = 37, 91
    k, v, g, beta = _rand_inputs(l1 + l2, H, dk, dv, gate, rng)
    E12, T12 = oracle.segment_encode(k, v, g, beta, _cu([l1 + l2]), gate)
    E, T = oracle.segment_encode(k, v, g, beta, _cu([l1, l2]), gate)
    for h in range(H):
        np.testing.assert_allclose(T12[0, h], T[0, h] @ T[1, h], rtol=1e-11, atol=1e-14)
        np.testing.assert_allclose(E12[0, h], E[0, h] @ T[1, h] + E[1, h], rtol=1e-11, atol=1e-13)
    # T and E of the second segment do not depend on what precedes it
    E2, T2 = oracle.segment_encode(k[l1:], v[l1:], g[l1:], beta[l1:], _cu([l2]), gate)
    assert np.array_equal(E2[0], E[1]) and np.array_equal(T2[0], T[1])


# ---------------------------------------------------------------------------------------------------------
# P6: orthonormal keys k_t = e_{pi(t)} (L <= dk): factors commute; closed form
# ---------------------------------------------------------------------------------------------------------
def test_P6_orthonormal_keys_closed_form():
    rng = np.random.default_rng(6)
    dk, dv, L = 12, 9, 8
    pi = rng.permutation(dk)[:L]
    k = np.zeros((L, 1, dk), dtype=np.float32)
    k[np.arange(L), 0, pi] = 1.0
    v = rng.standard_normal((L, 1, dv)).astype(np.float32)
    g = (rng.random((L, 1)) * -0.3).astype(np.float32)
    beta = rng.random((L, 1)).astype(np.float32)
    E, T = oracle.segment_encode(k, v, g, beta, _cu([L]))
    a = np.exp(g[:, 0].astype(np.float64))
    b = beta[:, 0].astype(np.float64)
    T_ref = np.eye(dk)
    for t in range(L):
        T_ref[pi[t], pi[t]] -= b[t]
    T_ref *= a.prod()
    E_ref = np.zeros((dv, dk))
    for t in range(L):
        E_ref[:, pi[t]] += b[t] * a[t + 1:].prod() * v[t, 0].astype(np.float64)
    np.testing.assert_allclose(T[0, 0], T_ref, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(E[0, 0], E_ref, rtol=1e-12, atol=1e-15)


# ---------------------------------------------------------------------------------------------------------
# P7: one repeated unit key, alpha = 1: T = I - (1 - prod(1-beta_t)) k k^T; constant v: E k = (1 - prod(1-beta)) v
# ---------------------------------------------------------------------------------------------------------
def test_P7_repeated_key_lms_convergence():
    rng = np.random.default_rng(7)
    dk, dv, L = 9, 5, 25
    kd = rng.standard_normal(dk)
    kd /= np.linalg.norm(kd)
    k32 = kd.astype(np.float32)
    k = np.tile(k32[None, None, :], (L, 1, 1))
    v0 = rng.standard_normal(dv).astype(np.float32)
    v = np.tile(v0[None, None, :], (L, 1, 1))
    g = np.zeros((L, 1), dtype=np.float32)
    beta = (rng.random((L, 1)) * 0.9).astype(np.float32)
    E, T = oracle.segment_encode(k, v, g, beta, _cu([L]))
    kk = k32.astype(np.float64)
    n2 = kk @ kk  # fp32-rounded key is not exactly unit: use the general closed form with |k|^2
    resid = np.prod(1.0 - beta[:, 0].astype(np.float64) * n2)
    T_ref = np.eye(dk) - (1.0 - resid) * np.outer(kk, kk) / n2
    np.testing.assert_allclose(T[0, 0], T_ref, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(E[0, 0] @ kk, (1.0 - resid) * v0.astype(np.float64), rtol=1e-12, atol=1e-15)


# ---------------------------------------------------------------------------------------------------------
# P8: the paper's two-invocation route: the E recurrence with dv := dk, v = 0, S_0 = I gives T
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
def test_P8_two_invocation_route(gate):
    rng = np.random.default_rng(8 + gate)
    L, H, dk = 70, 2, 12
    k, _, g, beta = _rand_inputs(L, H, dk, dk, gate, rng)
    v0 = np.zeros((L, H, dk), dtype=np.float32)
    _, T = oracle.segment_encode(k, v0, g, beta, _cu([L]), gate)
    S_I = np.tile(np.eye(dk)[None, None], (1, H, 1, 1))
    S_end = oracle.sequential(S_I, k, v0, g, beta, np.array([0, L], dtype=np.int32), gate)
    np.testing.assert_allclose(S_end[0], T[0], rtol=1e-13, atol=1e-300)


# ---------------------------------------------------------------------------------------------------------
# P9: det T = prod_t alpha_t^{dk} (1 - beta_t |k_t|^2)   (per-channel: prod_t (prod_c alpha_{t,c}) (1 - beta_t |k_t|^2))
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
def test_P9_determinant(gate):
    rng = np.random.default_rng(9 + gate)
    L, dk, dv = 11, 6, 4
    k, v, g, beta = _rand_inputs(L, 1, dk, dv, gate, rng, normalise=False, beta_hi=0.1)
    _, T = oracle.segment_encode(k, v, g, beta, _cu([L]), gate)
    sign, logdet = np.linalg.slogdet(T[0, 0])
    k64, b64, g64 = k[:, 0].astype(np.float64), beta[:, 0].astype(np.float64), g[:, 0].astype(np.float64)
    fac = 1.0 - b64 * (k64 * k64).sum(-1)
    log_ref = np.log(np.abs(fac)).sum() + (dk * g64.sum() if gate == GATE_SCALAR else g64.sum())
    assert sign == np.prod(np.sign(fac))
    assert abs(logdet - log_ref) < 1e-10


# ---------------------------------------------------------------------------------------------------------
# P10: beta_L = 1, |k_L| = 1  =>  T k_L = 0 and E k_L = v_L;  ||T||_2 <= prod alpha_t for beta |k|^2 in [0,2]
# ---------------------------------------------------------------------------------------------------------
def test_P10_last_pair_recalled_and_contraction():
    rng = np.random.default_rng(10)
    L, dk, dv = 40, 8, 6
    k, v, g, beta = _rand_inputs(L, 1, dk, dv, GATE_SCALAR, rng)
    k[-1, 0] = 0.0
    k[-1, 0, 3] = 1.0  # exactly unit in fp32
    beta[-1, 0] = 1.0
    E, T = oracle.segment_encode(k, v, g, beta, _cu([L]))
    kL = k[-1, 0].astype(np.float64)
    assert np.abs(T[0, 0] @ kL).max() < 1e-15
    np.testing.assert_allclose(E[0, 0] @ kL, v[-1, 0].astype(np.float64), rtol=1e-13)
    # contraction bound on a run with beta |k|^2 in (0, 1]
    k2, v2, g2, b2 = _rand_inputs(L, 1, dk, dv, GATE_SCALAR, rng)
    _, T2 = oracle.segment_encode(k2, v2, g2, b2, _cu([L]))
    assert np.linalg.norm(T2[0, 0], 2) <= np.exp(g2.astype(np.float64).sum()) * (1 + 1e-6)


# ---------------------------------------------------------------------------------------------------------
# Degenerate cases and layout
# ---------------------------------------------------------------------------------------------------------
def test_empty_segment_is_identity():
    rng = np.random.default_rng(11)
    k, v, g, beta = _rand_inputs(5, 2, 4, 3, GATE_SCALAR, rng)
    E, T = oracle.segment_encode(k, v, g, beta, _cu([0, 5, 0]))
    for s in (0, 2):
        assert np.all(E[s] == 0)
        assert np.array_equal(T[s], np.tile(np.eye(4)[None], (2, 1, 1)))


def test_compose_empty_list_copies_s_in_and_f32_pools_match_f64():
    rng = np.random.default_rng(12)
    P, H, dk, dv = 5, 2, 6, 4
    E = rng.standard_normal((P, H, dv, dk)).astype(np.float32)
    T = (rng.standard_normal((P, H, dk, dk)) * 0.3).astype(np.float32)
    S_in = rng.standard_normal((2, H, dv, dk))
    ids = np.array([3, 1, 4], dtype=np.int32)
    cu = np.array([0, 0, 3], dtype=np.int32)
    out = oracle.compose(S_in, E, T, ids, cu)
    assert np.array_equal(out[0], S_in[0])  # empty list
    out64 = oracle.compose(S_in, E.astype(np.float64), T.astype(np.float64), ids, cu)
    assert np.array_equal(out, out64)
    # explicit fold with numpy matmul for request 1
    for h in range(H):
        S = S_in[1, h].copy()
        for i in ids:
            S = S @ T[i, h].astype(np.float64) + E[i, h].astype(np.float64)
        np.testing.assert_allclose(out[1, h], S, rtol=1e-13, atol=1e-15)


def test_heads_and_segments_are_independent_units():
    """Layout pin: unit (s,h) of a packed multi-head batch equals the same tokens run alone (catches a wrong
    stride / index in the packed [Ttot,H,d] addressing)."""
    rng = np.random.default_rng(13)
    lens, H, dk, dv = [9, 17, 4], 3, 6, 5
    k, v, g, beta = _rand_inputs(sum(lens), H, dk, dv, GATE_CHANNEL, rng)
    E, T = oracle.segment_encode(k, v, g, beta, _cu(lens), GATE_CHANNEL)
    cu = _cu(lens)
    for s in range(len(lens)):
        for h in range(H):
            sl = slice(cu[s], cu[s + 1])
            e1, t1 = oracle.segment_encode(k[sl, h:h + 1], v[sl, h:h + 1], g[sl, h:h + 1], beta[sl, h:h + 1],
                                           _cu([lens[s]]), GATE_CHANNEL)
            assert np.array_equal(e1[0, 0], E[s, h]) and np.array_equal(t1[0, 0], T[s, h])


# ---------------------------------------------------------------------------------------------------------
# W-pins: seam-window step (Fig. 8): token recurrence from a non-zero running state with the
# per-token read-out o_i = q_i^T S_i (Eq. 2).
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
@pytest.mark.parametrize("w,dk,dv", [(1, 4, 4), (3, 4, 5), (8, 6, 3)])
def test_W1_seam_bruteforce_paper_convention(gate, w, dk, dv):
    """Explicit T_i, u_i matrices in the paper's column convention, S_0 = S_in^T, o_i = q_i^T S_i read AFTER the
    update of token i (a read before the update, a transposed S or q on the wrong side all fail)."""
    rng = np.random.default_rng(4100 + w + dk + 7 * gate)
    k, v, g, beta = _rand_inputs(w, 1, dk, dv, gate, rng, g_lo=-0.5, normalise=False)
    q = rng.standard_normal((w, 1, dk)).astype(np.float32)
    S_in = rng.standard_normal((1, 1, dv, dk))
    S_out, o = oracle.seam_window(S_in, q, k, v, g, beta, _cu([w]), gate)
    for i in range(w):
        S_p, _ = _paper_convention_bruteforce(k[:i + 1, 0].astype(np.float64), v[:i + 1, 0].astype(np.float64),
                                              g[:i + 1, 0].astype(np.float64), beta[:i + 1, 0].astype(np.float64),
                                              gate, S0_paper=S_in[0, 0].T)
        o_p = q[i, 0].astype(np.float64)[None, :] @ S_p  # 1 x dv
        np.testing.assert_allclose(o[i, 0], o_p[0], rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(S_out[0, 0], S_p.T, rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
def test_W2_seam_via_composition_law(gate):
    """the seam's own (T, S) inserted into Eq. 6.  For every prefix 1..t of the window,
    o_t = (S_in T_{1..t} + E_{1..t}) q_t with (E, T) from segment_encode + compose (pinned by P1-P10), and the
    state handed on equals hypic_oracle_sequential's."""
    rng = np.random.default_rng(4200 + gate)
    w, H, dk, dv = 8, 2, 16, 12
    k, v, g, beta = _rand_inputs(w, H, dk, dv, gate, rng, g_lo=-0.3)
    q = rng.standard_normal((w, H, dk)).astype(np.float32)
    S_in = rng.standard_normal((1, H, dv, dk))
    S_out, o = oracle.seam_window(S_in, q, k, v, g, beta, _cu([w]), gate)
    for t in range(1, w + 1):
        E, T = oracle.segment_encode(k[:t], v[:t], g[:t], beta[:t], _cu([t]), gate)
        S_t = oracle.compose(S_in, E, T, np.array([0], dtype=np.int32), _cu([1]))
        o_t = np.einsum("hic,hc->hi", S_t[0], q[t - 1].astype(np.float64))
        np.testing.assert_allclose(o[t - 1], o_t, rtol=1e-11, atol=1e-12)
    S_seq = oracle.sequential(S_in, k, v, g, beta, _cu([w]), gate)
    np.testing.assert_allclose(S_out, S_seq, rtol=0, atol=0)


@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
def test_W3_seam_recall_closed_form(gate):
    """Delta rule closed form: with beta_t ||k_t||^2 = 1 the write makes S_t k_t = v_t whatever S_{t-1} and the
    gate were, so q_t = k_t reads back o_t = v_t exactly (a read-out taken before the write fails)."""
    rng = np.random.default_rng(4300 + gate)
    w, H, dk, dv = 8, 3, 8, 5
    k, v, g, _ = _rand_inputs(w, H, dk, dv, gate, rng, g_lo=-1.0, normalise=False)
    beta = (1.0 / np.sum(k.astype(np.float64) ** 2, axis=-1))
    beta32 = beta.astype(np.float32)
    S_in = 10.0 * rng.standard_normal((1, H, dv, dk))
    _, o = oracle.seam_window(S_in, k, k, v, g, beta32, _cu([w]), gate)
    # beta is rounded to float32, so beta ||k||^2 = 1 + O(2^-24): the residual is that relative error times |S k|
    np.testing.assert_allclose(o, v.astype(np.float64), rtol=0, atol=2e-5)


def test_W4_seam_requests_are_independent_and_empty_window_copies():
    rng = np.random.default_rng(4400)
    H, dk, dv = 2, 8, 8
    lens = [3, 0, 8, 1]
    ttot = sum(lens) + 2  # two trailing tokens belong to no request
    k, v, g, beta = _rand_inputs(ttot, H, dk, dv, GATE_SCALAR, rng)
    q = rng.standard_normal((ttot, H, dk)).astype(np.float32)
    S_in = rng.standard_normal((len(lens), H, dv, dk))
    cu = _cu(lens)
    S_out, o = oracle.seam_window(S_in, q, k, v, g, beta, cu, GATE_SCALAR)
    assert np.array_equal(S_out[1], S_in[1])  # empty window: state handed on unchanged
    assert np.all(np.isnan(o[cu[-1]:])) and not np.any(np.isnan(o[:cu[-1]]))
    for r, L in enumerate(lens):
        sl = slice(int(cu[r]), int(cu[r + 1]))
        S_r, o_r = oracle.seam_window(S_in[r:r + 1], q[sl], k[sl], v[sl], g[sl], beta[sl], _cu([L]), GATE_SCALAR)
        assert np.array_equal(S_r[0], S_out[r]) and np.array_equal(o_r, o[sl])
    # S_in = None is the zero state
    S0, o0 = oracle.seam_window(None, q, k, v, g, beta, cu, GATE_SCALAR)
    Sz, oz = oracle.seam_window(np.zeros_like(S_in), q, k, v, g, beta, cu, GATE_SCALAR)
    assert np.array_equal(S0, Sz) and np.array_equal(o0[:cu[-1]], oz[:cu[-1]])


# ---------------------------------------------------------------------------------------------------------
# D-pins: scalar and diagonal families (Table 1; Table 3):
# T_i = a_i I or diag(g_i), u_i = k_i v_i^T, T_C kept as one scalar / one dk-vector.
# ---------------------------------------------------------------------------------------------------------
def _paper_convention_diag(k, v, g, gate, S0_paper=None):
    """Explicit T_i matrices in the paper's column convention: S_i = T_i S_{i-1} + k_i v_i^T (S: dk x dv)."""
    L, dk = k.shape
    S = np.zeros((dk, v.shape[1])) if S0_paper is None else S0_paper.copy()
    Tc = np.eye(dk)
    for i in range(L):
        Ti = np.exp(g[i]) * np.eye(dk) if gate == GATE_SCALAR else np.diag(np.exp(g[i]))
        S = Ti @ S + k[i][:, None] @ v[i][None, :]
        Tc = Ti @ Tc
    return S, Tc


@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
@pytest.mark.parametrize("L,dk,dv", [(1, 3, 2), (5, 4, 4), (9, 5, 7)])
def test_D1_diag_bruteforce_paper_convention(gate, L, dk, dv):
    rng = np.random.default_rng(5100 + L + 3 * dk + 7 * gate)
    k, v, g, _ = _rand_inputs(L, 1, dk, dv, gate, rng, g_lo=-0.7, normalise=False)
    E, tvec = oracle.diag_encode(k, v, g, _cu([L]), gate)
    S_p, T_p = _paper_convention_diag(k[:, 0].astype(np.float64), v[:, 0].astype(np.float64),
                                      g[:, 0].astype(np.float64), gate)
    np.testing.assert_allclose(E[0, 0], S_p.T, rtol=1e-12, atol=1e-14)
    full = tvec[0, 0] * np.eye(dk) if gate == GATE_SCALAR else np.diag(tvec[0, 0])
    np.testing.assert_allclose(full, T_p.T, rtol=1e-12, atol=0)
    # from a non-zero state
    S0 = rng.standard_normal((1, 1, dv, dk))
    S = oracle.diag_sequential(S0, k, v, g, _cu([L]), gate)
    S_p2, _ = _paper_convention_diag(k[:, 0].astype(np.float64), v[:, 0].astype(np.float64),
                                     g[:, 0].astype(np.float64), gate, S0_paper=S0[0, 0].T)
    np.testing.assert_allclose(S[0, 0], S_p2.T, rtol=1e-12, atol=1e-14)


def test_D2_table3_closed_forms():
    """Table 3: RetNet / Lightning T_C = gamma^{|C|} I, Mamba2 (prod_t a_t) I, GLA diag(prod_t g_t);
    and E = sum_t (prod_{s>t} a_s) v_t k_t^T written as one weighted matrix product."""
    rng = np.random.default_rng(5200)
    L, H, dk, dv = 50, 2, 6, 4
    k, v, _, _ = _rand_inputs(L, H, dk, dv, GATE_SCALAR, rng, normalise=False)
    gamma = 1.0 - 2.0 ** -5
    g_const = np.full((L, H), np.log(gamma), dtype=np.float32)
    g_eff = np.exp(np.float64(g_const[0, 0]))  # the decay the oracle actually sees (fp32-rounded log)
    E, t = oracle.diag_encode(k, v, g_const, _cu([L]), GATE_SCALAR)
    np.testing.assert_allclose(t, g_eff ** L, rtol=1e-12)
    w = g_eff ** (L - 1 - np.arange(L))  # token t is decayed by the L-1-t tokens after it
    for h in range(H):
        ref = (v[:, h].astype(np.float64) * w[:, None]).T @ k[:, h].astype(np.float64)
        np.testing.assert_allclose(E[0, h], ref, rtol=1e-11, atol=1e-13)
    g_s = (rng.random((L, H)) * -0.4).astype(np.float32)
    _, t_s = oracle.diag_encode(k, v, g_s, _cu([L]), GATE_SCALAR)
    np.testing.assert_allclose(t_s[0], np.exp(g_s.astype(np.float64).sum(0)), rtol=1e-12)
    g_c = (rng.random((L, H, dk)) * -0.4).astype(np.float32)
    E_c, t_c = oracle.diag_encode(k, v, g_c, _cu([L]), GATE_CHANNEL)
    np.testing.assert_allclose(t_c[0], np.exp(g_c.astype(np.float64).sum(0)), rtol=1e-12)
    G = np.cumsum(g_c.astype(np.float64), axis=0)
    wt = np.exp(G[-1][None] - G)  # [L,H,dk]: decay of channel c from token t to the end
    for h in range(H):
        ref = v[:, h].astype(np.float64).T @ (k[:, h].astype(np.float64) * wt[:, h])
        np.testing.assert_allclose(E_c[0, h], ref, rtol=1e-11, atol=1e-13)


@pytest.mark.parametrize("gate", [GATE_SCALAR, GATE_CHANNEL])
@pytest.mark.parametrize("zero_start", [True, False])
def test_D3_diag_compose_equals_sequential(gate, zero_start):
    """PAPER.md:118 Eq. 4 / PAPER.md:182 Eq. 6 for the compressed transitions: composing the cached (E, tvec) of the
    segments in order reproduces the recurrence over the concatenation; a different order does not."""
    rng = np.random.default_rng(5300 + gate)
    lens = [17, 1, 40, 0, 9]
    H, dk, dv = 2, 8, 5
    k, v, g, _ = _rand_inputs(sum(lens), H, dk, dv, gate, rng, g_lo=-0.2, normalise=False)
    E, t = oracle.diag_encode(k, v, g, _cu(lens), gate)
    S0 = None if zero_start else rng.standard_normal((1, H, dv, dk))
    ids = np.arange(len(lens), dtype=np.int32)
    S = oracle.diag_compose(S0, E, t, ids, _cu([len(lens)]))
    S_seq = oracle.diag_sequential(S0, k, v, g, _cu([sum(lens)]), gate)
    np.testing.assert_allclose(S, S_seq, rtol=1e-11, atol=1e-13)
    S_rev = oracle.diag_compose(S0, E, t, ids[::-1].copy(), _cu([len(lens)]))
    assert oracle.rel_fro(S_rev, S_seq) > 1e-3


def test_D4_table2_printed_values_with_real_suffix(golden_dir):
    """Table 2 on the scalar family itself: adding the two zero-start end-states instead of composing
    them leaves the error Delta = (1 - gamma^{|C2|}) S_{C1|0}, whatever the suffix holds."""
    rows = []
    with open(os.path.join(golden_dir, "table2_naive_addition_error.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                e, n, val = line.split()
                rows.append((int(e), int(n), float(val)))
    rng = np.random.default_rng(5400)
    H, dk, dv, l1 = 1, 6, 4, 30
    for e, n, printed in rows:
        gamma = 1.0 - 2.0 ** e
        k, v, _, _ = _rand_inputs(l1 + n, H, dk, dv, GATE_SCALAR, rng, normalise=False)
        g = np.full((l1 + n, H), np.log(gamma), dtype=np.float32)
        E, t = oracle.diag_encode(k, v, g, _cu([l1, n]), GATE_SCALAR)
        S_true = oracle.diag_compose(None, E, t, np.array([0, 1], dtype=np.int32), _cu([2]))
        delta = (E[0] + E[1]) - S_true[0]
        ratio = np.linalg.norm(delta) / np.linalg.norm(E[0])
        assert abs(ratio - printed) <= 5.1e-4, (e, n, ratio, printed)


def test_D5_diag_family_is_the_dense_family_without_erasure():
    """Cross-family check against the pinned dense oracle: the dense token step with the erase term removed
    (T_i = g_i (I - beta_i k_i k_i^T) -> g_i I) is linear in v, so for ORTHONORMAL keys in a segment
    (k_s . k_t = 0: nothing is ever erased) and beta = 1 the dense end-state equals the scalar family's, and the dense
    T equals tvec (I - sum_t k_t k_t^T)."""
    rng = np.random.default_rng(5500)
    L, dk, dv = 6, 8, 5
    q, _ = np.linalg.qr(rng.standard_normal((dk, dk)))
    k = q[:L][:, None, :].astype(np.float32)  # float32 rounding leaves k_s . k_t ~ 1e-8
    v = rng.standard_normal((L, 1, dv)).astype(np.float32)
    g = (rng.random((L, 1)) * -0.5).astype(np.float32)
    beta = np.ones((L, 1), dtype=np.float32)
    E_dense, T_dense = oracle.segment_encode(k, v, g, beta, _cu([L]), GATE_SCALAR)
    E_diag, t = oracle.diag_encode(k, v, g, _cu([L]), GATE_SCALAR)
    np.testing.assert_allclose(E_dense, E_diag, rtol=0, atol=1e-6)
    kk = k[:, 0].astype(np.float64)
    np.testing.assert_allclose(T_dense[0, 0], t[0, 0] * (np.eye(dk) - kk.T @ kk), rtol=0, atol=1e-6)


# ------------------------------------------------------------------------------------------------ state RoPE re-rotation
def _rope_matrix(p, inv_freq):
    """R(p) as an explicit dense dk x dk matrix of 2 x 2 rotation blocks on the pairs (c, c + dk/2): a different code
    path from the oracle's column loop.  k_rot = R(p) k."""
    half = len(inv_freq)
    Rm = np.zeros((2 * half, 2 * half))
    for c in range(half):
        phi = p * inv_freq[c]
        Rm[c, c] = Rm[c + half, c + half] = np.cos(phi)
        Rm[c, c + half] = -np.sin(phi)
        Rm[c + half, c] = np.sin(phi)
    return Rm


def _rope_keys(k, start, inv_freq):
    """Keys of one stretch of tokens with RoPE applied at positions start, start + 1, ... (float64 [L,H,dk])."""
    out = np.empty(k.shape, dtype=np.float64)
    for t in range(k.shape[0]):
        out[t] = k[t].astype(np.float64) @ _rope_matrix(start + t, inv_freq).T
    return out


def test_R1_eq7_rerotation_of_a_cached_end_state():
    """PAPER.md:212 Eq. 7: S_{C|b} = R(b - a) S_{C|a} for a scalar transition.  The end state of a segment whose keys
    were rotated from start position b equals the re-rotation (oracle.rope_compose, one step, t = 1) of the end state
    computed from start position a; the rotation preserves the Frobenius norm; p = 0 is the identity."""
    rng = np.random.default_rng(7100)
    L, H, dk, dv = 23, 2, 8, 5
    inv_freq = 10000.0 ** (-np.arange(dk // 2) / (dk // 2))
    k, v, g, _ = _rand_inputs(L, H, dk, dv, GATE_SCALAR, rng, g_lo=-0.2, normalise=False)
    a, b = 3, 1000
    E_a, t_a = oracle.diag_encode(_rope_keys(k, a, inv_freq).astype(np.float32), v, g, _cu([L]), GATE_SCALAR)
    E_b, _ = oracle.diag_encode(_rope_keys(k, b, inv_freq).astype(np.float32), v, g, _cu([L]), GATE_SCALAR)
    one = np.ones_like(t_a)
    ids, cu = np.zeros(1, dtype=np.int32), _cu([1])
    rot = oracle.rope_compose(None, E_a, one, ids, cu, np.array([b - a], dtype=np.int32), inv_freq)
    assert oracle.rel_fro(rot[0], E_b[0]) < 5e-7  # keys pass through float32 on the way into diag_encode
    assert oracle.rel_fro(rot[0], E_a[0]) > 1e-2  # and the rotation is not a no-op
    np.testing.assert_allclose(np.linalg.norm(rot), np.linalg.norm(E_a), rtol=1e-13)
    same = oracle.rope_compose(None, E_a, one, ids, cu, np.zeros(1, dtype=np.int32), inv_freq)
    np.testing.assert_array_equal(same[0], E_a[0])
    # dense-matrix form of the same statement: every row of E is rotated like a key
    for h in range(H):
        np.testing.assert_allclose(rot[0, h], E_a[0, h] @ _rope_matrix(b - a, inv_freq).T, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("zero_start", [True, False])
def test_R2_rope_compose_equals_sequential_with_global_positions(zero_start):
    """replacing each S_{C_i|0} by R(p_i) S_{C_i|0} in Eq. 6, p_i = the segment's global start position,
    reproduces the recurrence over the spliced sequence whose keys carry RoPE at their global positions."""
    rng = np.random.default_rng(7200)
    lens = [17, 1, 40, 0, 9]
    H, dk, dv = 2, 8, 5
    inv_freq = 10000.0 ** (-np.arange(dk // 2) / (dk // 2))
    k, v, g, _ = _rand_inputs(sum(lens), H, dk, dv, GATE_SCALAR, rng, g_lo=-0.2, normalise=False)
    starts = np.concatenate([[0], np.cumsum(lens)[:-1]]).astype(np.int32)
    k_local = np.concatenate([_rope_keys(k[s:s + n], 0, inv_freq) for s, n in zip(starts, lens)]).astype(np.float32)
    k_global = _rope_keys(k, 0, inv_freq).astype(np.float32)
    E, t = oracle.diag_encode(k_local, v, g, _cu(lens), GATE_SCALAR)  # position-independent tuples (cache time)
    S0 = None if zero_start else rng.standard_normal((1, H, dv, dk))
    ids = np.arange(len(lens), dtype=np.int32)
    S = oracle.rope_compose(S0, E, t, ids, _cu([len(lens)]), starts, inv_freq)
    S_seq = oracle.diag_sequential(S0, k_global, v, g, _cu([sum(lens)]), GATE_SCALAR)
    assert oracle.rel_fro(S, S_seq) < 5e-7
    S_norot = oracle.diag_compose(S0, E, t, ids, _cu([len(lens)]))
    assert oracle.rel_fro(S_norot, S_seq) > 1e-2  # without the re-rotation the cached states do not splice


def test_R3_rope_compose_at_position_zero_is_diag_compose():
    """p_i = 0 for every entry: R(0) = I, so the routine reduces to the scalar family's plain composition."""
    rng = np.random.default_rng(7300)
    P, H, dk, dv = 6, 3, 16, 4
    E = rng.standard_normal((P, H, dv, dk))
    t = rng.uniform(0.5, 1.0, (P, H))
    ids = np.array([4, 0, 5, 2, 2, 1], dtype=np.int32)
    cu = np.array([0, 4, 4, 6], dtype=np.int32)
    S0 = rng.standard_normal((3, H, dv, dk))
    inv_freq = 10000.0 ** (-np.arange(dk // 2) / (dk // 2))
    S = oracle.rope_compose(S0, E, t, ids, cu, np.zeros(6, dtype=np.int32), inv_freq)
    np.testing.assert_allclose(S, oracle.diag_compose(S0, E, t, ids, cu), rtol=1e-15, atol=0)
