#!/usr/bin/env python
"""bench.py -- HYPIC hot path (segment encode + composition) on B200, through the C ABI of libhypic.so.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--layers L]

A "step" is one pass of the whole hot path (rows a0..a6 of SURVEY.md section 8(a)) over the RAG-shaped request
of BASELINE.json configs[2] (cfg2): for each of the `--layers` (default 36) independent linear layers, encode
the 20 x 4096-token segments (H=32, dk=dv=128, bf16 k/v, fp32 g/beta) into (E, T), then compose the 20 segments
per head.  cfg2 is the configuration the encode target of north_star is judged on;
configs[1] (cfg1, 12 us of ideal work) and configs[4] (cfg4, the compose stress) are timed beside it and
reported in the "extra" object.  Metric: tokens/s, a token being one sequence position of one layer (all H
heads).  Inputs are synthetic and seeded (paper_2607_01299_b200/workloads.py); every layer has its own
buffers, so one step streams 49 GB of inputs -- far larger than the 126 MB L2 -- and no flush is needed.

N > 1 (torchrun): weak scaling, one request (its own seeds) per rank, no data-path collective (DESIGN.md
"Multi-GPU"); value = tokens of all ranks / max-over-ranks time.

--impl reference: the fp64 CPU oracle (oracle/), as it stands, on the host cores, on a bounded sample of the
same workload per step (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2607_01299_b200 import workloads as wl  # noqa: E402

METRIC = "cfg2 segment-encode + compose tokens/s (token = one position of one layer, all H heads)"
UNIT = "tokens/s"
SEG_LEN, N_SEG, H, D = 4096, 20, 32, 128
ENC_FLOP_PER_TOKEN_HEAD = 4 * D * (D + D) + 64 * D + 64 * (D + D)  # 155,648 at d=128, C=64
ENC_BYTES_PER_TOKEN_HEAD = 2 * D + 2 * D + 4 + 4                   # bf16 k, v + fp32 g, beta = 520 B
COMPOSE_BYTES_PER_STEP = 4 * (D * D + D * D)                       # T_i + E_i fp32 = 131,072 B
COMPOSE_FLOP_PER_STEP = 2 * D * D * D
FP32_ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12              # 148 SMs x 128 FMA lanes x max clock


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm_gbs": p["hbm_gbs"], "bf16_tflops": p["bf16_tflops"],
                "bf16_tflops_sustained": p.get("bf16_tflops_sustained"), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx = float(parts[1])
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


# ------------------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of our arm, and the whole --impl reference arm).  The only place bench.py
# touches oracle/.
# ------------------------------------------------------------------------------------------------------------
def oracle_sample_rates(units_per_core: int = 2, chains_per_core: int = 2):
    """Time the oracle, as it stands, on a bounded sample of cfg2: `cores * units_per_core` (segment, head)
    units of 4096 tokens for encode, and `cores * chains_per_core` (layer, head) chains of 20 steps for compose.
    Returns token-heads/s, compose head-steps/s, cores, and a description of the sample."""
    import numpy as np

    import oracle

    cores = oracle.num_threads()
    n_units = min(768, max(1, cores * units_per_core))  # cap bounds host memory on many-core boxes
    inp = wl.make_encode_inputs([SEG_LEN] * n_units, 1, D, D, kv_dtype=torch.bfloat16, g_lo=-0.05,
                                beta_kind="sigmoid", seed=wl.seed_for(2, 0), device="cpu")
    kf, vf = inp.k.float().numpy(), inp.v.float().numpy()
    t0 = time.perf_counter()
    E, T = oracle.segment_encode(kf, vf, inp.g.numpy(), inp.beta.numpy(), inp.cu_seqlens.numpy(), gate=inp.gate)
    t_enc = time.perf_counter() - t0
    n_chains = max(1, cores * chains_per_core)
    rng = np.random.default_rng(7)
    Ep = rng.standard_normal((N_SEG, n_chains, D, D)).astype(np.float32)
    Tp = (rng.standard_normal((N_SEG, n_chains, D, D)) * 0.05).astype(np.float32)
    ids = np.arange(N_SEG, dtype=np.int32)
    cu = np.array([0, N_SEG], dtype=np.int32)
    t0 = time.perf_counter()
    oracle.compose(None, Ep, Tp, ids, cu)
    t_cmp = time.perf_counter() - t0
    return {
        "token_heads_per_s": n_units * SEG_LEN / t_enc,
        "head_steps_per_s": n_chains * N_SEG / t_cmp,
        "cores": cores,
        "sample": (f"encode: {n_units} (segment, head) units x {SEG_LEN} tokens of cfg2 in {t_enc:.2f} s; compose: "
                   f"{n_chains} head-chains x {N_SEG} steps in {t_cmp:.2f} s; combined per layer as "
                   f"t = {N_SEG * SEG_LEN * H} token-heads / rate_enc + {N_SEG * H} head-steps / rate_cmp"),
        "seconds": t_enc + t_cmp,
    }


def tokens_per_s_from_rates(r):
    t_layer = N_SEG * SEG_LEN * H / r["token_heads_per_s"] + N_SEG * H / r["head_steps_per_s"]
    return N_SEG * SEG_LEN / t_layer


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    for _ in range(args.warmup):
        oracle_sample_rates(1, 1)
    vals, secs, last = [], 0.0, None
    for _ in range(args.steps):
        last = oracle_sample_rates(8, 8)
        vals.append(tokens_per_s_from_rates(last))
        secs += last["seconds"]
    value = sum(vals) / len(vals)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg2 (BASELINE.json configs[2]): bounded per-step sample, see cpu_baseline.sample",
                   "layers": args.layers, "segments": N_SEG, "seg_len": SEG_LEN, "H": H, "dk": D, "dv": D},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle",
                         "sample": last["sample"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------------------
class Cfg2Request:
    """One RAG-shaped request (cfg2) resident in HBM: inputs, (E, T) pools and composed state of its layers.

    The layers are independent (BASELINE.json configs[2]), so ``fold`` of them at a time are laid out along the head
    axis ([Ttot, fold*H, d]) and go through ONE hypic_segment_encode and ONE hypic_compose call:
    head l*H + h of a group is head h of its l-th layer, each layer with its own seeded k/v/g/beta."""

    def __init__(self, hb, n_layers: int, seed_base: int, device, fold: int = 1):
        self.hb = hb
        self.fold = fold = max(1, min(fold, n_layers))
        self.groups, self.sizes = [], []
        for l0 in range(0, n_layers, fold):
            ls = [wl.cfg2_layer(seed_base + l, device=device) for l in range(l0, min(l0 + fold, n_layers))]
            self.groups.append(wl.fold_layers(ls) if len(ls) > 1 else ls[0])
            self.sizes.append(len(ls))
            del ls
        mk = lambda n, G: torch.empty((n, G * H, D, D), dtype=torch.float32, device=device)
        self.E = [mk(N_SEG, G) for G in self.sizes]
        self.T = [mk(N_SEG, G) for G in self.sizes]
        self.S = [mk(1, G) for G in self.sizes]
        self.ids = torch.arange(N_SEG, dtype=torch.int32, device=device)
        self.cu = torch.tensor([0, N_SEG], dtype=torch.int32, device=device)
        need = hb.hypic_segment_encode_workspace(N_SEG, N_SEG * SEG_LEN, fold * H, D, D, hb.HYPIC_DT_BF16,
                                                 hb.HYPIC_GATE_SCALAR)
        self.ws = torch.empty(max(need, 16), dtype=torch.uint8, device=device)
        self.launches = 0

    def encode(self, i, inp=None):
        x = inp if inp is not None else self.groups[i]
        self.hb.hypic_segment_encode(x.k, x.v, x.g, x.beta, x.cu_seqlens, x.gate, E=self.E[i], T=self.T[i],
                                     workspace=self.ws)
        self.launches += self.hb.hypic_last_launch_count()

    def compose(self, i):
        self.hb.hypic_compose(None, self.E[i], self.T[i], self.ids, self.cu, total_steps=N_SEG, S_out=self.S[i])
        self.launches += self.hb.hypic_last_launch_count()

    def step(self, events=None):
        for i in range(len(self.groups)):
            if events is not None:
                events[i][0].record()
            self.encode(i)
            if events is not None:
                events[i][1].record()
            self.compose(i)
            if events is not None:
                events[i][2].record()


def time_extra_cfg1(hb, device, peaks, reps=20):
    """cfg1 (H=16, 4 x 2048): encode + compose; 4 rotating input copies (272 MB > L2) so inputs come from HBM."""
    copies = [wl.make_encode_inputs([2048] * 4, 16, D, D, kv_dtype=torch.bfloat16, g_lo=-0.05, beta_kind="sigmoid",
                                    seed=wl.seed_for(1, i), device=device) for i in range(4)]
    ids = torch.arange(4, dtype=torch.int32, device=device)
    cu = torch.tensor([0, 4], dtype=torch.int32, device=device)
    E = torch.empty((4, 16, D, D), dtype=torch.float32, device=device)
    T = torch.empty_like(E)
    S = torch.empty((1, 16, D, D), dtype=torch.float32, device=device)
    ws = torch.empty(max(16, hb.hypic_segment_encode_workspace(4, 8192, 16, D, D, hb.HYPIC_DT_BF16, 0)),
                     dtype=torch.uint8, device=device)

    def one(i):
        x = copies[i % 4]
        hb.hypic_segment_encode(x.k, x.v, x.g, x.beta, x.cu_seqlens, x.gate, E=E, T=T, workspace=ws)
        hb.hypic_compose(None, E, T, ids, cu, total_steps=4, S_out=S)

    for i in range(4):
        one(i)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(reps):
        one(i)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    return {"workload": "cfg1: H=16, 4 x 2048, encode + compose", "ms": ms, "tokens_per_s": 8192 / (ms * 1e-3),
            "tc_frac_of_bf16_burst_peak": 8192 * 16 * ENC_FLOP_PER_TOKEN_HEAD / (ms * 1e-3) / 1e12 / peaks["bf16_tflops"]}


def time_extra_cfg3(hb, device, peaks, reps=3):
    """cfg3 (64 varlen segments ~ U[512,16384], H=32, per-channel gate): encode only; HBM-bound by its 1,028 B per
    token-head, so the binding fraction is reported against the measured HBM peak."""
    inp = wl.cfg3(device=device)
    n_seg, ttot = inp.n_seg, inp.t_total
    E = torch.empty((n_seg, H, D, D), dtype=torch.float32, device=device)
    T = torch.empty_like(E)
    ws = torch.empty(max(16, hb.hypic_segment_encode_workspace(n_seg, ttot, H, D, D, hb.HYPIC_DT_BF16,
                                                               hb.HYPIC_GATE_CHANNEL)), dtype=torch.uint8, device=device)

    def one():
        hb.hypic_segment_encode(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, inp.gate, E=E, T=T, workspace=ws)

    one()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        one()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    th = ttot * H
    gbs = (th * (2 * D + 2 * D + 4 * D + 4) + n_seg * H * COMPOSE_BYTES_PER_STEP) / (ms * 1e-3) / 1e9
    tfl = th * ENC_FLOP_PER_TOKEN_HEAD / (ms * 1e-3) / 1e12
    fam = hb.hypic_encode_impl_for(H, D, D, hb.HYPIC_DT_BF16, hb.HYPIC_GATE_CHANNEL)
    return {"workload": f"cfg3: {n_seg} varlen segments, {ttot} tokens, H=32, per-channel gate, encode only (17.8 GB of "
                        "inputs: larger than L2)", "ms": ms, "tokens_per_s": ttot / (ms * 1e-3),
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"]},
            "tc_frac_of_bf16_burst_peak": tfl / peaks["bf16_tflops"],
            "kernel_family": "tensor" if fam == hb.HYPIC_IMPL_TENSOR else "simt"}


def time_extra_cfg4(hb, device, peaks, iters=48):
    """cfg4 compose stress: pool P=1024 resident (4.3 GB, reading S7), 48 layer-iterations with their own request
    lists (R=128, n_r ~ U{16..64}); compose only is timed."""
    pin = wl.cfg4_pool_inputs(device=device)
    E_tmp, T = hb.hypic_segment_encode(pin.k, pin.v, pin.g, pin.beta, pin.cu_seqlens, pin.gate)
    del pin, E_tmp
    E = wl.cfg4_pool_E(device=device)
    reqs = [wl.cfg4_requests(device=device, layer=i) for i in range(iters)]
    S_out = torch.empty_like(reqs[0].S_in)
    for i in range(3):
        hb.hypic_compose(reqs[i].S_in, E, T, reqs[i].seg_ids, reqs[i].cu_segs, S_out=S_out)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for rq in reqs:
        hb.hypic_compose(rq.S_in, E, T, rq.seg_ids, rq.cu_segs, S_out=S_out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    head_steps = sum(r.n_steps for r in reqs) * H
    gbs = head_steps * COMPOSE_BYTES_PER_STEP / (ms * 1e-3) / 1e9
    fam = hb.hypic_compose_impl_for(H, D, D)
    # the same requests over fp16-stored pools (hypic_compose_f16; the paper's cache precision)
    Eh, Th = hb.hypic_tuple_pack_f16(E), hb.hypic_tuple_pack_f16(T)
    del E, T
    for i in range(3):
        hb.hypic_compose_f16(reqs[i].S_in, Eh, Th, reqs[i].seg_ids, reqs[i].cu_segs, S_out=S_out)
    torch.cuda.synchronize()
    e0.record()
    for rq in reqs:
        hb.hypic_compose_f16(rq.S_in, Eh, Th, rq.seg_ids, rq.cu_segs, S_out=S_out)
    e1.record()
    torch.cuda.synchronize()
    ms16 = e0.elapsed_time(e1)
    gbs16 = head_steps * (COMPOSE_BYTES_PER_STEP // 2) / (ms16 * 1e-3) / 1e9
    f16 = {"ms_total": ms16, "compose_ops_per_s": head_steps / (ms16 * 1e-3),
           "roofline": {"bound": "hbm", "achieved": gbs16, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                        "frac": gbs16 / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"]},
           "note": "hypic_compose_f16: 65,536 B of fp16 (T_i, E_i) per head-step"}
    return {"workload": f"cfg4: P=1024, H=32, R=128, n~U{{16..64}}, {iters} layer-iterations, compose only",
            "fp16_pools": f16,
            "ms_total": ms, "head_steps": head_steps, "compose_ops_per_s": head_steps / (ms * 1e-3),
            "request_layer_ops_per_s": head_steps / H / (ms * 1e-3),
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"]},
            "kernel_family": "tensor" if fam == hb.HYPIC_IMPL_TENSOR else "simt"}


def time_extra_seam(hb, device, peaks, reps=20, w=8):
    """Seam-window step (hypic_seam_window): one seam of w = 8 tokens per request of cfg4's batch
    (R = 128, H = 32, dk = dv = 128, bf16 q/k/v).  S_in + S_out are 537 MB per call (larger than L2), so the state is
    read from and written to HBM every call; algorithmic bytes per (request, head): 2 * 64 KiB of state +
    w * (3 * 256 B of q, k, v + 8 B of g, beta + 512 B of o)."""
    si = wl.seam_cfg(w=w, device=device)
    e = si.enc
    R = si.S_in.shape[0]
    S_out = torch.empty_like(si.S_in)
    o = torch.empty((e.t_total, H, D), dtype=torch.float32, device=device)

    def one():
        hb.hypic_seam_window(si.S_in, si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate, S_out=S_out, o=o)

    for _ in range(3):
        one()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        one()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    unit_bytes = 2 * D * D * 4 + w * (3 * D * 2 + 8 + D * 4)
    gbs = R * H * unit_bytes / (ms * 1e-3) / 1e9
    return {"workload": f"seam window: R={R}, H=32, w={w}, bf16 q/k/v, S_in/S_out fp32 (537 MB: larger than L2)",
            "ms": ms, "seam_tokens_per_s": R * w / (ms * 1e-3), "request_layer_ops_per_s": R / (ms * 1e-3),
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"]},
            "kernel_family": "simt"}


def time_extra_forward(hb, device):
    """hypic_forward_encode (encode folded into the forward) on one cfg2-shaped layer: fp32 CUDA-core
    token recurrence over the stacked state [S ; T] (256 rows), 8 dk flop per row and token (decay, read, write,
    read-out).  Bound by the fp32 pipe: peak = 148 SMs x 128 lanes x 2 flop x the SM clock under load."""
    si = wl.make_seam_inputs([4096] * N_SEG, H, D, D, kv_dtype=torch.bfloat16, seed=wl.seed_for(7, 0), device=device)
    e = si.enc

    def one():
        return hb.hypic_forward_encode(si.q, e.k, e.v, e.g, e.beta, e.cu_seqlens, e.gate)

    one()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    one()
    one()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 2
    tfl = e.t_total * H * (2 * D) * D * 8 / (ms * 1e-3) / 1e12
    peak = 148 * 128 * 2 * 1.92e9 / 1e12
    return {"workload": "forward + encode in one pass, one cfg2-shaped layer (20 x 4096, H=32, bf16 q/k/v, fp32 arithmetic)",
            "ms": ms, "tokens_per_s": e.t_total / (ms * 1e-3),
            "roofline": {"bound": "alu", "achieved": tfl, "peak": peak, "unit": "TFLOP/s", "frac": tfl / peak,
                         "traffic": None, "peak_source": "148 SMs x 128 fp32 lanes x 2 flop x 1.92 GHz (DESIGN.md 6.5e)"},
            "kernel_family": "simt"}


def time_extra_diag(hb, device, peaks, iters=16):
    """Scalar family (Table 1: RetNet / Mamba2-style scalar gate; compressed T_C of Table 3): hypic_diag_encode on one
    cfg2-shaped layer (20 x 4096 tokens, H = 32, bf16 k/v) and hypic_diag_compose on cfg4's request lists over a
    resident pool of P = 1024 end-states (2.1 GB) with one scalar per (segment, head)."""
    inp = wl.cfg2_layer(0, device=device)
    n_seg, ttot = inp.n_seg, inp.t_total
    E = torch.empty((n_seg, H, D, D), dtype=torch.float32, device=device)
    tv = torch.empty((n_seg, H), dtype=torch.float32, device=device)

    def enc():
        hb.hypic_diag_encode(inp.k, inp.v, inp.g, inp.cu_seqlens, hb.HYPIC_GATE_SCALAR, E=E, tvec=tv)

    enc()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(3):
        enc()
    e1.record()
    torch.cuda.synchronize()
    ms_enc = e0.elapsed_time(e1) / 3
    th = ttot * H
    enc_gbs = th * (2 * D + 2 * D + 4) / (ms_enc * 1e-3) / 1e9
    fam = hb.hypic_diag_encode_impl_for(H, D, D, hb.HYPIC_DT_BF16, hb.HYPIC_GATE_SCALAR)
    del inp
    # diagonal family (GLA): the same layer shape with a per-channel gate (1,028 B per token-head)
    inp = wl.make_encode_inputs([4096] * 20, H, D, D, kv_dtype=torch.bfloat16, gate=wl.GATE_CHANNEL, g_lo=-0.05,
                                seed=wl.seed_for(6, 0), device=device)
    tvc = torch.empty((n_seg, H, D), dtype=torch.float32, device=device)

    def enc_ch():
        hb.hypic_diag_encode(inp.k, inp.v, inp.g, inp.cu_seqlens, hb.HYPIC_GATE_CHANNEL, E=E, tvec=tvc)

    enc_ch()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(3):
        enc_ch()
    e1.record()
    torch.cuda.synchronize()
    ms_ch = e0.elapsed_time(e1) / 3
    ch_gbs = th * (2 * D + 2 * D + 4 * D) / (ms_ch * 1e-3) / 1e9
    fam_ch = hb.hypic_diag_encode_impl_for(H, D, D, hb.HYPIC_DT_BF16, hb.HYPIC_GATE_CHANNEL)
    del inp, E
    E_pool = wl.cfg4_pool_E(device=device)
    t_pool = torch.rand((E_pool.shape[0], H), device=device) * 0.5 + 0.5
    reqs = [wl.cfg4_requests(device=device, layer=i) for i in range(iters)]
    S_out = torch.empty_like(reqs[0].S_in)
    for i in range(3):
        hb.hypic_diag_compose(reqs[i].S_in, E_pool, t_pool, reqs[i].seg_ids, reqs[i].cu_segs, S_out=S_out)
    torch.cuda.synchronize()
    e0.record()
    for rq in reqs:
        hb.hypic_diag_compose(rq.S_in, E_pool, t_pool, rq.seg_ids, rq.cu_segs, S_out=S_out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    head_steps = sum(r.n_steps for r in reqs) * H
    gbs = (head_steps * (D * D * 4 + 4) + iters * 128 * H * 2 * D * D * 4) / (ms * 1e-3) / 1e9
    # diagonal family (GLA): the same lists with a dk-vector of decays per tuple
    t_pool_ch = torch.rand((E_pool.shape[0], H, D), device=device) * 0.5 + 0.5
    for i in range(3):
        hb.hypic_diag_compose(reqs[i].S_in, E_pool, t_pool_ch, reqs[i].seg_ids, reqs[i].cu_segs, S_out=S_out)
    torch.cuda.synchronize()
    e0.record()
    for rq in reqs:
        hb.hypic_diag_compose(rq.S_in, E_pool, t_pool_ch, rq.seg_ids, rq.cu_segs, S_out=S_out)
    e1.record()
    torch.cuda.synchronize()
    ms_dch = e0.elapsed_time(e1)
    gbs_dch = (head_steps * (D * D * 4 + 4 * D) + iters * 128 * H * 2 * D * D * 4) / (ms_dch * 1e-3) / 1e9
    del t_pool_ch
    # state RoPE re-rotation: the same lists, every entry with a start position < 131,072
    inv_freq = (10000.0 ** (-torch.arange(D // 2, dtype=torch.float64) / (D // 2))).float().to(device)
    poss = [torch.randint(0, 131072, (r.n_steps,), device=device, dtype=torch.int32) for r in reqs]
    ws_r = torch.empty(max(hb.hypic_rope_compose_workspace(max(r.n_steps for r in reqs), D), 16), dtype=torch.uint8,
                       device=device)
    for i in range(3):
        hb.hypic_rope_compose(reqs[i].S_in, E_pool, t_pool, reqs[i].seg_ids, reqs[i].cu_segs, poss[i], inv_freq,
                              S_out=S_out, workspace=ws_r)
    torch.cuda.synchronize()
    e0.record()
    for rq, ps in zip(reqs, poss):
        hb.hypic_rope_compose(rq.S_in, E_pool, t_pool, rq.seg_ids, rq.cu_segs, ps, inv_freq, S_out=S_out, workspace=ws_r)
    e1.record()
    torch.cuda.synchronize()
    ms_rope = e0.elapsed_time(e1)
    gbs_rope = (head_steps * (D * D * 4 + 4) + iters * 128 * H * 2 * D * D * 4) / (ms_rope * 1e-3) / 1e9
    Eh = hb.hypic_tuple_pack_f16(E_pool)
    del E_pool
    for i in range(3):
        hb.hypic_diag_compose(reqs[i].S_in, Eh, t_pool, reqs[i].seg_ids, reqs[i].cu_segs, S_out=S_out)
    torch.cuda.synchronize()
    e0.record()
    for rq in reqs:
        hb.hypic_diag_compose(rq.S_in, Eh, t_pool, rq.seg_ids, rq.cu_segs, S_out=S_out)
    e1.record()
    torch.cuda.synchronize()
    ms16 = e0.elapsed_time(e1)
    gbs16 = (head_steps * (D * D * 2 + 4) + iters * 128 * H * 2 * D * D * 4) / (ms16 * 1e-3) / 1e9
    return {"compose_f16": {"ms_total": ms16, "compose_ops_per_s": head_steps / (ms16 * 1e-3),
                            "roofline": {"bound": "hbm", "achieved": gbs16, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                         "frac": gbs16 / peaks["hbm_gbs"], "traffic": None,
                                         "peak_source": peaks["source"]}},
            "workload": "scalar / diagonal families: encode of one cfg2-shaped layer; compose over cfg4's request lists "
                        f"({iters} layer-iterations, pool of 1024 end-states + one scalar each)",
            "encode": {"ms": ms_enc, "tokens_per_s": ttot / (ms_enc * 1e-3),
                       "kernel_family": "tensor" if fam == hb.HYPIC_IMPL_TENSOR else "simt",
                       "roofline": {"bound": "hbm", "achieved": enc_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                    "frac": enc_gbs / peaks["hbm_gbs"], "traffic": None,
                                    "peak_source": peaks["source"]}},
            "encode_diagonal": {"ms": ms_ch, "tokens_per_s": ttot / (ms_ch * 1e-3),
                                "kernel_family": "tensor" if fam_ch == hb.HYPIC_IMPL_TENSOR else "simt",
                                "roofline": {"bound": "hbm", "achieved": ch_gbs, "peak": peaks["hbm_gbs"],
                                             "unit": "GB/s", "frac": ch_gbs / peaks["hbm_gbs"], "traffic": None,
                                             "peak_source": peaks["source"]}},
            "compose_diagonal": {"ms_total": ms_dch, "compose_ops_per_s": head_steps / (ms_dch * 1e-3),
                                 "roofline": {"bound": "hbm", "achieved": gbs_dch, "peak": peaks["hbm_gbs"],
                                              "unit": "GB/s", "frac": gbs_dch / peaks["hbm_gbs"], "traffic": None,
                                              "peak_source": peaks["source"]}},
            "rope_compose": {"ms_total": ms_rope, "compose_ops_per_s": head_steps / (ms_rope * 1e-3),
                             "note": "hypic_rope_compose: cos/sin table kernel + fold, per call",
                             "roofline": {"bound": "hbm", "achieved": gbs_rope, "peak": peaks["hbm_gbs"],
                                          "unit": "GB/s", "frac": gbs_rope / peaks["hbm_gbs"], "traffic": None,
                                          "peak_source": peaks["source"]}},
            "compose": {"ms_total": ms, "compose_ops_per_s": head_steps / (ms * 1e-3),
                        "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                     "frac": gbs / peaks["hbm_gbs"], "traffic": None,
                                     "peak_source": peaks["source"]}}}



def run_strong(args):
    """--scaling strong: segment parallelism on devices (Eq. 9).  ONE cfg2 request:
    its 20 segments are LPT-sharded over the ranks; per group of folded layers every rank encodes its shard in two calls
    (finalize-and-ship: the first call's tuples are exchanged on a side stream while the second call runs), the tuples
    make an all-to-all (NCCL) to the head-sharded layout and every rank composes its heads."""
    from paper_2607_01299_b200 import binding as hb
    from paper_2607_01299_b200 import segment_parallel as sp
    from paper_2607_01299_b200 import sharding

    rank, local_rank, world = dist_env()
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")  # so that a scaling run can count the ranks of the communicator
        os.environ.setdefault("NCCL_DEBUG_FILE", os.path.join(ROOT, "gpurun_out", "nccl_rank%h_%p.log"))
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    hb.load_library()
    peaks = load_peaks()
    L, fold = args.layers, max(1, min(args.fold, args.layers))
    lens = [SEG_LEN] * N_SEG
    parts, groups_all = sp.plan(lens, world, 2)
    shards, sizes = [], []
    for l0 in range(0, L, fold):
        ls = [wl.cfg2_layer(l, device=device) for l in range(l0, min(l0 + fold, L))]  # the SAME request on every rank
        full = wl.fold_layers(ls) if len(ls) > 1 else ls[0]
        del ls
        shards.append([sp.take_segments(full, groups_all[g][rank]) for g in range(2)])
        sizes.append(full.H // H)
        del full
        torch.cuda.empty_cache()
    ids = torch.arange(N_SEG, dtype=torch.int32, device=device)
    cu = torch.tensor([0, N_SEG], dtype=torch.int32, device=device)
    comm = torch.cuda.Stream(device)

    def step():
        sent = 0
        for my in shards:
            res = sp.encode_exchange_compose(hb, my, groups_all, N_SEG, rank, world, ids, cu, group=None, comm_stream=comm)
            sent += res.exchanged_bytes
        return sent

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for _ in range(args.steps):
        sent = step()
    t1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_step = t0.elapsed_time(t1) / args.steps
    if dist is not None:
        ms_step = sharding.max_over_ranks(ms_step, device=device)
        sent_all = torch.tensor([float(sent)], dtype=torch.float64, device=device)
        dist.all_reduce(sent_all)
        sent = int(sent_all.item())
    if rank == 0:
        tokens = L * N_SEG * SEG_LEN  # ONE request, whatever the number of ranks
        my_tokens = sum(lens[i] for i in parts[0])
        tfl = tokens * H * ENC_FLOP_PER_TOKEN_HEAD / (ms_step * 1e-3) / 1e12
        line = {"metric": METRIC, "value": tokens / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": {"workload": "cfg2 (BASELINE.json configs[2]): ONE RAG-shaped request, segment-parallel",
                           "layers": L, "segments": N_SEG, "seg_len": SEG_LEN, "H": H, "dk": D, "dv": D,
                           "parallelism": f"segments LPT-sharded over {world} ranks (Eq. 9), 2 encode calls per rank and "
                                          "group (finalize-and-ship), all-to-all of (T_C, S_C|0) to head-sharded compose",
                           "segments_of_rank0": len(parts[0]), "tokens_of_rank0": my_tokens,
                           "exchanged_bytes_per_step": sent, "layers_per_call": fold,
                           "l2": "inputs larger than L2; no flush needed"},
                "clocks": clocks, "e2e": None, "gpu_launches": None,
                "roofline": {"bound": "tensor", "achieved": tfl / world, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                             "frac": tfl / world / peaks["bf16_tflops"], "traffic": None,
                             "note": "whole step (encode + exchange + compose) per GPU, algorithmic encode flops"},
                "cpu_baseline": None}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_ours(args):
    from paper_2607_01299_b200 import binding as hb

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libhypic has no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    hb.load_library()
    peaks = load_peaks()
    L = args.layers

    # weak scaling: every rank owns one full request with its own seeds (layer index offset by rank)
    req = Cfg2Request(hb, L, seed_base=L * rank, device=device, fold=args.fold)
    NG = len(req.groups)
    req_fold = req.fold
    for _ in range(args.warmup):
        req.step()
    torch.cuda.synchronize()

    events = [[[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(NG)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    req.launches = 0
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for s in range(args.steps):
        req.step(events[s])
    t1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = t0.elapsed_time(t1)
    launches = req.launches
    if dist is not None:
        from paper_2607_01299_b200 import sharding
        ms_total = sharding.max_over_ranks(ms_total, device=device)
    ms_step = ms_total / args.steps
    tokens_per_step = L * N_SEG * SEG_LEN * world
    value = tokens_per_step / (ms_step * 1e-3)

    # per-kernel durations measured live inside the timed region (CUDA events on the launching stream)
    # (per call of `fold` layers; the last group may be smaller, so durations are normalised to one layer first)
    enc_ms = [ev[0].elapsed_time(ev[1]) / req.sizes[i] for st in events for i, ev in enumerate(st)]
    cmp_ms = [ev[1].elapsed_time(ev[2]) / req.sizes[i] for st in events for i, ev in enumerate(st)]
    G = req.fold
    enc_layer, cmp_layer = sum(enc_ms) / len(enc_ms), sum(cmp_ms) / len(cmp_ms)
    enc_avg, cmp_avg = enc_layer * G, cmp_layer * G  # one launch of a full group
    th_per_launch = N_SEG * SEG_LEN * H * G
    enc_family = hb.hypic_encode_impl_for(H, D, D, hb.HYPIC_DT_BF16, hb.HYPIC_GATE_SCALAR)
    enc_tflops = th_per_launch * ENC_FLOP_PER_TOKEN_HEAD / (enc_avg * 1e-3) / 1e12
    enc_gbs = (th_per_launch * ENC_BYTES_PER_TOKEN_HEAD + N_SEG * H * G * COMPOSE_BYTES_PER_STEP) / (enc_avg * 1e-3) / 1e9
    # fractions are reported against the BURST figure (a kernel timed alone), the sustained one beside it
    if enc_family == hb.HYPIC_IMPL_TENSOR:
        roofline = {"bound": "tensor", "achieved": enc_tflops, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                    "frac": enc_tflops / peaks["bf16_tflops"], "traffic": None,
                    "peak_kind": f"bf16 dense, burst, {peaks['source']}",
                    "peak_sustained": peaks["bf16_tflops_sustained"],
                    "frac_sustained": enc_tflops / peaks["bf16_tflops_sustained"]}
    else:
        roofline = {"bound": "alu", "achieved": enc_tflops, "peak": FP32_ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": enc_tflops / FP32_ALU_PEAK_TFLOPS, "traffic": None,
                    "peak_kind": "fp32 FMA: 148 SMs x 128 lanes x 2 x 1.965 GHz (DESIGN.md)"}
    fam = "tensor" if enc_family == hb.HYPIC_IMPL_TENSOR else "simt"
    tpath = os.path.join(ROOT, "profiles", "traffic.json")  # dram bytes per launch from the committed ncu capture
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        per_layer = tj.get(f"encode_{fam}_cfg2_layer_dram_bytes")
        # a capture of this very launch shape if there is one, else the per-layer capture scaled to the launch
        roofline["traffic"] = tj.get(f"encode_{fam}_cfg2_fold{G}_dram_bytes",
                                     None if per_layer is None else per_layer * G)
        roofline["traffic_source"] = tj.get("source", "profiles/traffic.json (a committed ncu capture, not this run)")
    alg_bytes = th_per_launch * ENC_BYTES_PER_TOKEN_HEAD + N_SEG * H * G * COMPOSE_BYTES_PER_STEP
    roofline.update({"kernel": ("hypic_segment_encode = chunk_offsets_kernel + scan4_kernel (tensor family, scalar gate: "
                                "one fused tcgen05 kernel; the fp32 fallback-list kernel runs empty)") if fam == "tensor" else
                     "hypic_segment_encode = encode_simt_kernel (simt family)",
                     "units_per_launch": f"{th_per_launch} token-heads x {ENC_FLOP_PER_TOKEN_HEAD} flop",
                     "algorithmic_bytes_per_launch": alg_bytes,
                     "avg_launch_ms": enc_avg, "layers_per_launch": G, "ms_per_layer": enc_layer,
                     "share_of_step": enc_layer * L / ms_step,
                     "frac_of_bf16_burst_peak": enc_tflops / peaks["bf16_tflops"], "hbm_gbs": enc_gbs,
                     "hbm_frac": enc_gbs / peaks["hbm_gbs"]})

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- end to end: pinned host inputs -> H2D -> C-ABI calls -> D2H of the composed state, every step
    # (one folded group of Le layers per step, through the same two calls as the device-resident run)
    if req.sizes[0] > args.e2e_layers:
        del req
        torch.cuda.empty_cache()
        req = Cfg2Request(hb, args.e2e_layers, seed_base=L * rank, device=device, fold=args.e2e_layers)
    Le = req.sizes[0]
    stage = req.groups[0]
    host = [t.cpu().pin_memory() for t in (stage.k, stage.v, stage.g, stage.beta)]
    s_host = torch.empty((1, Le * H, D, D), dtype=torch.float32).pin_memory()
    h2d = sum(t.numel() * t.element_size() for t in host)
    d2h = s_host.numel() * 4

    def e2e_step():
        for dst, src in zip((stage.k, stage.v, stage.g, stage.beta), host):
            dst.copy_(src, non_blocking=True)
        req.encode(0, stage)
        req.compose(0)
        s_host.copy_(req.S[0], non_blocking=True)
        torch.cuda.synchronize()

    e2e_step()
    torch.cuda.synchronize()
    w0 = time.perf_counter()
    n_e2e = max(2, min(args.steps, 5))
    for _ in range(n_e2e):
        e2e_step()
    e2e_s = (time.perf_counter() - w0) / n_e2e
    e2e = {"value": Le * N_SEG * SEG_LEN / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "layers_per_step": Le,
           "note": "pinned host k/v/g/beta of one folded group of layers -> device, encode + compose via the C ABI, "
                   "composed S -> host"}
    del host, stage

    extra = {}
    if not args.no_extra:
        del req
        torch.cuda.empty_cache()
        extra["cfg1"] = time_extra_cfg1(hb, device, peaks)
        extra["cfg4_compose"] = time_extra_cfg4(hb, device, peaks)
        torch.cuda.empty_cache()
        extra["cfg3_encode"] = time_extra_cfg3(hb, device, peaks)
        torch.cuda.empty_cache()
        extra["seam_window"] = time_extra_seam(hb, device, peaks)
        torch.cuda.empty_cache()
        extra["diag_family"] = time_extra_diag(hb, device, peaks)
        torch.cuda.empty_cache()
        extra["forward_encode"] = time_extra_forward(hb, device)
        extra["cfg2_compose"] = {"avg_launch_ms": cmp_avg, "layers_per_launch": G,
                                 "compose_ops_per_s": N_SEG * H * G / (cmp_avg * 1e-3),
                                 "hbm_gbs": N_SEG * H * G * COMPOSE_BYTES_PER_STEP / (cmp_avg * 1e-3) / 1e9}
        # the compose half of BASELINE.json's metric and the other configs, where the driver keeps them (it drops "extra")
        c4 = extra["cfg4_compose"]
        roofline["compose"] = {"workload": extra["cfg4_compose"]["workload"], "ms_total": c4["ms_total"],
                               "head_steps": extra["cfg4_compose"]["head_steps"],
                               "compose_ops_per_s": c4["compose_ops_per_s"], "bound": "hbm",
                               "achieved": c4["roofline"]["achieved"], "peak": c4["roofline"]["peak"], "unit": "GB/s",
                               "frac": c4["roofline"]["frac"],
                               "traffic_source": "profiles/traffic.json: compose_tensor_cfg4_dram_bytes_per_head_step"}
        c3 = extra["cfg3_encode"]
        roofline["cfg3_encode"] = {"ms": c3["ms"], "tokens_per_s": c3["tokens_per_s"], "bound": "hbm",
                                   "achieved": c3["roofline"]["achieved"], "peak": c3["roofline"]["peak"], "unit": "GB/s",
                                   "frac": c3["roofline"]["frac"],
                                   "tc_frac_of_bf16_burst_peak": c3["tc_frac_of_bf16_burst_peak"]}
        c1 = extra["cfg1"]
        roofline["cfg1"] = {"ms": c1["ms"], "tokens_per_s": c1["tokens_per_s"],
                            "tc_frac_of_bf16_burst_peak": c1["tc_frac_of_bf16_burst_peak"]}

    cpu = None
    if not args.no_cpu_baseline:
        r = oracle_sample_rates(48, 48)
        cpu = {"value": tokens_per_s_from_rates(r), "unit": UNIT, "cores": r["cores"], "kind": "oracle",
               "sample": r["sample"], "token_heads_per_s": r["token_heads_per_s"],
               "compose_head_steps_per_s": r["head_steps_per_s"]}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": "cfg2 (BASELINE.json configs[2]): RAG-shaped request, encode all segments then compose "
                               "per layer", "layers": L, "segments": N_SEG, "seg_len": SEG_LEN, "H": H, "dk": D,
                   "dv": D, "kv_dtype": "bf16", "gate": "scalar", "requests_per_gpu": 1,
                   "layers_per_call": req_fold, "layout": f"[Ttot, {req_fold} layers x {H} heads, d] (layers folded "
                   "into the head axis, SURVEY.md 8(b); each layer keeps its own seeded inputs)",
                   "l2": "inputs larger than L2 (1.35 GB per layer, own buffers per layer group); no flush needed",
                   "token_heads_per_s": value * H},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
        "extra": extra,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layers", type=int, default=36, help="linear layers of the cfg2 request (36 = as written)")
    ap.add_argument("--e2e-layers", type=int, default=4, help="layers per end-to-end step (bounds pinned host memory)")
    ap.add_argument("--fold", type=int, default=6,
                    help="independent layers folded into the head axis per library call (1 = one call per layer)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: one private cfg2 request per rank (default); strong: ONE request, its segments LPT-sharded "
                         "over the ranks, tuples exchanged by one all-to-all per group, compose sharded by heads "
                         "(segment parallelism, PAPER.md:246-267)")
    ap.add_argument("--no-extra", action="store_true", help="skip the cfg1 / cfg4 side measurements")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.scaling == "strong":
        return run_strong(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
