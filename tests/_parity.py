"""Helpers shared by the GPU parity tests: run the CUDA path (through the C ABI binding) and the CPU
oracle on the same blob and token stream and compare them element by element."""
from __future__ import annotations

import os

import numpy as np

REL_L2_TOL = 1e-3     # BASELINE.json north_star: "within max relative L2 error 1e-3 ... after every step"

INT_TAPS = ("XQ_IN", "ACC_IN", "T_IN", "GQ", "ACC_OUT", "T_OUT")
FLOAT_TAPS = ("S_IN", "ZXBCDT", "XBC_CONV", "DT", "Y", "G", "S_G", "HIDDEN")


def n_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def rel_l2(got: np.ndarray, want: np.ndarray) -> float:
    g = np.asarray(got, np.float64).ravel()
    w = np.asarray(want, np.float64).ravel()
    den = np.linalg.norm(w)
    num = np.linalg.norm(g - w)
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return float(num / den)


def n_diff_bits(got: np.ndarray, want: np.ndarray) -> int:
    a = np.ascontiguousarray(got, np.float32).view(np.uint32).ravel()
    b = np.ascontiguousarray(want, np.float32).view(np.uint32).ravel()
    return int(np.count_nonzero(a != b))


class Stats:
    def __init__(self):
        self.max_rel_hidden = 0.0
        self.max_rel_logits = 0.0
        self.diff_hidden = 0
        self.diff_logits = 0
        self.steps = 0

    def __repr__(self):
        return (f"steps={self.steps} max_rel_l2(hidden)={self.max_rel_hidden:.3e} max_rel_l2(logits)="
                f"{self.max_rel_logits:.3e} non-identical hidden={self.diff_hidden} logits={self.diff_logits}")


def compare_step(gpu, orc, seq_gpu: int, stats: Stats, step: int, what: str = ""):
    """Compare sequence `seq_gpu` of the GPU model with sequence 0 of the (batch-1) oracle."""
    import torch

    gpu.sync()
    gh = gpu.hidden()[seq_gpu].cpu().numpy()
    gl = gpu.logits()[seq_gpu].cpu().numpy()
    gt = int(gpu.next_tokens()[seq_gpu].item())
    oh, ol, ot = orc.hidden()[0], orc.logits()[0], int(orc.next_tokens()[0])
    rh, rl = rel_l2(gh, oh), rel_l2(gl, ol)
    stats.max_rel_hidden = max(stats.max_rel_hidden, rh)
    stats.max_rel_logits = max(stats.max_rel_logits, rl)
    stats.diff_hidden += n_diff_bits(gh, oh)
    stats.diff_logits += n_diff_bits(gl, ol)
    stats.steps += 1
    assert np.all(np.isfinite(gl)), f"{what} step {step}: non-finite logits"
    assert rh <= REL_L2_TOL, f"{what} step {step} seq {seq_gpu}: hidden rel-L2 {rh:.3e} > {REL_L2_TOL}"
    assert rl <= REL_L2_TOL, f"{what} step {step} seq {seq_gpu}: logits rel-L2 {rl:.3e} > {REL_L2_TOL}"
    assert gt == ot, f"{what} step {step} seq {seq_gpu}: argmax {gt} != oracle {ot}"
    return gt


def compare_taps(gpu, orc, layer: int, seq_gpu: int, step: int, exact_float: bool = True):
    for name in INT_TAPS:
        g = gpu.debug_tensor(layer, name, seq_gpu)
        o = orc.tap(layer, name, 0)
        assert g.shape == o.shape, (name, g.shape, o.shape)
        bad = np.flatnonzero(g != o)
        assert bad.size == 0, f"step {step} layer {layer} tap {name}: {bad.size} integer mismatches, first at {bad[:4]} gpu={g[bad[:4]]} oracle={o[bad[:4]]}"
    for name in FLOAT_TAPS:
        g = gpu.debug_tensor(layer, name, seq_gpu)
        o = orc.tap(layer, name, 0)
        r = rel_l2(g, o)
        assert r <= REL_L2_TOL, f"step {step} layer {layer} tap {name}: rel-L2 {r:.3e}"
        if exact_float:
            nd = n_diff_bits(g, o)
            if nd:
                i = np.flatnonzero(g.view(np.uint32) != o.view(np.uint32))[:4]
                raise AssertionError(f"step {step} layer {layer} tap {name}: {nd} float values not bit-identical "
                                     f"(arithmetic contract, DESIGN.md section 5); first {i}: gpu={g[i]} oracle={o[i]}")


def copy_state_gpu_to_oracle(gpu, orc, seq_gpu: int = 0):
    """Inject the GPU's recurrent state of one sequence into a batch-1 oracle (late-step sampled parity)."""
    for l in range(gpu.cfg.n_layers):
        ssm, conv = gpu.get_state(l, seq_gpu)
        orc.ssm_state(l, 0)[...] = ssm
        orc.conv_state(l, 0)[...] = conv
