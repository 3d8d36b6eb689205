"""Pins for the oracle's floating-point parts (no GPU): specified transcendentals, conv step,
SSM step, gate.  Closed forms, brute force and libm/numpy float64, never the oracle itself."""
import math

import numpy as np
import pytest


def _ulp_err(got32, want64):
    got32 = np.asarray(got32, np.float32)
    want64 = np.asarray(want64, np.float64)
    ulp = np.spacing(np.abs(want64).astype(np.float32)).astype(np.float64)
    return np.abs(got32.astype(np.float64) - want64) / ulp


# ---------------------------------------------------------------- sp_expf / log1p / softplus / silu
def test_sp_expf_vs_libm(oracle_mod):
    xs = np.concatenate([np.linspace(-87, 88, 6001), np.linspace(-1, 1, 2001), np.linspace(-20, 0, 2001)]).astype(np.float32)
    got = oracle_mod.sp_expf(xs)
    want = np.exp(xs.astype(np.float64))
    assert _ulp_err(got, want).max() <= 4.0
    assert oracle_mod.sp_expf(np.float32(0.0)) == 1.0
    assert oracle_mod.sp_expf(np.float32(-100.0)) == 0.0
    assert np.isfinite(oracle_mod.sp_expf(np.float32(1000.0)))
    m = oracle_mod.sp_expf(np.linspace(-10, 10, 4001).astype(np.float32))
    assert np.all(np.diff(m.astype(np.float64)) >= 0)          # monotone on a sweep


def test_sp_log1pf_and_softplus_vs_libm(oracle_mod):
    ts = np.linspace(0, 1, 5001).astype(np.float32)
    got = oracle_mod.sp_log1pf(ts)
    assert _ulp_err(got[1:], np.log1p(ts[1:].astype(np.float64))).max() <= 4.0 and got[0] == 0.0
    xs = np.linspace(-30, 30, 6001).astype(np.float32)
    sp = oracle_mod.sp_softplusf(xs)
    want = np.logaddexp(0.0, xs.astype(np.float64))
    assert np.max(np.abs(sp.astype(np.float64) - want) / want) < 1e-6
    assert oracle_mod.sp_softplusf(np.float32(25.0)) == 25.0      # returns x for x > 20
    # inverse of the synthetic dt_bias recipe: softplus(softplus^-1(dt0)) = dt0
    dt0 = np.array([1e-3, 1e-2, 1e-1])
    b = (dt0 + np.log(-np.expm1(-dt0))).astype(np.float32)
    assert np.allclose(oracle_mod.sp_softplusf(b), dt0, rtol=2e-5)


def test_silu_vs_float64(oracle_mod):
    xs = np.linspace(-30, 30, 4001).astype(np.float32)
    want = xs.astype(np.float64) / (1 + np.exp(-xs.astype(np.float64)))
    got = oracle_mod.siluf(xs).astype(np.float64)
    assert np.max(np.abs(got - want)) <= 1e-6 * np.maximum(1.0, np.abs(want)).max()
    assert oracle_mod.siluf(np.float32(0.0)) == 0.0
    assert abs(oracle_mod.siluf(np.float32(40.0)) - 40.0) < 1e-5    # silu(z) -> z for large z


def test_half_to_float_all_codes(oracle_mod):
    codes = np.arange(0, 1 << 16, 7, dtype=np.uint16)
    codes = np.concatenate([codes, np.array([0, 1, 0x03FF, 0x0400, 0x7BFF, 0x8000, 0x8001, 0xFBFF], np.uint16)])
    want = codes.view(np.float16).astype(np.float32)
    got = oracle_mod.half_to_float(codes)
    ok = np.isfinite(want)
    assert np.array_equal(got[ok].view(np.uint32), want[ok].view(np.uint32))


# ---------------------------------------------------------------- conv step (S4)
def _silu64(x):
    return x / (1 + np.exp(-x))


def test_conv_step_equals_causal_correlation(oracle_mod):
    # P:122 "convolution step (stateful shift register)"; tap 3 multiplies the newest sample
    g = np.random.default_rng(10)
    C, T = 9, 11
    w = (g.standard_normal((C, 4)) * 0.2).astype(np.float32)
    bias = (g.standard_normal(C) * 0.1).astype(np.float32)
    x = g.standard_normal((T, C)).astype(np.float32)
    state = np.zeros((C, 3), np.float32)
    outs = np.stack([oracle_mod.conv_step(state, w, bias, x[t]) for t in range(T)])
    xp = np.concatenate([np.zeros((3, C)), x.astype(np.float64)])       # zero history after reset
    for t in range(T):
        pre = bias.astype(np.float64) + sum(w[:, j].astype(np.float64) * xp[t + j] for j in range(4))
        assert np.allclose(outs[t], _silu64(pre), rtol=2e-6, atol=2e-7)
    # the state holds the last three raw inputs, oldest first
    assert np.array_equal(state, x[-3:].T)


def test_conv_impulse_and_bias_only(oracle_mod):
    C = 3
    w = np.array([[1, 2, 3, 4]] * C, np.float32)
    bias = np.zeros(C, np.float32)
    state = np.zeros((C, 3), np.float32)
    seq = [np.ones(C, np.float32)] + [np.zeros(C, np.float32)] * 4
    pre = [4.0, 3.0, 2.0, 1.0, 0.0]                       # impulse returns taps 3,2,1,0 then 0
    for x, p in zip(seq, pre):
        out = oracle_mod.conv_step(state, w, bias, x)
        assert np.allclose(out, _silu64(p), rtol=1e-6, atol=1e-7)
    b2 = np.array([0.5, -1.0, 2.0], np.float32)
    out = oracle_mod.conv_step(np.zeros((C, 3), np.float32), w, b2, np.zeros(C, np.float32))
    assert np.allclose(out, _silu64(b2.astype(np.float64)), rtol=1e-6)


# ---------------------------------------------------------------- SSM step (S5)
def _ssm_inputs(g, nh=3, hd=4, ds=8):
    H = g.standard_normal((nh, hd, ds)).astype(np.float32)
    x = g.standard_normal(nh * hd).astype(np.float32)
    B = g.standard_normal(ds).astype(np.float32)
    Cv = g.standard_normal(ds).astype(np.float32)
    dt = g.uniform(1e-3, 1e-1, nh).astype(np.float32)
    A = -g.uniform(1, 16, nh).astype(np.float32)
    D = g.uniform(0.5, 1.5, nh).astype(np.float32)
    return H, x, B, Cv, dt, A, D


def test_ssm_dt_zero_leaves_state(oracle_mod):
    # BASELINE.json check 2: dt = 0 -> dA = exp(0) = 1, input term 0
    g = np.random.default_rng(11)
    H, x, B, Cv, dt, A, D = _ssm_inputs(g)
    H0 = H.copy()
    y = oracle_mod.ssm_step(H, x, B, Cv, np.zeros_like(dt), A, D)
    assert np.array_equal(H, H0)
    want = (H0.astype(np.float64) @ Cv.astype(np.float64)).reshape(-1) + np.repeat(D, 4).astype(np.float64) * x
    assert np.allclose(y, want, rtol=1e-6, atol=1e-6)


def test_ssm_c_zero_gives_dx(oracle_mod):
    # BASELINE.json check 3
    g = np.random.default_rng(12)
    H, x, B, Cv, dt, A, D = _ssm_inputs(g)
    y = oracle_mod.ssm_step(H, x, B, np.zeros_like(Cv), dt, A, D)
    assert np.array_equal(y, (np.repeat(D, 4) * x).astype(np.float32))


def test_ssm_T_steps_equal_bruteforce_sum(oracle_mod):
    # BASELINE.json check 4: H_T = sum_s (prod_{r>s} dA_r) dt_s x_s (x) B_s ; y_T = C_T.H_T + D x_T
    g = np.random.default_rng(13)
    nh, hd, ds, T = 2, 3, 5, 9
    H = np.zeros((nh, hd, ds), np.float32)
    xs = g.standard_normal((T, nh * hd)).astype(np.float32)
    Bs = g.standard_normal((T, ds)).astype(np.float32)
    Cs = g.standard_normal((T, ds)).astype(np.float32)
    dts = g.uniform(1e-2, 0.5, (T, nh)).astype(np.float32)
    A = -g.uniform(1, 4, nh).astype(np.float32)
    D = g.uniform(0.5, 1.5, nh).astype(np.float32)
    ys = [oracle_mod.ssm_step(H, xs[t], Bs[t], Cs[t], dts[t], A, D) for t in range(T)]
    f = np.float64
    dA = np.exp(dts.astype(f) * A.astype(f))                        # [T][nh]
    Hb = np.zeros((nh, hd, ds))
    for s in range(T):
        decay = np.prod(dA[s + 1:], axis=0)                         # [nh]
        contrib = (dts[s].astype(f)[:, None] * xs[s].astype(f).reshape(nh, hd))[:, :, None] * Bs[s].astype(f)
        Hb += decay[:, None, None] * contrib
    assert np.allclose(H, Hb, rtol=2e-5, atol=1e-6)
    yT = (Hb @ Cs[-1].astype(f)).reshape(-1) + np.repeat(D, hd).astype(f) * xs[-1]
    assert np.allclose(ys[-1], yT, rtol=2e-5, atol=1e-5)


def test_ssm_constant_input_geometric_limit_and_head_permutation(oracle_mod):
    g = np.random.default_rng(14)
    nh, hd, ds = 2, 2, 4
    x = g.standard_normal(nh * hd).astype(np.float32)
    B = g.standard_normal(ds).astype(np.float32)
    Cv = g.standard_normal(ds).astype(np.float32)
    dt = np.array([0.5, 0.25], np.float32)
    A = np.array([-2.0, -3.0], np.float32)
    D = np.array([1.0, 0.5], np.float32)
    H = np.zeros((nh, hd, ds), np.float32)
    for _ in range(200):
        oracle_mod.ssm_step(H, x, B, Cv, dt, A, D)
    f = np.float64
    dA = np.exp(dt.astype(f) * A.astype(f))
    Hinf = (dt.astype(f)[:, None] * x.astype(f).reshape(nh, hd))[:, :, None] * B.astype(f) / (1 - dA)[:, None, None]
    assert np.allclose(H, Hinf, rtol=1e-5, atol=1e-7)
    # heads are independent: permuting heads permutes state and output
    H1 = g.standard_normal((nh, hd, ds)).astype(np.float32)
    H2 = H1[::-1].copy()
    y1 = oracle_mod.ssm_step(H1, x, B, Cv, dt, A, D)
    y2 = oracle_mod.ssm_step(H2, x.reshape(nh, hd)[::-1].reshape(-1).copy(), B, Cv, dt[::-1].copy(),
                             A[::-1].copy(), D[::-1].copy())
    assert np.array_equal(H2[::-1], H1) and np.array_equal(y2.reshape(nh, hd)[::-1].reshape(-1), y1)


def test_ssm_groups(oracle_mod):
    # ngroups = 2: head h reads B/C group h // (nheads/ngroups)
    g = np.random.default_rng(15)
    nh, hd, ds = 4, 2, 3
    H = np.zeros((nh, hd, ds), np.float32)
    x = g.standard_normal(nh * hd).astype(np.float32)
    B = g.standard_normal(2 * ds).astype(np.float32)
    Cv = g.standard_normal(2 * ds).astype(np.float32)
    dt = g.uniform(0.1, 0.5, nh).astype(np.float32)
    A = -np.ones(nh, np.float32)
    D = np.zeros(nh, np.float32)
    y = oracle_mod.ssm_step(H, x, B, Cv, dt, A, D, ngroups=2)
    f = np.float64
    for h in range(nh):
        grp = h // 2
        Hh = (dt[h].astype(f) * x.reshape(nh, hd)[h].astype(f))[:, None] * B[grp * ds:(grp + 1) * ds].astype(f)
        assert np.allclose(H[h], Hh, rtol=1e-6)
        assert np.allclose(y.reshape(nh, hd)[h], Hh @ Cv[grp * ds:(grp + 1) * ds].astype(f), rtol=1e-5, atol=1e-6)


def test_gate_then_norm_order(oracle_mod):
    # P:395 "norm(y . silu(z))": gate = y*silu(z); for large z the gate is y*z
    y = np.array([1.0, -2.0, 0.5, 3.0], np.float32)
    z = np.array([0.0, 1.0, -1.0, 30.0], np.float32)
    gt = oracle_mod.gate(y, z)
    want = y.astype(np.float64) * (z.astype(np.float64) / (1 + np.exp(-z.astype(np.float64))))
    assert np.allclose(gt, want, rtol=1e-6, atol=1e-7) and gt[0] == 0.0 and abs(gt[3] - 90.0) < 1e-4
