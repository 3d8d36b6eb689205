"""Property tests (hypothesis) of the oracle on tiny random shapes -- SURVEY section 4 item 5: K not a multiple of 128, r = 1,
batch = 3, zero vectors.  Each property is something the definition fixes for EVERY input, checked against numpy float64 /
integer arithmetic written here (not against the oracle itself)."""
import numpy as np
import pytest
from hypothesis import HealthCheck, given, settings, strategies as st

import dfssm_synth as ds

SET = dict(max_examples=40, deadline=None, suppress_health_check=[HealthCheck.function_scoped_fixture])


@settings(**SET)
@given(rows=st.integers(1, 9), words=st.integers(1, 5), seed=st.integers(0, 2**31 - 1))
def test_sign_matvec_is_the_dense_pm1_product(oracle_mod, rows, words, seed):
    g = np.random.default_rng(seed)
    K = 32 * words
    sign = g.integers(0, 2**32, size=(rows, words), dtype=np.uint64).astype(np.uint32)
    xq = g.integers(-127, 128, size=K).astype(np.int8)
    bits = ((sign[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(rows, K).astype(np.int64)
    want = (2 * bits - 1) @ xq.astype(np.int64)
    got = oracle_mod.sign_matvec(sign, xq)
    assert np.array_equal(got.astype(np.int64), want)
    assert np.abs(got.astype(np.int64)).max() <= 127 * K


@settings(**SET)
@given(d=st.integers(1, 70), seed=st.integers(0, 2**31 - 1), scale=st.sampled_from([0.0, 1e-30, 1.0, 3e4]))
def test_quantiser_properties(oracle_mod, d, seed, scale):
    g = np.random.default_rng(seed)
    v = (g.standard_normal(d) * scale).astype(np.float32)
    w = (1.0 + 0.1 * g.standard_normal(d)).astype(np.float32)
    q, s, rstd, amax = oracle_mod.norm_quant(v, w)
    t = (v * w).astype(np.float32)
    assert amax == np.abs(t).max()
    if amax == 0.0:
        assert not q.any() and s == 0.0
        return
    assert np.abs(q.astype(np.int32)).max() == 127                                  # the arg-max element maps to +-127
    assert np.all(np.abs(q.astype(np.int32)) <= 127)
    # |t - (amax/127) q| <= half a step (+ rounding slack of the binary32 product t * inv)
    step = np.float64(amax) / 127.0
    assert np.all(np.abs(t.astype(np.float64) - step * q) <= 0.5 * step * (1 + 1e-5) + 1e-38)
    assert np.all(np.sign(q) * np.sign(t) >= 0)


@settings(**SET)
@given(T=st.integers(1, 12), seed=st.integers(0, 2**31 - 1))
def test_ssm_steps_equal_the_unrolled_sum(oracle_mod, T, seed):
    """T steps of one head from a zero state == H_T = sum_s (prod_{r>s} dA_r) dt_s x_s (x) B_s, and y_T = C_T.H_T + D x_T (float64)."""
    g = np.random.default_rng(seed)
    P, N = 4, 8
    A = -np.exp(g.uniform(0, 2, 1)).astype(np.float32)
    D = g.standard_normal(1).astype(np.float32)
    H = np.zeros((1, P, N), np.float32)
    xs, Bs, Cs, dts = (g.standard_normal((T, P)).astype(np.float32), g.standard_normal((T, N)).astype(np.float32),
                       g.standard_normal((T, N)).astype(np.float32), g.uniform(1e-3, 1e-1, (T, 1)).astype(np.float32))
    y = None
    for t in range(T):
        y = oracle_mod.ssm_step(H, xs[t], Bs[t], Cs[t], dts[t], A, D)
    Hd = np.zeros((P, N))
    for s_ in range(T):
        decay = np.prod([np.exp(np.float64(dts[r, 0]) * np.float64(A[0])) for r in range(s_ + 1, T)]) if s_ + 1 < T else 1.0
        Hd += decay * np.float64(dts[s_, 0]) * np.outer(xs[s_].astype(np.float64), Bs[s_].astype(np.float64))
    assert np.allclose(H[0], Hd, rtol=2e-5, atol=1e-6)
    assert np.allclose(y, Hd @ Cs[T - 1].astype(np.float64) + np.float64(D[0]) * xs[T - 1], rtol=2e-4, atol=1e-5)


@settings(max_examples=8, deadline=None, suppress_health_check=[HealthCheck.function_scoped_fixture])
@given(d_model=st.sampled_from([32, 96, 160]), r=st.sampled_from([1, 3, 8]), groups=st.sampled_from([1, 2]), seed=st.integers(0, 1000))
def test_whole_step_batch_invariance_and_zero_embedding(oracle_mod, d_model, r, groups, seed):
    """batch = 3: sequence i inside a batch == the same sequence alone, bit for bit; a zero embedding row (amax = 0) stays finite."""
    s = ds.tiny_shape(n_layers=2, d_model=d_model, d_inner=2 * d_model, headdim=16, d_state=16, ngroups=groups, lora_rank=r, vocab=50)
    blob = ds.make_blob(s, seed=seed, variant="varied")
    _, views = ds.blob_views(blob)
    views["G.emb"][5, :] = 0
    toks = ds.token_batch(s.vocab, 4, seed=seed, batch=3)
    toks[1, 2] = 5                                             # the zero row goes through sequence 2 at step 1
    mb = oracle_mod.OracleModel(blob, 3)
    solo = [oracle_mod.OracleModel(blob, 1) for _ in range(3)]
    for t in range(4):
        mb.step(toks[t])
        for b in range(3):
            solo[b].step(toks[t, b:b + 1])
            assert np.array_equal(mb.logits()[b].view(np.uint32), solo[b].logits()[0].view(np.uint32))
            assert np.array_equal(mb.hidden()[b].view(np.uint32), solo[b].hidden()[0].view(np.uint32))
        assert np.all(np.isfinite(mb.logits()))
