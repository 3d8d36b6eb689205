"""Whole-model checks of the oracle (no GPU): stage wiring against a dense float64 numpy
restatement fed from the oracle's own taps, batch invariance, reset replay, degenerate models.

End-to-end numerical values are "parity unpinned" (the paper prints no worked example); what
is pinned here is the wiring: split order z|x|B|C|dt, which tensor feeds which stage, residual,
tied head, state persistence."""
import numpy as np
import pytest

import dfssm_synth as S


def _pm1(sign_words):
    rows, W = sign_words.shape
    bits = np.unpackbits(np.ascontiguousarray(sign_words).view(np.uint8).reshape(rows, W * 4), axis=1, bitorder="little")
    return bits.astype(np.float64) * 2 - 1


def _silu(x):
    return x / (1 + np.exp(-x))


def _softplus(x):
    return np.logaddexp(0.0, x)


@pytest.fixture(scope="module")
def tiny():
    s = S.tiny_shape(n_layers=2, ngroups=1)
    return s, S.make_blob(s, seed=11, variant="varied")


def test_stage_wiring_against_dense_float64(oracle_mod, tiny):
    s, blob = tiny
    _, W = S.blob_views(blob)
    m = oracle_mod.OracleModel(blob, 1, taps=True)
    f = np.float64
    toks = S.token_stream(s.vocab, 6, seed=5)
    conv_hist = [np.zeros((3, s.conv_dim)) for _ in range(s.n_layers)]
    Hs = [np.zeros((s.nheads, s.headdim, s.d_state)) for _ in range(s.n_layers)]
    di, gs = s.d_inner, s.ngroups * s.d_state
    for tok in toks:
        m.step([tok])
        u = W["G.emb_s"][tok].astype(f) * W["G.emb"][tok].astype(f)
        for l in range(s.n_layers):
            P = lambda n: W[f"L{l}.{n}"]
            # --- S1: the int8 codes/scale the oracle produced must dequantise to RMSNorm(u)*w
            xq, sx = m.tap(l, "XQ_IN").astype(f), f(m.tap(l, "S_IN")[0])
            xn = u / np.sqrt(np.mean(u * u) + s.norm_eps) * P("norm_w").astype(f)
            assert np.max(np.abs(sx * xq - xn)) <= 0.5 * sx * (1 + 1e-4)
            # --- S2/S3 from the oracle's own codes: dense +-1 matvec + dense LoRA
            acc = _pm1(P("in.sign")) @ xq
            assert np.array_equal(m.tap(l, "ACC_IN").astype(f), acc)
            t = P("in.A").astype(f) @ xq
            assert np.array_equal(m.tap(l, "T_IN").astype(f), t)
            zx = sx * (P("in.row_scale").astype(f) * acc
                       + P("in.b_s").astype(f) * (P("in.B").astype(f) @ (P("in.a_s").astype(f) * t)))
            zx_o = m.tap(l, "ZXBCDT").astype(f)
            assert np.allclose(zx_o, zx, rtol=1e-5, atol=1e-6)
            # --- S4 from the oracle's zxbcdt: split z | x | B | C | dt, depthwise causal conv + SiLU
            z, xBC, dt_raw = zx_o[:di], zx_o[di:di + s.conv_dim], zx_o[di + s.conv_dim:]
            assert dt_raw.size == s.nheads
            win = np.concatenate([conv_hist[l], xBC[None]])                     # [4][C], oldest first
            pre = P("conv_b").astype(f) + np.einsum("jc,cj->c", win, P("conv_w").astype(f))
            xbc_o = m.tap(l, "XBC_CONV").astype(f)
            assert np.allclose(xbc_o, _silu(pre), rtol=1e-5, atol=1e-6)
            conv_hist[l] = win[1:]
            # --- S5 from the oracle's conv output
            dt = _softplus(dt_raw + P("dt_bias").astype(f))
            assert np.allclose(m.tap(l, "DT"), dt, rtol=1e-5)
            dt = m.tap(l, "DT").astype(f)
            A = -np.exp(P("A_log").astype(f))
            x, Bv, Cv = xbc_o[:di].reshape(s.nheads, s.headdim), xbc_o[di:di + gs], xbc_o[di + gs:]
            Hs[l] = np.exp(dt * A)[:, None, None] * Hs[l] + (dt[:, None] * x)[:, :, None] * Bv
            assert np.allclose(m.ssm_state(l), Hs[l], rtol=1e-4, atol=1e-6)
            y = Hs[l] @ Cv + P("D").astype(f)[:, None] * x
            y_o = m.tap(l, "Y").astype(f)
            assert np.allclose(y_o, y.reshape(-1), rtol=1e-4, atol=1e-5)
            # --- S6 gate then norm
            g_o = m.tap(l, "G").astype(f)
            assert np.allclose(g_o, y_o * _silu(z), rtol=1e-5, atol=1e-6)
            gq, sg = m.tap(l, "GQ").astype(f), f(m.tap(l, "S_G")[0])
            gn = g_o / np.sqrt(np.mean(g_o * g_o) + s.norm_eps) * P("gnorm_w").astype(f)
            assert np.max(np.abs(sg * gq - gn)) <= 0.5 * sg * (1 + 1e-4)
            # --- S7 + residual
            acc2 = _pm1(P("out.sign")) @ gq
            assert np.array_equal(m.tap(l, "ACC_OUT").astype(f), acc2)
            t2 = P("out.A").astype(f) @ gq
            assert np.array_equal(m.tap(l, "T_OUT").astype(f), t2)
            o = sg * (P("out.row_scale").astype(f) * acc2
                      + P("out.b_s").astype(f) * (P("out.B").astype(f) @ (P("out.a_s").astype(f) * t2)))
            hid = m.tap(l, "HIDDEN").astype(f)
            assert np.allclose(hid, u + o, rtol=1e-5, atol=1e-5)
            u = hid
        assert np.array_equal(m.hidden()[0], u.astype(np.float32))
        # --- S8 tied head on the quantised final-normed hidden
        hq, sh, _, _ = oracle_mod.norm_quant(u.astype(np.float32), W["G.normf_w"], s.norm_eps)
        lg = (W["G.emb"].astype(f) @ hq.astype(f)) * (f(sh) * W["G.emb_s"].astype(f))
        assert np.allclose(m.logits()[0], lg, rtol=1e-6, atol=1e-9)
        assert m.next_tokens()[0] == int(np.argmax(m.logits()[0]))


def test_batch_invariance_and_reset_replay(oracle_mod, tiny):
    s, blob = tiny
    T, Bn = 5, 3
    tb = S.token_batch(s.vocab, T, seed=9, batch=Bn)
    mb = oracle_mod.OracleModel(blob, Bn)
    outs = []
    for t in range(T):
        mb.step(tb[t])
        outs.append((mb.logits(), mb.hidden(), mb.next_tokens()))
    for i in range(Bn):                                   # sequence alone == inside the batch, bit for bit
        m1 = oracle_mod.OracleModel(blob, 1)
        for t in range(T):
            m1.step(tb[t, i:i + 1])
            assert np.array_equal(m1.logits()[0], outs[t][0][i])
            assert np.array_equal(m1.hidden()[0], outs[t][1][i])
            assert m1.next_tokens()[0] == outs[t][2][i]
    mb.reset()                                            # reset -> replay is bit-identical
    for t in range(T):
        mb.step(tb[t])
        assert np.array_equal(mb.logits(), outs[t][0])
    mb.reset(1)                                           # per-sequence reset touches only that sequence
    assert not mb.ssm_state(0, 1).any() and mb.ssm_state(0, 0).any()


def test_state_persists_across_tokens(oracle_mod, tiny):
    # same token twice gives different logits because conv + SSM state carried over
    s, blob = tiny
    m = oracle_mod.OracleModel(blob, 1)
    m.step([3]); a = m.logits().copy()
    m.step([3]); b = m.logits().copy()
    assert not np.array_equal(a, b)
    m.reset(); m.step([3])
    assert np.array_equal(m.logits(), a)


def test_zero_layers_logits_depend_on_token_only(oracle_mod):
    s = S.tiny_shape(n_layers=0)
    blob = S.make_blob(s, seed=2)
    _, W = S.blob_views(blob)
    m = oracle_mod.OracleModel(blob, 1)
    m.step([7]); a = m.logits().copy()
    m.step([5]); m.step([7])
    assert np.array_equal(m.logits(), a)
    u = oracle_mod.embed(W["G.emb"][7], W["G.emb_s"][7])
    hq, sh, _, _ = oracle_mod.norm_quant(u, W["G.normf_w"], s.norm_eps)
    _, lg = oracle_mod.lm_head(W["G.emb"], W["G.emb_s"], hq, sh)
    assert np.array_equal(lg, a[0])


def test_bad_inputs_rejected(oracle_mod, tiny):
    s, blob = tiny
    with pytest.raises(ValueError):
        oracle_mod.OracleModel(blob[:-64], 1)
    bad = blob.copy(); bad[0] = 0
    with pytest.raises(ValueError):
        oracle_mod.OracleModel(bad, 1)
    m = oracle_mod.OracleModel(blob, 2)
    with pytest.raises(ValueError):
        m.step([s.vocab])
    with pytest.raises(ValueError):
        m.step([0, 1, 2])


def test_fp64_accumulation_is_order_independent_after_rounding():
    # premise of the arithmetic contract: a float64 sum of exact float32 products,
    # rounded once to float32, does not depend on the summation order (up to ~1e-8 probability)
    g = np.random.default_rng(0)
    flips = 0
    for _ in range(300):
        a = g.standard_normal(2048).astype(np.float32).astype(np.float64)
        b = g.standard_normal(2048).astype(np.float32).astype(np.float64)
        p = a * b
        s1 = np.float32(np.sum(p))
        s2 = np.float32(np.sum(p[g.permutation(p.size)]))
        s3 = np.float32(np.sum(p.reshape(32, 64).sum(axis=0)))
        flips += int(s1 != s2) + int(s1 != s3)
    assert flips == 0


import dfssm_synth as ds  # noqa: E402


def _run_mode(oracle_mod, blob, toks, mode):
    oracle_mod.set_mode(mode)
    try:
        m = oracle_mod.OracleModel(blob, 1)
        out = []
        for t in range(len(toks)):
            m.step(toks[t:t + 1])
            out.append((m.hidden()[0].copy(), m.logits()[0].copy(), int(m.next_tokens()[0])))
        return out
    finally:
        oracle_mod.set_mode(oracle_mod.MODE_CONTRACT)


def test_contract_mode_is_stable_under_reversed_reduction_order_and_fp64_everything_departs(oracle_mod):
    """SURVEY 8(c) item 7 / H1 as a permanent test ON THE ORACLE ITSELF (130M-like shape cut to 12 layers, 64 steps):
    (a) the contract mode with every binary64 reduction summed in REVERSED order is bit-identical in hidden state, logits
        and greedy token at every step -- the GPU may therefore use any reduction tree;
    (b) the "float64 everything" mode (a perfectly reasonable implementation) leaves the 1e-3 band of BASELINE.json within
        a few steps and never comes back: the parity bar can only be met by making the quantiser inputs reproducible."""
    s = ds.tiny_shape(n_layers=12, d_model=384, d_inner=768, headdim=64, d_state=64, lora_rank=16, vocab=2048)
    blob = ds.make_blob(s, seed=1)
    toks = ds.token_stream(s.vocab, 64, seed=1, seq_index=0)
    ref = _run_mode(oracle_mod, blob, toks, oracle_mod.MODE_CONTRACT)
    assert oracle_mod.get_mode() == oracle_mod.MODE_CONTRACT
    rev = _run_mode(oracle_mod, blob, toks, oracle_mod.MODE_REVERSED)
    for t, ((h0, l0, k0), (h1, l1, k1)) in enumerate(zip(ref, rev)):
        assert np.array_equal(h0.view(np.uint32), h1.view(np.uint32)), f"reversed reduction order changed the hidden state at step {t}"
        assert np.array_equal(l0.view(np.uint32), l1.view(np.uint32)) and k0 == k1, f"... the logits at step {t}"
    f64 = _run_mode(oracle_mod, blob, toks, oracle_mod.MODE_F64)
    rel = [float(np.linalg.norm(h0.astype(np.float64) - h1) / np.linalg.norm(h0.astype(np.float64))) for (h0, _, _), (h1, _, _) in zip(ref, f64)]
    first = next((t for t, r in enumerate(rel) if r > 1e-3), None)
    assert first is not None, f"float64-everything stayed within 1e-3 for all 64 steps: {rel[:8]}"
    assert max(rel[:first], default=0.0) < 1e-5          # before the first flipped code the two agree to rounding
    assert min(rel[first + 1:] or [1.0]) > 1e-4          # and afterwards the state carries the difference
