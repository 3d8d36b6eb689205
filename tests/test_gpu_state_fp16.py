"""DFSSM_FLAG_STATE_FP16 (SURVEY 8(f) NEXT-2 first step, R24): the SSM state stored as binary16.  The CUDA path in
that mode must be bit-identical to the oracle in the same mode (kernel chain with dp4a and tcgen05 projections, prefill,
state get / set), and the drift against the fp32-state model is reported."""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import Stats, compare_step, n_cores, n_diff_bits, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    import oracle
    from paper_2606_10932_b200 import build
    build.build()
    oracle.build()
    oracle.set_threads(n_cores())
    import paper_2606_10932_b200 as pk
    return dict(torch=torch, oracle=oracle, pk=pk)


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a, np.int32)).cuda()


SHAPES = [
    dict(n_layers=2),
    dict(n_layers=3, d_model=96, d_inner=192, headdim=32, d_state=32, ngroups=2, lora_rank=5, vocab=101),
    dict(n_layers=2, d_model=128, d_inner=256, headdim=16, d_state=128, lora_rank=16, vocab=300),      # tcgen05 projections from batch 16
]


@pytest.mark.parametrize("kw", SHAPES, ids=[f"h{i}" for i in range(len(SHAPES))])
@pytest.mark.parametrize("batch", [1, 6, 17])
def test_steps_bit_identical_to_oracle_fp16_mode(env, kw, batch):
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    from paper_2606_10932_b200 import binding
    s = ds.tiny_shape(**kw)
    blob = ds.make_blob(s, seed=11, variant="varied")
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch, flags=binding.FLAG_STATE_FP16), blob)
    seqs = sorted({0, batch - 1, batch // 2})
    orcs = {q: oracle.OracleModel(blob, 1) for q in seqs}
    for o in orcs.values():
        o.set_state_fp16(True)
    toks = np.stack([ds.token_stream(s.vocab, 20, seed=11, seq_index=q) for q in range(batch)], 1)      # [step][seq]
    st = Stats()
    for t in range(20):
        gpu.step(dev(torch, toks[t]))
        for q, o in orcs.items():
            o.step(toks[t, q:q + 1])
            compare_step(gpu, o, q, st, t, "fp16-state")
    assert st.diff_hidden == 0 and st.diff_logits == 0, st
    for q, o in orcs.items():
        for l in range(s.n_layers):
            sg, cg = gpu.get_state(l, q)
            assert n_diff_bits(sg, o.ssm_state(l, 0)) == 0 and n_diff_bits(cg, o.conv_state(l, 0)) == 0
            assert np.array_equal(sg.astype(np.float16).astype(np.float32), sg)          # representable: really stored as halves


def test_cfg0_fp16_state_vs_oracle_and_drift(env):
    """BASELINE.json config 0, 16-token prompt + 48 greedy steps at batch 8: bit-identical to the oracle in fp16-state mode;
    prints the drift of the logits against the fp32-state oracle fed the same tokens."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    from paper_2606_10932_b200 import binding
    s = ds.shape_for_config(0)
    blob = ds.make_blob(s, 0)
    B = 8
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=B, flags=binding.FLAG_STATE_FP16), blob)
    o16, o32 = oracle.OracleModel(blob, 1), oracle.OracleModel(blob, 1)
    o16.set_state_fp16(True)
    q = 5
    prompt = np.stack([ds.token_stream(s.vocab, 16, seed=0, seq_index=i) for i in range(B)], 1)
    st, drift = Stats(), []
    nxt = None
    for t in range(64):
        tk = dev(torch, prompt[t]) if t < 16 else nxt
        gpu.step(tk)
        fed = tk[q:q + 1].cpu().numpy()
        o16.step(fed); o32.step(fed)
        compare_step(gpu, o16, q, st, t, "cfg0-fp16-state")
        drift.append(rel_l2(o16.logits()[0], o32.logits()[0]))
        nxt = gpu.next_tokens()[:B].clone()
    assert st.diff_hidden == 0 and st.diff_logits == 0, st
    print(f"cfg 0, fp16 state vs fp32 state (oracle, same tokens): max logits rel-L2 drift over 64 steps {max(drift):.2e}, last {drift[-1]:.2e}")


@pytest.mark.parametrize("T", [1, 19, 131])
def test_prefill_equals_steps_with_fp16_state(env, T):
    pk, torch = env["pk"], env["torch"]
    from paper_2606_10932_b200 import binding
    s = ds.tiny_shape(n_layers=3, d_model=96, d_inner=192, headdim=32, d_state=32, ngroups=2, lora_rank=5, vocab=101)
    blob = ds.make_blob(s, seed=44, variant="varied")
    toks = ds.token_stream(s.vocab, T, seed=9, seq_index=0)
    cfg = pk.Config.from_shape(s, max_batch=2, flags=binding.FLAG_STATE_FP16)
    a, b = pk.Model(cfg, blob), pk.Model(cfg, blob)
    a.prefill(dev(torch, toks), seq=1)
    for t in range(T):
        b.step(dev(torch, np.array([toks[t], toks[t]])))
    a.sync(); b.sync()
    assert n_diff_bits(a.logits()[1].cpu().numpy(), b.logits()[1].cpu().numpy()) == 0
    for l in range(s.n_layers):
        sa, ca = a.get_state(l, 1)
        sb, cb = b.get_state(l, 1)
        assert n_diff_bits(sa, sb) == 0 and n_diff_bits(ca, cb) == 0 and sa.any()


def test_set_state_rounds_and_roundtrips(env):
    pk, oracle = env["pk"], env["oracle"]
    from paper_2606_10932_b200 import binding
    s = ds.tiny_shape(n_layers=2)
    blob = ds.make_blob(s, seed=1)
    m = pk.Model(pk.Config.from_shape(s, max_batch=2, flags=binding.FLAG_STATE_FP16), blob)
    s0, c0 = m.get_state(1, 1)
    rng = np.random.default_rng(2)
    x = (rng.standard_normal(s0.shape) * 3).astype(np.float32)
    c = rng.standard_normal(c0.shape).astype(np.float32)
    m.set_state(1, 1, x, c)
    s1, c1 = m.get_state(1, 1)
    want = oracle.float_to_half(x).view(np.float16).astype(np.float32)            # the oracle's rounding, not the library's
    assert n_diff_bits(s1, want) == 0 and n_diff_bits(c1, c) == 0
    m.reset_state(1)
    s2, _ = m.get_state(1, 1)
    assert not s2.any()
