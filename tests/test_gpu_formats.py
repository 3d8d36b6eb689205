"""Weight-format variants on the GPU (R25): 17-level scaffold (five bit planes unpacked to int8
tiles by k_proj_mma) and int4 LoRA (nibbles unpacked by k_proj_mma and lora_up4), alone and together, against the oracle in the
same format: every tap bit for bit on small shapes that still span several tiles, K slices and a ragged row tile; BASELINE.json
configs 0 and 1 through prompt + decode; prefill == steps; config errors."""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import Stats, compare_step, compare_taps, n_cores, n_diff_bits

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
    dict(n_layers=2, d_model=128, d_inner=256, headdim=32, d_state=16, lora_rank=8, vocab=101),
    dict(n_layers=2, d_model=384, d_inner=640, headdim=64, d_state=32, ngroups=2, lora_rank=16, vocab=300),      # K = 384 / 640: half stages
    dict(n_layers=1, d_model=256, d_inner=512, headdim=16, d_state=128, lora_rank=64, vocab=77),
]


@pytest.mark.parametrize("fmt", [1, 2, 3], ids=["lvl17", "int4", "lvl17+int4"])
@pytest.mark.parametrize("kw", SHAPES, ids=[f"f{i}" for i in range(len(SHAPES))])
@pytest.mark.parametrize("batch", [1, 6, 70])
def test_taps_bit_exact(env, kw, fmt, batch):
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.tiny_shape(fmt=fmt, **kw)
    blob = ds.make_blob(s, seed=50 + fmt, variant="varied")
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch, flags=pk.binding.FLAG_TAPS), blob)
    seqs = sorted({0, batch - 1, batch // 2})
    orcs = {q: oracle.OracleModel(blob, 1, taps=True) for q in seqs}
    T = 4
    toks = np.stack([ds.token_stream(s.vocab, T, seed=9, seq_index=q) for q in range(batch)], 1)
    st = Stats()
    for t in range(T):
        gpu.step(dev(torch, toks[t]))
        for q, o in orcs.items():
            o.step(toks[t, q:q + 1])
            for l in range(s.n_layers):
                compare_taps(gpu, o, l, q, t, exact_float=True)
            compare_step(gpu, o, q, st, t, f"fmt{fmt}")
    assert st.diff_hidden == 0 and st.diff_logits == 0, st


@pytest.mark.parametrize("cfg_idx,fmt,batch,n_prompt,n_decode", [(0, 3, 1, 0, 16), (0, 1, 8, 4, 12), (1, 3, 1, 8, 24), (1, 2, 17, 2, 6)])
def test_baseline_shapes_prompt_and_decode(env, cfg_idx, fmt, batch, n_prompt, n_decode):
    """graph path (no taps): teacher-forced prompt, then greedy decode fed back on the device; the oracle gets the GPU's tokens"""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.shape_for_config(cfg_idx).with_(fmt=fmt)
    blob = ds.make_blob(s, cfg_idx)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch), blob)
    q = batch - 1
    orc = oracle.OracleModel(blob, 1)
    prompt = np.stack([ds.token_stream(s.vocab, max(n_prompt, 1), seed=cfg_idx, seq_index=i) for i in range(batch)], 1)
    st = Stats()
    nxt = dev(torch, prompt[0])
    for t in range(n_prompt + n_decode):
        tk = dev(torch, prompt[t]) if t < n_prompt else nxt
        gpu.step(tk)
        orc.step(tk[q:q + 1].cpu().numpy())
        compare_step(gpu, orc, q, st, t, f"cfg{cfg_idx}-fmt{fmt}")
        nxt = gpu.next_tokens()[:batch].clone()
    assert st.diff_hidden == 0 and st.diff_logits == 0, st
    for l in (0, s.n_layers - 1):
        sg, cg = gpu.get_state(l, q)
        assert n_diff_bits(sg, orc.ssm_state(l, 0)) == 0 and n_diff_bits(cg, orc.conv_state(l, 0)) == 0


@pytest.mark.parametrize("T", [1, 19, 140])
def test_prefill_equals_steps(env, T):
    pk, torch = env["pk"], env["torch"]
    s = ds.tiny_shape(fmt=3, **SHAPES[1])
    blob = ds.make_blob(s, seed=61, variant="varied")
    toks = ds.token_stream(s.vocab, T, seed=4, seq_index=0)
    cfg = pk.Config.from_shape(s, max_batch=2)
    a, b = pk.Model(cfg, blob), pk.Model(cfg, blob)
    a.prefill(dev(torch, toks), seq=1)
    for t in range(T):
        b.step(dev(torch, np.array([toks[t], toks[t]])))
    a.sync(); b.sync()
    assert n_diff_bits(a.logits()[1].cpu().numpy(), b.logits()[1].cpu().numpy()) == 0
    assert int(a.next_tokens()[1].item()) == int(b.next_tokens()[1].item())
    for l in range(s.n_layers):
        sa, ca = a.get_state(l, 1)
        sb, cb = b.get_state(l, 1)
        assert n_diff_bits(sa, sb) == 0 and n_diff_bits(ca, cb) == 0 and sa.any()


def test_config_and_blob_errors(env):
    pk = env["pk"]
    from paper_2606_10932_b200 import binding
    ok = ds.tiny_shape(fmt=1, **SHAPES[0])
    blob = ds.make_blob(ok, 1)
    # the blob's format word must agree with the config flags
    with pytest.raises(binding.DfssmError) as ei:
        pk.Model(pk.Config.from_shape(ok.with_(fmt=0), max_batch=1), blob)
    assert ei.value.code in (-1, -2)
    with pytest.raises(binding.DfssmError):
        pk.Model(pk.Config.from_shape(ok.with_(fmt=3), max_batch=1), blob)
    # shapes the variants do not serve: K not a multiple of 128, rank outside {8, 16, 32, 64}, dp4a projections forced
    for bad in (dict(d_model=96, d_inner=192, lora_rank=8), dict(d_model=128, d_inner=256, lora_rank=4)):
        s = ds.tiny_shape(fmt=2, n_layers=1, headdim=32, d_state=16, vocab=50, **bad)
        assert binding.dfssm_arena_bytes(pk.Config.from_shape(s)) == 0
    assert binding.dfssm_arena_bytes(pk.Config.from_shape(ok, flags=binding.FLAG_NO_MMA)) == 0
    assert binding.dfssm_arena_bytes(pk.Config.from_shape(ok)) > 0
