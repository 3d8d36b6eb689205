"""dfssm_prefill: feeding a prompt in chunks of positions must leave exactly what feeding it token by
token through dfssm_step leaves -- recurrent state (SSM + conv), hidden state, logits and greedy token of the last position,
bit for bit -- and decoding must continue identically afterwards.  Pin: "prefill(T) then step == T + 1 steps", against the
step path of the library and against the CPU oracle."""
import time

import numpy as np
import pytest

import dfssm_synth as ds
from _parity import Stats, compare_step, n_cores, n_diff_bits

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
    dict(n_layers=2),                                                                                  # d_state 16: one state value per lane
    dict(n_layers=3, d_model=96, d_inner=192, headdim=32, d_state=32, ngroups=2, lora_rank=5, vocab=101),
    dict(n_layers=2, d_model=256, d_inner=512, headdim=64, d_state=64, lora_rank=8, vocab=1000),       # cfg 0's shape
    dict(n_layers=2, d_model=128, d_inner=256, headdim=16, d_state=128, lora_rank=16, vocab=300),      # K % 128 == 0: tcgen05 path from T = 16
]


@pytest.mark.parametrize("kw", SHAPES, ids=[f"pf{i}" for i in range(len(SHAPES))])
@pytest.mark.parametrize("T", [1, 5, 17, 131])
def test_prefill_equals_steps(env, kw, T):
    """prefill(T) on sequence 1 of a batch-2 context == T steps on a batch-1 context; then 3 greedy steps on both."""
    pk, torch = env["pk"], env["torch"]
    s = ds.tiny_shape(**kw)
    blob = ds.make_blob(s, seed=40 + len(kw), variant="varied")
    toks = ds.token_stream(s.vocab, T, seed=7, seq_index=1)
    a = pk.Model(pk.Config.from_shape(s, max_batch=2), blob)
    b = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    a.prefill(dev(torch, toks), seq=1)
    for t in range(T):
        b.step(dev(torch, toks[t:t + 1]))
    a.sync(); b.sync()

    def same(what):
        assert n_diff_bits(a.hidden()[1].cpu().numpy(), b.hidden()[0].cpu().numpy()) == 0, f"{what}: hidden"
        assert n_diff_bits(a.logits()[1].cpu().numpy(), b.logits()[0].cpu().numpy()) == 0, f"{what}: logits"
        assert int(a.next_tokens()[1].item()) == int(b.next_tokens()[0].item()), f"{what}: greedy token"
        for l in range(s.n_layers):
            sa, ca = a.get_state(l, 1)
            sb, cb = b.get_state(l, 0)
            assert n_diff_bits(sa, sb) == 0, f"{what}: SSM state of layer {l}"
            assert n_diff_bits(ca, cb) == 0, f"{what}: conv state of layer {l}"

    same(f"after prefill({T})")
    # sequence 0 of the batch-2 context was never touched
    s0, c0 = a.get_state(0, 0)
    assert not s0.any() and not c0.any()
    for k in range(3):                                   # decoding continues from the prefilled state (sequence 1 only)
        nb = b.next_tokens()[:1].clone()
        b.step(nb)
        a.step(torch.cat([nb, nb]))                      # both sequences of a get the token; only sequence 1 is compared
        a.sync(); b.sync()
        assert n_diff_bits(a.logits()[1].cpu().numpy(), b.logits()[0].cpu().numpy()) == 0, f"decode step {k} after prefill"


@pytest.mark.parametrize("cfg_idx,T", [(1, 128), (2, 128)])
def test_prefill_vs_oracle_baseline_prompts(env, cfg_idx, T):
    """The 128-token prompts of BASELINE.json configs 1 and 2 through dfssm_prefill, then 4 greedy decode steps, against the
    oracle stepping token by token; also prints the prefill time against T single steps."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.shape_for_config(cfg_idx)
    blob = ds.make_blob(s, cfg_idx)
    prompt = ds.token_stream(s.vocab, T, seed=cfg_idx, seq_index=0)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    orc = oracle.OracleModel(blob, 1)
    for t in range(T):
        orc.step(prompt[t:t + 1])
    pd = dev(torch, prompt)
    gpu.prefill(pd)
    st = Stats()
    otok = compare_step(gpu, orc, 0, st, T - 1, f"cfg{cfg_idx}-prefill")
    for l in (0, s.n_layers - 1):
        sa, ca = gpu.get_state(l, 0)
        assert n_diff_bits(sa, orc.ssm_state(l, 0)) == 0 and n_diff_bits(ca, orc.conv_state(l, 0)) == 0
    nxt = gpu.next_tokens()[:1]
    for k in range(4):
        gpu.step(nxt)
        orc.step(np.array([otok], np.int32))
        otok = compare_step(gpu, orc, 0, st, T + k, f"cfg{cfg_idx}-decode-after-prefill")
    assert st.diff_hidden == 0 and st.diff_logits == 0, st
    # timing (device, CUDA events on the library's stream)
    gpu.reset_state(-1)
    gpu.sync()
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    e0.record(gpu.stream)
    gpu.prefill(pd)
    e1.record(gpu.stream)
    gpu.sync()
    gpu.reset_state(-1)
    toks_dev = [pd[t:t + 1] for t in range(T)]
    gpu.sync()
    e1b = torch.cuda.Event(enable_timing=True)
    e1b.record(gpu.stream)
    for t in range(T):
        gpu.step(toks_dev[t])
    e2.record(gpu.stream)
    gpu.sync()
    print(f"cfg{cfg_idx}: prefill of {T} tokens {e0.elapsed_time(e1):.2f} ms; the same through {T} steps {e1b.elapsed_time(e2):.2f} ms")
