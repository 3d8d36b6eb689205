"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded blob and token streams.  Bar (BASELINE.json north_star): int32 scaffold / LoRA
accumulations and argmax ids bit-exact; hidden states and logits within rel-L2 1e-3 after every step."""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import (REL_L2_TOL, Stats, compare_step, compare_taps, copy_state_gpu_to_oracle, n_cores,
                     n_diff_bits, rel_l2)

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


_blob_cache = {}


def blob_for(cfg_idx: int):
    if cfg_idx not in _blob_cache:
        _blob_cache.clear()                      # keep at most one big blob alive
        s = ds.shape_for_config(cfg_idx)
        _blob_cache[cfg_idx] = (s, ds.make_blob(s, cfg_idx))
    return _blob_cache[cfg_idx]


def dev_tokens(torch, arr):
    return torch.from_numpy(np.ascontiguousarray(arr, np.int32)).cuda()


# ------------------------------------------------------------------------------------------------
# kernel-level: every tap of every layer, tiny shapes that still span several tiles + ragged tails
# ------------------------------------------------------------------------------------------------
TINY = [
    dict(),                                                               # 1 layer, d_model 64
    dict(n_layers=3, d_model=96, d_inner=192, headdim=32, d_state=16, lora_rank=1, vocab=101),
    dict(n_layers=2, d_model=160, d_inner=320, headdim=16, d_state=20, ngroups=2, lora_rank=5, vocab=257),
    dict(n_layers=2, d_model=256, d_inner=512, headdim=64, d_state=64, ngroups=4, lora_rank=64, vocab=1000),
    dict(n_layers=1, d_model=1056, d_inner=2080, headdim=32, d_state=36, lora_rank=3, vocab=77),   # K not /64
]


@pytest.mark.parametrize("kw", TINY, ids=[f"tiny{i}" for i in range(len(TINY))])
@pytest.mark.parametrize("batch", [1, 3])
def test_taps_bit_exact_tiny(env, kw, batch):
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.tiny_shape(**kw)
    blob = ds.make_blob(s, seed=100 + len(kw), variant="varied")
    T = 6
    toks = ds.token_batch(s.vocab, T, seed=5, batch=batch)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch, flags=pk.binding.FLAG_TAPS), blob)
    orcs = [oracle.OracleModel(blob, 1, taps=True) for _ in range(batch)]
    st = Stats()
    for t in range(T):
        gpu.step(dev_tokens(torch, toks[t]))
        for b in range(batch):
            orcs[b].step(toks[t, b:b + 1])
            for l in range(s.n_layers):
                compare_taps(gpu, orcs[b], l, b, t, exact_float=True)
            compare_step(gpu, orcs[b], b, st, t, "tiny")
    assert st.diff_hidden == 0 and st.diff_logits == 0, st


def test_cfg0_tiny_16_steps(env):
    """BASELINE.json config 0: 2 layers, d_model 256, 16 steps from seed 0, batch 1."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(0)
    toks = ds.token_batch(s.vocab, 16, seed=0, batch=1)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    orc = oracle.OracleModel(blob, 1)
    st = Stats()
    for t in range(16):
        gpu.step(dev_tokens(torch, toks[t]))
        orc.step(toks[t])
        compare_step(gpu, orc, 0, st, t, "cfg0")
    print("cfg0", st)
    assert st.diff_hidden == 0 and st.diff_logits == 0, st


def _prompt_then_greedy(env, cfg_idx, n_prompt, n_decode, what):
    """Prompt teacher-forced, then greedy decode with the token kept on the device (the launch
    configuration bench.py times); the oracle decodes greedily on its own; compared every step."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(cfg_idx)
    prompt = ds.token_stream(s.vocab, n_prompt, seed=cfg_idx, seq_index=0)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    orc = oracle.OracleModel(blob, 1)
    st = Stats()
    nxt = gpu.next_tokens()[:1]
    otok = None
    for t in range(n_prompt + n_decode):
        if t < n_prompt:
            tok = prompt[t:t + 1]
            gpu.step(dev_tokens(torch, tok))
        else:
            tok = np.array([otok], np.int32)
            gpu.step(nxt)                       # device-resident greedy token of the previous step
        orc.step(tok)
        otok = compare_step(gpu, orc, 0, st, t, what)
    print(what, st)
    return st


def test_cfg1_130m_prompt_and_decode(env):
    """BASELINE.json config 1: 130M shape, 128-token prompt then 256 greedy decode tokens."""
    st = _prompt_then_greedy(env, 1, 128, 256, "cfg1")
    assert st.steps == 384


def test_cfg2_1p3b_first_steps(env):
    """BASELINE.json config 2 (headline shape): element-by-element for a 16-token prompt + 8 decode."""
    st = _prompt_then_greedy(env, 2, 16, 8, "cfg2-head")
    assert st.diff_hidden == 0, st


def test_cfg2_1p3b_full_run_sampled(env):
    """Config 2 at full length (128 + 512) in the timed launch configuration (graph, device tokens).
    The oracle cannot follow 640 steps in seconds, so: (a) the run is repeated and must be
    bit-identical (determinism), (b) at sampled late steps the GPU state is injected into the
    oracle, both take the same next step, and everything is compared."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(2)
    prompt = ds.token_stream(s.vocab, 128, seed=2, seq_index=0)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    orc = oracle.OracleModel(blob, 1)
    nxt = gpu.next_tokens()[:1]
    samples = {127, 300, 639}
    prompt_dev = [dev_tokens(torch, prompt[t:t + 1]) for t in range(128)]

    def run(check):
        gpu.reset_state(-1)
        toks, st = [], Stats()
        for t in range(640):
            if check and t in samples:
                gpu.sync()
                copy_state_gpu_to_oracle(gpu, orc, 0)
                tok_in = prompt[t:t + 1] if t < 128 else gpu.next_tokens()[:1].cpu().numpy()
                orc.step(tok_in)
            gpu.step(prompt_dev[t] if t < 128 else nxt)
            if check and t in samples:
                compare_step(gpu, orc, 0, st, t, "cfg2-sampled")
            if t >= 128:
                with torch.cuda.stream(gpu.stream):          # the library's stream orders this copy after the step
                    toks.append(gpu.next_tokens()[:1].clone())
        gpu.sync()
        return torch.cat(toks).cpu().numpy(), gpu.logits()[0].cpu().numpy().copy(), st

    toks1, logits1, st = run(True)
    toks2, logits2, _ = run(False)
    print("cfg2-sampled", st)
    assert st.steps == len(samples)
    assert np.array_equal(toks1, toks2), "two identical runs produced different tokens"
    assert n_diff_bits(logits1, logits2) == 0, "two identical runs are not bit-identical"
    assert np.all(np.isfinite(logits1))


@pytest.mark.parametrize("batch", [4, 16, 64])
def test_cfg3_batch_sweep(env, batch):
    """Config 3: independent sequences, each with its own state.  First steps of sampled sequences
    against the oracle; then batch invariance: a sequence inside the batch == the same sequence alone."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(2)
    T_or, T_inv = 3, 12
    toks = ds.token_batch(s.vocab, T_inv, seed=3, batch=batch)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch), blob)
    seqs = sorted({0, batch // 2, batch - 1})
    orcs = {b: oracle.OracleModel(blob, 1) for b in seqs}
    st = Stats()
    keep = {b: [] for b in seqs}
    for t in range(T_inv):
        gpu.step(dev_tokens(torch, toks[t]))
        gpu.sync()
        for b in seqs:
            keep[b].append((gpu.hidden()[b].cpu().numpy().copy(), gpu.logits()[b].cpu().numpy().copy()))
            if t < T_or:
                orcs[b].step(toks[t, b:b + 1])
                compare_step(gpu, orcs[b], b, st, t, f"cfg3-b{batch}")
    print(f"cfg3 b={batch}", st)
    del gpu
    solo = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    for b in seqs:
        solo.reset_state(-1)
        for t in range(T_inv):
            solo.step(dev_tokens(torch, toks[t, b:b + 1]))
            solo.sync()
            h, lg = keep[b][t]
            assert n_diff_bits(solo.hidden()[0].cpu().numpy(), h) == 0, f"batch invariance (hidden) seq {b} step {t}"
            assert n_diff_bits(solo.logits()[0].cpu().numpy(), lg) == 0, f"batch invariance (logits) seq {b} step {t}"


@pytest.mark.parametrize("batch", [1, 8])
def test_cfg4_2p7b(env, batch):
    """Config 4: 2.7B shape, batch 1 and 8, first steps against the oracle."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(4)
    T = 6 if batch == 1 else 3
    toks = ds.token_batch(s.vocab, T, seed=4, batch=batch)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch), blob)
    seqs = sorted({0, batch - 1})
    orcs = {b: oracle.OracleModel(blob, 1) for b in seqs}
    st = Stats()
    for t in range(T):
        gpu.step(dev_tokens(torch, toks[t]))
        for b in seqs:
            orcs[b].step(toks[t, b:b + 1])
            compare_step(gpu, orcs[b], b, st, t, f"cfg4-b{batch}")
    print(f"cfg4 b={batch}", st)


# ------------------------------------------------------------------------------------------------
# API behaviour and the degenerate cases of the method
# ------------------------------------------------------------------------------------------------
def test_reset_state_and_get_set_roundtrip(env):
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.tiny_shape(n_layers=2)
    blob = ds.make_blob(s, 9, "varied")
    toks = ds.token_batch(s.vocab, 9, seed=1, batch=2)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=2), blob)
    orc = oracle.OracleModel(blob, 1)
    for t in range(5):                                   # 5 steps: ring position is 1, not 0
        gpu.step(dev_tokens(torch, toks[t]))
        orc.step(toks[t, 1:2])
    for l in range(s.n_layers):
        ssm, conv = gpu.get_state(l, 1)
        assert n_diff_bits(ssm, orc.ssm_state(l, 0)) == 0
        assert n_diff_bits(conv, orc.conv_state(l, 0)) == 0
    # reset only sequence 0; sequence 1 must be untouched
    gpu.reset_state(0)
    ssm0, conv0 = gpu.get_state(0, 0)
    assert not ssm0.any() and not conv0.any()
    ssm1, _ = gpu.get_state(0, 1)
    assert n_diff_bits(ssm1, orc.ssm_state(0, 0)) == 0
    # set_state: move sequence 1's state into sequence 0, continue both with the same tokens
    for l in range(s.n_layers):
        a, c = gpu.get_state(l, 1)
        gpu.set_state(l, 0, a, c)
    st = Stats()
    for t in range(5, 9):
        tk = np.array([toks[t, 1], toks[t, 1]], np.int32)
        gpu.step(dev_tokens(torch, tk))
        orc.step(tk[:1])
        compare_step(gpu, orc, 0, st, t, "set_state")
        compare_step(gpu, orc, 1, st, t, "set_state")
    assert st.diff_hidden == 0 and st.diff_logits == 0


def test_errors(env):
    pk, torch = env["pk"], env["torch"]
    s = ds.tiny_shape()
    blob = ds.make_blob(s, 1)
    m = pk.Model(pk.Config.from_shape(s, max_batch=2))
    tok = dev_tokens(torch, [1, 2])
    with pytest.raises(pk.DfssmError) as e:
        m.step(tok)
    assert e.value.code == -3                                   # step before load
    with pytest.raises(pk.DfssmError) as e:
        m.load_weights(blob[:-64])
    assert e.value.code == -2
    bad = blob.copy(); bad[16] ^= 1                               # d_model field
    with pytest.raises(pk.DfssmError):
        m.load_weights(bad)
    m.load_weights(blob)
    with pytest.raises(pk.DfssmError) as e:
        m.step(dev_tokens(torch, [1, 2, 3]))
    assert e.value.code == -1                                   # batch > max_batch
    m.step(dev_tokens(torch, [s.vocab + 5, -1]))                # clamped + sticky error
    with pytest.raises(pk.DfssmError) as e:
        m.sync()
    assert e.value.code == -6
    m.sync()                                                    # reported once
    with pytest.raises(pk.DfssmError):
        m.debug_tensor(0, "Y")                                  # no taps in this context


def test_zero_vector_quantiser_and_host_step(env):
    """amax == 0 (a zero embedding row) must give q = 0, s = 0 and finite outputs; dfssm_step_host
    returns the same tokens / logits as the device-pointer form."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.tiny_shape(n_layers=2)
    blob = ds.make_blob(s, 3, "varied")
    _, views = ds.blob_views(blob)
    views["G.emb"][7, :] = 0
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    orc = oracle.OracleModel(blob, 1)
    st = Stats()
    nxt, lg = np.zeros(1, np.int32), np.zeros(s.vocab, np.float32)
    for t, tok in enumerate([7, 7, 3, 7]):
        tk = np.array([tok], np.int32)
        gpu.step_host(tk, nxt, lg)
        orc.step(tk)
        compare_step(gpu, orc, 0, st, t, "zero-row")
        assert nxt[0] == orc.next_tokens()[0]
        assert n_diff_bits(lg, gpu.logits()[0].cpu().numpy()) == 0
    assert st.diff_logits == 0


def test_graph_equals_eager_chain(env):
    pk, torch = env["pk"], env["torch"]
    s, blob = blob_for(0)
    toks = ds.token_batch(s.vocab, 8, seed=11, batch=2)
    a = pk.Model(pk.Config.from_shape(s, max_batch=2), blob)
    b = pk.Model(pk.Config.from_shape(s, max_batch=2, flags=pk.binding.FLAG_NO_GRAPH), blob)
    for t in range(8):
        tk = dev_tokens(torch, toks[t])
        a.step(tk); b.step(tk)
        a.sync(); b.sync()
        assert n_diff_bits(a.logits().cpu().numpy(), b.logits().cpu().numpy()) == 0
        assert torch.equal(a.next_tokens(), b.next_tokens())


def test_mega_path_is_the_batch1_path_and_equals_chain(env):
    """Batch 1 runs as ONE persistent cooperative kernel; it must be bit-identical to the kernel chain
    (DFSSM_FLAG_NO_MEGA), step after step, including the recurrent state, and they share the state layout."""
    pk, torch = env["pk"], env["torch"]
    s, blob = blob_for(0)
    toks = ds.token_batch(s.vocab, 10, seed=12, batch=1)
    a = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    b = pk.Model(pk.Config.from_shape(s, max_batch=1, flags=pk.binding.FLAG_NO_MEGA), blob)
    assert a.launches_per_step(1) == 1, "the mega path is not active on this device"
    assert b.launches_per_step(1) > 1
    for t in range(10):
        tk = dev_tokens(torch, toks[t])
        a.step(tk); b.step(tk)
        a.sync(); b.sync()
        assert n_diff_bits(a.logits().cpu().numpy(), b.logits().cpu().numpy()) == 0, f"logits differ at step {t}"
        assert n_diff_bits(a.hidden().cpu().numpy(), b.hidden().cpu().numpy()) == 0, f"hidden differs at step {t}"
        assert torch.equal(a.next_tokens(), b.next_tokens())
    for l in range(s.n_layers):
        sa, ca = a.get_state(l, 0)
        sb, cb = b.get_state(l, 0)
        assert n_diff_bits(sa, sb) == 0 and n_diff_bits(ca, cb) == 0


# ------------------------------------------------------------------------------------------------
# batch >= 16: the projections run as tcgen05 kind::i8 tiles (+-1 unpacked in shared memory, int32 in TMEM)
# ------------------------------------------------------------------------------------------------
MMA_SHAPES = [
    dict(n_layers=2, d_model=128, d_inner=256, headdim=32, d_state=16, lora_rank=3, vocab=211),       # 1 K chunk, ragged M tile
    dict(n_layers=2, d_model=256, d_inner=512, headdim=64, d_state=64, ngroups=2, lora_rank=64, vocab=300),
    dict(n_layers=1, d_model=384, d_inner=640, headdim=32, d_state=32, lora_rank=17, vocab=97),       # 3 / 5 K chunks
]


@pytest.mark.gpu
@pytest.mark.parametrize("kw", MMA_SHAPES, ids=[f"mma{i}" for i in range(len(MMA_SHAPES))])
@pytest.mark.parametrize("batch", [17, 70])
def test_tensor_core_projection_taps_bit_exact(env, kw, batch):
    """int32 scaffold / LoRA accumulators (and everything downstream) of the tcgen05 path against the oracle, every tap,
    with a ragged last row tile, a ragged sequence tile (17) and two sequence tiles (70)."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.tiny_shape(**kw)
    blob = ds.make_blob(s, seed=300 + len(kw), variant="varied")
    T = 3
    toks = ds.token_batch(s.vocab, T, seed=9, batch=batch)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch, flags=pk.binding.FLAG_TAPS), blob)
    check = sorted(set([0, 1, 15, 16, batch // 2, batch - 1]))
    orcs = {b: oracle.OracleModel(blob, 1, taps=True) for b in check}
    st = Stats()
    for t in range(T):
        gpu.step(dev_tokens(torch, toks[t]))
        for b in check:
            orcs[b].step(toks[t, b:b + 1])
            for l in range(s.n_layers):
                compare_taps(gpu, orcs[b], l, b, t, exact_float=True)
            compare_step(gpu, orcs[b], b, st, t, "mma")
    assert st.diff_hidden == 0 and st.diff_logits == 0, st


@pytest.mark.gpu
def test_tensor_core_path_equals_dp4a_path(env):
    """Same model, batch 32, with and without DFSSM_FLAG_NO_MMA: logits, hidden states and greedy tokens identical."""
    pk, torch = env["pk"], env["torch"]
    s, blob = blob_for(1)
    B, T = 32, 6
    toks = ds.token_batch(s.vocab, T, seed=21, batch=B)
    a = pk.Model(pk.Config.from_shape(s, max_batch=B), blob)
    b = pk.Model(pk.Config.from_shape(s, max_batch=B, flags=pk.binding.FLAG_NO_MMA), blob)
    for t in range(T):
        a.step(dev_tokens(torch, toks[t]))
        b.step(dev_tokens(torch, toks[t]))
        a.sync(); b.sync()
        assert torch.equal(a.logits(), b.logits()) and torch.equal(a.hidden(), b.hidden())
        assert torch.equal(a.next_tokens(), b.next_tokens())


@pytest.mark.gpu
@pytest.mark.parametrize("cfg_idx", [0, 1, 2, 4])
def test_every_baseline_shape_runs_the_persistent_kernel_at_batch_1(env, cfg_idx):
    """A shape that silently falls back to the 300-launch chain at batch 1 is a performance regression, not a parity one:
    every BASELINE.json shape must fit the one-launch persistent kernel."""
    pk = env["pk"]
    s = ds.shape_for_config(cfg_idx)
    m = pk.Model(pk.Config.from_shape(s, max_batch=1))
    assert m.launches_per_step(1) == 1
    m.close()


# k_epi_norm4 (out_proj epilogue + the norm / quantiser behind it as one cluster launch): the graph path of the
# tensor-core chain on shapes that take 1, 3, 8 CTAs of 256 threads and 5 CTAs of 512 threads per sequence, and one (d_model 384)
# that keeps the two kernels apart; the taps path (two kernels) must agree bit for bit with it.
EPN_SHAPES = [
    dict(n_layers=2, d_model=256, d_inner=512, headdim=64, d_state=16, lora_rank=8, vocab=97, batch=9),
    dict(n_layers=3, d_model=768, d_inner=768, headdim=32, d_state=32, lora_rank=16, vocab=211, batch=8),
    dict(n_layers=2, d_model=2048, d_inner=1024, headdim=64, d_state=16, lora_rank=32, vocab=150, batch=5),
    dict(n_layers=2, d_model=2560, d_inner=1280, headdim=64, d_state=16, lora_rank=64, vocab=131, batch=4),
    dict(n_layers=2, d_model=384, d_inner=768, headdim=64, d_state=16, lora_rank=8, vocab=90, batch=8),
]


@pytest.mark.gpu
@pytest.mark.parametrize("kw", EPN_SHAPES, ids=[f"d{k['d_model']}" for k in EPN_SHAPES])
def test_fused_epilogue_norm_graph_path(env, kw):
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    kw = dict(kw)
    B = kw.pop("batch")
    s = ds.tiny_shape(**kw)
    blob = ds.make_blob(s, seed=77, variant="varied")
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=B), blob)
    tap = pk.Model(pk.Config.from_shape(s, max_batch=B, flags=pk.binding.FLAG_TAPS), blob)
    seqs = sorted({0, B - 1})
    orcs = {q: oracle.OracleModel(blob, 1) for q in seqs}
    T = 6
    toks = ds.token_batch(s.vocab, T, seed=31, batch=B)
    st = Stats()
    for t in range(T):
        gpu.step(dev_tokens(torch, toks[t]))
        tap.step(dev_tokens(torch, toks[t]))
        gpu.sync(); tap.sync()
        assert torch.equal(gpu.logits(), tap.logits()) and torch.equal(gpu.hidden(), tap.hidden())
        for q, o in orcs.items():
            o.step(toks[t, q:q + 1])
            compare_step(gpu, o, q, st, t, f"epn-d{s.d_model}")
    assert st.diff_hidden == 0 and st.diff_logits == 0, st
    for q, o in orcs.items():
        for l in range(s.n_layers):
            sg, cg = gpu.get_state(l, q)
            assert n_diff_bits(sg, o.ssm_state(l, 0)) == 0 and n_diff_bits(cg, o.conv_state(l, 0)) == 0
