"""GPU parity at BASELINE.json's full run lengths and a soak of the persistent kernel.

Every step of every compared sequence is checked element by element against the CPU oracle
(hidden state and logits: rel-L2 <= 1e-3 per BASELINE.json, and the count of non-identical values,
expected 0 under the arithmetic contract of DESIGN.md section 5; greedy token ids equal).

  cfg 2, batch 1 : all 128 + 512 steps          cfg 4, batch 1 : all 64 + 512 steps
  cfg 3, batch 4 / 16 / 64 : the first 32 steps of EVERY sequence; the rest of the 256 steps is covered by
                              batch invariance in test_gpu_parity.py
  cfg 4, batch 8 : the first 32 steps of all 8 sequences
"""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import REL_L2_TOL, Stats, n_cores, n_diff_bits, rel_l2

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
        _blob_cache.clear()
        s = ds.shape_for_config(cfg_idx)
        _blob_cache[cfg_idx] = (s, ds.make_blob(s, cfg_idx))
    return _blob_cache[cfg_idx]


def compare_all(gpu, orc, batch, st, step, what):
    """every sequence of the batch: GPU model vs a batch-`batch` oracle"""
    gpu.sync()
    gh = gpu.hidden()[:batch].cpu().numpy()
    gl = gpu.logits()[:batch].cpu().numpy()
    gt = gpu.next_tokens()[:batch].cpu().numpy()
    oh, ol, ot = orc.hidden(), orc.logits(), orc.next_tokens()
    assert np.all(np.isfinite(gl)), f"{what} step {step}: non-finite logits"
    for b in range(batch):
        rh, rl = rel_l2(gh[b], oh[b]), rel_l2(gl[b], ol[b])
        st.max_rel_hidden = max(st.max_rel_hidden, rh)
        st.max_rel_logits = max(st.max_rel_logits, rl)
        st.diff_hidden += n_diff_bits(gh[b], oh[b])
        st.diff_logits += n_diff_bits(gl[b], ol[b])
        assert rh <= REL_L2_TOL, f"{what} step {step} seq {b}: hidden rel-L2 {rh:.3e}"
        assert rl <= REL_L2_TOL, f"{what} step {step} seq {b}: logits rel-L2 {rl:.3e}"
        assert int(gt[b]) == int(ot[b]), f"{what} step {step} seq {b}: argmax {int(gt[b])} != oracle {int(ot[b])}"
    st.steps += 1
    return gt


def run_prompt_then_greedy(env, cfg_idx, batch, n_prompt, n_decode, what):
    """prompt teacher-forced (per-sequence streams), then greedy decode with the tokens kept on the device"""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(cfg_idx)
    prompt = np.stack([ds.token_stream(s.vocab, n_prompt, seed=cfg_idx, seq_index=b) for b in range(batch)], axis=1) if n_prompt else None
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch), blob)
    orc = oracle.OracleModel(blob, batch)
    st = Stats()
    nxt = gpu.next_tokens()[:batch]
    otok = None
    for t in range(n_prompt + n_decode):
        if t < n_prompt:
            tok = np.ascontiguousarray(prompt[t], np.int32)
            gpu.step(torch.from_numpy(tok).cuda())
        else:
            tok = np.ascontiguousarray(otok, np.int32)
            gpu.step(nxt)
        orc.step(tok)
        otok = compare_all(gpu, orc, batch, st, t, what)
    print(what, st)
    return st


def test_cfg2_1p3b_full_length_vs_oracle(env):
    """BASELINE.json config 2 (the headline workload), ALL 640 steps against the oracle."""
    st = run_prompt_then_greedy(env, 2, 1, 128, 512, "cfg2-full")
    assert st.steps == 640 and st.diff_hidden == 0 and st.diff_logits == 0, st


def test_cfg4_2p7b_full_length_vs_oracle(env):
    """BASELINE.json config 4 at batch 1, ALL 576 steps against the oracle."""
    st = run_prompt_then_greedy(env, 4, 1, 64, 512, "cfg4-full")
    assert st.steps == 576 and st.diff_hidden == 0 and st.diff_logits == 0, st


@pytest.mark.parametrize("batch", [4, 16, 64])
def test_cfg3_first_32_steps_every_sequence(env, batch):
    """Config 3: the first 32 decode steps of EVERY sequence of the batch against the oracle."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(2)
    T = 32
    toks = ds.token_batch(s.vocab, T, seed=3, batch=batch)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch), blob)
    orc = oracle.OracleModel(blob, batch)
    st = Stats()
    for t in range(T):
        gpu.step(torch.from_numpy(np.ascontiguousarray(toks[t], np.int32)).cuda())
        orc.step(toks[t])
        compare_all(gpu, orc, batch, st, t, f"cfg3-b{batch}")
    print(f"cfg3 b={batch}", st)
    assert st.steps == T and st.diff_hidden == 0 and st.diff_logits == 0, st


@pytest.mark.parametrize("cfg_idx,batch,n_prompt,n_decode,seqs", [(3, 64, 0, 256, (63,)), (3, 16, 0, 256, (15,)), (4, 8, 64, 512, (5,))],
                         ids=["cfg3-b64", "cfg3-b16", "cfg4-b8"])
def test_batched_full_length_sampled_sequences(env, cfg_idx, batch, n_prompt, n_decode, seqs):
    """BASELINE.json's full run lengths of the BATCHED configs (cfg 3: 256 greedy decode steps at batch 16 / 64; cfg 4: 64-token
    prompt + 512 decode steps at batch 8) on the CUDA-graph path, greedy tokens kept on the device; the sampled sequences against
    batch-1 oracles fed the GPU's own tokens, EVERY step: hidden state and logits bit for bit, greedy token equal."""
    import os
    from _parity import compare_step
    if cfg_idx == 4 and not os.environ.get("DFSSM_LONG_TESTS"):
        pytest.skip("3 minutes of CPU oracle (passed at commit time): set DFSSM_LONG_TESTS=1 to run")
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s, blob = blob_for(2 if cfg_idx == 3 else cfg_idx)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch), blob)
    orcs = {q: oracle.OracleModel(blob, 1) for q in seqs}
    first = np.stack([ds.token_stream(s.vocab, max(n_prompt, 1), seed=cfg_idx, seq_index=i) for i in range(batch)], 1)      # [step][seq]
    st = Stats()
    nxt = None
    for t in range(n_prompt + n_decode):
        tk = torch.from_numpy(np.ascontiguousarray(first[t], np.int32)).cuda() if (t < n_prompt or t == 0) else nxt
        gpu.step(tk)
        fed = tk.cpu().numpy()
        for q, o in orcs.items():
            o.step(fed[q:q + 1])
            compare_step(gpu, o, q, st, t, f"cfg{cfg_idx}-b{batch}")
        nxt = gpu.next_tokens()[:batch].clone()
    print(f"cfg{cfg_idx} b={batch} sequences {seqs}", st)
    assert st.steps == (n_prompt + n_decode) * len(seqs) and st.diff_hidden == 0 and st.diff_logits == 0, st


def test_cfg4_batch8_first_32_steps_every_sequence(env):
    st = run_prompt_then_greedy(env, 4, 8, 32, 0, "cfg4-b8")
    assert st.steps == 32 and st.diff_hidden == 0 and st.diff_logits == 0, st


def test_persistent_kernel_soak_under_memory_traffic(env):
    """5,000 greedy steps of config 2 on the persistent kernel while a second stream saturates HBM / L2 with copies (to
    perturb the timing of the exchanges between CTAs), against the kernel chain (DFSSM_FLAG_NO_MEGA) run without the
    perturbation: greedy tokens of every step, final logits, hidden state and recurrent state bit-identical."""
    pk, torch = env["pk"], env["torch"]
    s, blob = blob_for(2)
    N = 5000
    prompt = ds.token_stream(s.vocab, 8, seed=2, seq_index=0)

    def run(flags, perturb):
        m = pk.Model(pk.Config.from_shape(s, max_batch=1, flags=flags), blob)
        for t in range(8):
            m.step(torch.from_numpy(prompt[t:t + 1].astype(np.int32)).cuda())
        nxt = m.next_tokens()[:1]
        toks = torch.empty(N, dtype=torch.int32, device="cuda")
        side = torch.cuda.Stream()
        if perturb:
            a = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
            b = torch.empty_like(a)
        m.sync()
        for t in range(N):
            if perturb and t % 4 == 0:
                with torch.cuda.stream(side):
                    b.copy_(a, non_blocking=True)          # 512 MB of traffic, concurrent with ~4 steps
            m.step(nxt)
            with torch.cuda.stream(m.stream):
                toks[t:t + 1].copy_(nxt, non_blocking=True)
        m.sync()
        torch.cuda.synchronize()
        state = [m.get_state(l, 0) for l in (0, s.n_layers // 2, s.n_layers - 1)]
        out = (toks.cpu().numpy(), m.logits()[0].cpu().numpy().copy(), m.hidden()[0].cpu().numpy().copy(), state)
        assert (m.launches_per_step(1) == 1) == (not (flags & pk.binding.FLAG_NO_MEGA))
        m.close()
        return out

    mt, ml, mh, ms = run(0, True)
    ct, cl, ch, cs = run(pk.binding.FLAG_NO_MEGA, False)
    bad = np.flatnonzero(mt != ct)
    assert bad.size == 0, f"greedy tokens differ first at step {bad[0]}"
    assert n_diff_bits(ml, cl) == 0 and n_diff_bits(mh, ch) == 0
    for (sa, ca), (sb, cb) in zip(ms, cs):
        assert n_diff_bits(sa, sb) == 0 and n_diff_bits(ca, cb) == 0
