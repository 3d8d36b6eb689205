"""dfssm_sample (NEXT-4) against the oracle's dfo_sample on the SAME logits and the same uniform numbers: the sampled token ids
must be equal (an integer decision taken in the same arithmetic on both sides), for several temperatures and top-k values,
with ties in the logits, and a sampled decode loop must stay in lock-step with the oracle fed the same tokens."""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import n_cores, n_diff_bits

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


@pytest.mark.parametrize("batch", [1, 3])
def test_sample_equals_oracle_and_decode_loop(env, batch):
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.shape_for_config(0)
    blob = ds.make_blob(s, 0)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch), blob)
    orc = oracle.OracleModel(blob, batch)
    g = np.random.default_rng(5)
    tok = ds.token_batch(s.vocab, 1, seed=3, batch=batch)[0]
    nxt = gpu.next_tokens()[:batch]
    gpu.step(torch.from_numpy(tok).cuda())
    orc.step(tok)
    for t in range(24):
        temperature = float(g.choice([0.0, 0.3, 1.0, 2.5]))
        top_k = int(g.choice([1, 2, 7, 40, 64]))
        u = g.uniform(0, 1, batch).astype(np.float32)
        gpu.sample(temperature, top_k, torch.from_numpy(u).cuda())
        gpu.sync()
        lg = gpu.logits()[:batch].cpu().numpy()
        assert n_diff_bits(lg, orc.logits()) == 0
        want = np.array([oracle.sample(orc.logits()[b], temperature, top_k, float(u[b])) for b in range(batch)], np.int32)
        got = gpu.next_tokens()[:batch].cpu().numpy()
        assert np.array_equal(got, want), (t, temperature, top_k, u, got, want)
        gpu.step(nxt)                       # the sampled tokens, still on the device
        orc.step(want)
    gpu.sync()
    assert n_diff_bits(gpu.logits()[:batch].cpu().numpy(), orc.logits()) == 0


def test_sample_ties_and_bounds(env):
    """logits with many exact ties (written into the library's logits buffer): rank order by lower index; argument errors."""
    pk, oracle, torch = env["pk"], env["oracle"], env["torch"]
    s = ds.tiny_shape(vocab=777)
    blob = ds.make_blob(s, 1)
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=2), blob)
    gpu.step(torch.zeros(2, dtype=torch.int32, device="cuda"))
    g = np.random.default_rng(9)
    for trial in range(30):
        lg = np.round(g.standard_normal((2, s.vocab)) * 2, 0).astype(np.float32)      # integers: heavy ties
        gpu.sync()
        gpu.logits()[:2].copy_(torch.from_numpy(lg).cuda())
        torch.cuda.synchronize()
        temperature, top_k = float(g.uniform(0.2, 2.0)), int(g.integers(1, 65))
        u = g.uniform(0, 1, 2).astype(np.float32)
        gpu.sample(temperature, top_k, torch.from_numpy(u).cuda())
        gpu.sync()
        got = gpu.next_tokens()[:2].cpu().numpy()
        want = [oracle.sample(lg[b], temperature, top_k, float(u[b])) for b in range(2)]
        assert list(got) == want, (trial, temperature, top_k, u)
    with pytest.raises(pk.DfssmError):
        gpu.sample(1.0, 65, torch.zeros(2, device="cuda"))
    with pytest.raises(pk.DfssmError):
        gpu.sample(1.0, 0, torch.zeros(2, device="cuda"))
