"""dfssm_sched_* (second half): continuous batching must not change a single token.  Every request of a
mixed workload (more requests than slots, prompts of 1..40 tokens, 1..30 new tokens, so that slots free up and are refilled
while others are mid-generation) must produce exactly the tokens of running it ALONE through dfssm_step - and one of them is
checked against the CPU oracle.  Also: the host-side bookkeeping (FIFO order, stats, errors)."""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import n_cores

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


def solo(env, s, blob, prompt, n_new):
    """the request alone on a batch-1 context: teacher-forced prompt through dfssm_step, then greedy decode"""
    torch, pk = env["torch"], env["pk"]
    m = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
    for t in prompt:
        m.step(torch.tensor([int(t)], dtype=torch.int32, device="cuda"))
    out = []
    for _ in range(n_new):
        m.sync()
        tok = int(m.next_tokens()[0].item())
        out.append(tok)
        if len(out) < n_new:
            m.step(torch.tensor([tok], dtype=torch.int32, device="cuda"))
    m.close()
    return np.array(out, np.int32)


@pytest.mark.parametrize("slots,kw", [(3, dict(n_layers=2, d_model=96, d_inner=192, headdim=32, d_state=32, ngroups=2, lora_rank=5, vocab=101)),
                                      (7, dict(n_layers=2, d_model=128, d_inner=256, headdim=32, d_state=16, lora_rank=8, vocab=300))],
                         ids=["3slots-mega", "7slots-chain"])
def test_every_request_equals_its_solo_run(env, slots, kw):
    torch, pk, oracle = env["torch"], env["pk"], env["oracle"]
    s = ds.tiny_shape(**kw)
    blob = ds.make_blob(s, seed=21, variant="varied")
    rng = np.random.default_rng(slots)
    reqs = [(ds.token_stream(s.vocab, int(rng.integers(1, 41)), seed=100 + i), int(rng.integers(1, 31))) for i in range(3 * slots + 2)]
    m = pk.Model(pk.Config.from_shape(s, max_batch=slots), blob)
    sch = pk.Scheduler(m, max_prompt=64)
    ids = [sch.submit(p, n) for p, n in reqs]
    assert ids == list(range(len(reqs)))
    sch.run()
    st = sch.stats()
    assert st["slot_steps_used"] == sum(n - 1 for _, n in reqs)          # the first token of a request comes from its prefill
    assert st["slot_steps_used"] <= st["slot_steps_run"] <= st["steps"] * slots
    for rid, (p, n) in zip(ids, reqs):
        got, done = sch.result(rid)
        assert done and got.size == n
        want = solo(env, s, blob, p, n)
        assert np.array_equal(got, want), (rid, got, want)
    # one request against the oracle
    p, n = reqs[1]
    orc = oracle.OracleModel(blob, 1)
    for t in p:
        orc.step(np.array([t], np.int32))
    want = []
    for _ in range(n):
        want.append(int(orc.next_tokens()[0]))
        orc.step(np.array([want[-1]], np.int32))
    assert np.array_equal(sch.result(ids[1])[0], np.array(want, np.int32))
    sch.close()
    m.close()


def test_iterate_admits_in_fifo_order_and_errors(env):
    pk = env["pk"]
    from paper_2606_10932_b200 import binding
    s = ds.tiny_shape(n_layers=1)
    m = pk.Model(pk.Config.from_shape(s, max_batch=2), ds.make_blob(s, 3))
    sch = pk.Scheduler(m, max_prompt=8)
    a = sch.submit([1, 2, 3], 4)
    b = sch.submit([4], 2)
    c = sch.submit([5, 6], 3)
    assert sch.iterate() == 2                       # a and b admitted: first tokens from their prefill + one step; b is done, c waits
    assert [sch.result(r)[0].size for r in (a, b, c)] == [2, 2, 0]
    assert sch.result(b)[1] and not sch.result(a)[1]
    assert sch.iterate() == 2                       # c takes b's slot: first token + one step
    assert [sch.result(r)[0].size for r in (a, b, c)] == [3, 2, 2]
    sch.run()
    assert all(sch.result(r)[1] for r in (a, b, c)) and sch.iterate() == 0
    with pytest.raises(binding.DfssmError) as ei:
        sch.submit(list(range(9)), 1)               # longer than the scratch
    assert ei.value.code == -2
    with pytest.raises(binding.DfssmError):
        sch.submit([1], 0)
    with pytest.raises(binding.DfssmError):
        sch.result(99)
    sch.close()
    m.close()


def splitmix_uniform(seed: int, k: int) -> np.float32:
    """the generator of include/dfssm.h (dfssm_sched_uniform), restated"""
    M = (1 << 64) - 1
    x = (seed + (k + 1) * 0x9E3779B97F4A7C15) & M
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & M
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & M
    x ^= x >> 31
    return np.float32((x >> 40) / 16777216.0)


def test_sampled_generation_is_schedule_independent(env):
    """temperature / top-k through the scheduler: every request equals its solo run drawn with the same counter-based uniforms,
    and one request is re-derived on the CPU oracle (dfo_sample on the oracle's logits)."""
    torch, pk, oracle = env["torch"], env["pk"], env["oracle"]
    L = pk.lib()
    for seed, k in ((0, 0), (5, 3), (2 ** 63 + 11, 1000)):
        u = splitmix_uniform(seed, k)
        assert 0.0 <= u < 1.0 and np.float32(L.dfssm_sched_uniform(seed, k)) == u
    us = np.array([splitmix_uniform(9, k) for k in range(4000)])
    assert abs(us.mean() - 0.5) < 0.02 and np.unique(us).size > 3990
    s = ds.tiny_shape(n_layers=2, d_model=96, d_inner=192, headdim=32, d_state=32, ngroups=2, lora_rank=5, vocab=101)
    blob = ds.make_blob(s, seed=23, variant="varied")
    T, K, SEED, slots = 25.0, 12, 77, 3         # a temperature at which this model leaves the greedy token often
    rng = np.random.default_rng(8)
    reqs = [(ds.token_stream(s.vocab, int(rng.integers(1, 20)), seed=300 + i), int(rng.integers(1, 16))) for i in range(8)]
    m = pk.Model(pk.Config.from_shape(s, max_batch=slots), blob)
    sch = pk.Scheduler(m, max_prompt=32)
    sch.set_sampling(T, K, SEED)
    ids = [sch.submit(p, n) for p, n in reqs]
    sch.run()
    got = [sch.result(r)[0] for r in ids]
    greedy_same = 0
    for rid, (p, n) in zip(ids, reqs):
        # solo, on the GPU: prefill-free token-by-token run with dfssm_sample and the request's own uniforms
        g = pk.Model(pk.Config.from_shape(s, max_batch=1), blob)
        o = oracle.OracleModel(blob, 1)
        for t in p:
            g.step(torch.tensor([int(t)], dtype=torch.int32, device="cuda"))
            o.step(np.array([t], np.int32))
        want_g, want_o = [], []
        for k in range(n):
            u = splitmix_uniform(SEED + rid, k)
            g.sample(T, K, torch.tensor([u], dtype=torch.float32, device="cuda"))
            g.sync()
            want_g.append(int(g.next_tokens()[0].item()))
            want_o.append(oracle.sample(o.logits()[0], T, K, float(u)))
            greedy_same += want_o[-1] == int(o.next_tokens()[0])
            g.step(g.next_tokens()[:1])
            o.step(np.array([want_o[-1]], np.int32))
        assert np.array_equal(got[rid], np.array(want_g, np.int32)), (rid, got[rid], want_g)
        assert want_g == want_o, (rid, want_g, want_o)
        g.close()
    assert greedy_same < sum(n for _, n in reqs), "the sampler never left the greedy path: the test would not see a wrong uniform"
    with pytest.raises(pk.binding.DfssmError):
        sch.set_sampling(1.0, 65)
    sch.close()
    m.close()
