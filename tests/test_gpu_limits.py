"""The limits include/dfssm.h states: max_batch 256 (four sequence tiles of the tensor-core projections, 32 of the dp4a ones),
d_model = d_inner = 8192 (the widest rows: 64 K stages, the largest dynamic shared memory of k_proj / k_lmhead), lora_rank 64,
and the smallest legal model (0 layers: embedding -> final norm -> LM head).  Sampled sequences against the oracle, bit for bit."""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import Stats, compare_step, n_cores

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


def run(env, s, blob, batch, seqs, steps, flags=0):
    torch, pk, oracle = env["torch"], env["pk"], env["oracle"]
    gpu = pk.Model(pk.Config.from_shape(s, max_batch=batch, flags=flags), blob)
    orcs = {q: oracle.OracleModel(blob, 1) for q in seqs}
    toks = np.stack([ds.token_stream(s.vocab, steps, seed=13, seq_index=q) for q in range(batch)], 1)
    st = Stats()
    for t in range(steps):
        gpu.step(torch.from_numpy(np.ascontiguousarray(toks[t], np.int32)).cuda())
        for q, o in orcs.items():
            o.step(toks[t, q:q + 1])
            compare_step(gpu, o, q, st, t, "limits")
    assert st.diff_hidden == 0 and st.diff_logits == 0, st
    gpu.close()


@pytest.mark.parametrize("kw", [dict(n_layers=2, d_model=128, d_inner=256, headdim=32, d_state=16, lora_rank=8, vocab=300),       # tensor cores
                                dict(n_layers=2, d_model=96, d_inner=192, headdim=32, d_state=32, ngroups=2, lora_rank=5, vocab=101)],    # dp4a rows
                         ids=["mma", "dp4a"])
def test_max_batch_256(env, kw):
    s = ds.tiny_shape(**kw)
    run(env, s, ds.make_blob(s, seed=31, variant="varied"), 256, (0, 63, 64, 127, 128, 200, 255), 3)


@pytest.mark.parametrize("batch", [1, 5, 16])
def test_widest_model_8192(env, batch):
    """batch 1: the run-time-shape persistent kernel or the chain (whichever the plan fits); 5 and 16: tensor-core chain"""
    s = ds.tiny_shape(n_layers=1, d_model=8192, d_inner=8192, headdim=64, d_state=128, lora_rank=64, vocab=512)
    run(env, s, ds.make_blob(s, seed=32), batch, sorted({0, batch - 1}), 2)


def test_zero_layers(env):
    s = ds.tiny_shape(n_layers=0, d_model=64, d_inner=128, vocab=50)
    run(env, s, ds.make_blob(s, seed=33), 3, (0, 2), 2)
