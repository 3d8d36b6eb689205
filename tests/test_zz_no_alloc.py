"""dfssm_head_noalloc (include/dfssm.h, csrc/dfssm_noalloc.cu): S8 with its intermediates in the library's static device array
-- no allocation, no context, no arena -- against the existing path (the end of dfssm_step): logits bit for bit, greedy tokens
equal, on calls in a row that share the array (different hidden states, a smaller batch in between, another model shape after).
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import dfssm_synth as ds
from _parity import REL_L2_TOL, n_diff_bits, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from paper_2606_10932_b200 import build
    build.build()
    import paper_2606_10932_b200 as pk
    return dict(torch=torch, pk=pk)


def head_weights(torch, blob):
    _, v = ds.blob_views(blob)
    return tuple(torch.from_numpy(np.ascontiguousarray(v[k])).cuda() for k in ("G.normf_w", "G.emb", "G.emb_s"))


def run_case(env, s, blob, seed, B, n_steps=3):
    """n_steps decode steps through the existing path; after each one the new entry point is given the same hidden state."""
    torch, pk = env["torch"], env["pk"]
    m = pk.Model(pk.Config.from_shape(s, max_batch=B), blob)
    normf_w, emb, emb_s = head_weights(torch, blob)
    toks = np.stack([ds.token_stream(s.vocab, n_steps, seed=seed, seq_index=q) for q in range(B)], 1)      # [step][seq]
    nxt = torch.empty(B, dtype=torch.int32, device="cuda")
    lg = torch.empty(B, s.vocab, dtype=torch.float32, device="cuda")
    for t in range(n_steps):
        m.step(torch.from_numpy(np.ascontiguousarray(toks[t], np.int32)).cuda())
        m.sync()
        want_l = m.logits()[:B].cpu().numpy()
        want_t = m.next_tokens()[:B].cpu().numpy()
        hidden = m.hidden()[:B].contiguous()
        free0 = torch.cuda.mem_get_info()[0]
        nxt.fill_(-1)
        lg.fill_(float("nan"))
        pk.head_noalloc(hidden, normf_w, emb, emb_s, nxt, lg, eps=s.norm_eps)
        torch.cuda.synchronize()
        if t > 0:       # (the first call on a device loads the module that holds the static array: CUDA loads modules lazily)
            assert torch.cuda.mem_get_info()[0] == free0, "device memory changed across the call"
        got_l, got_t = lg.cpu().numpy(), nxt.cpu().numpy()
        assert rel_l2(got_l, want_l) <= REL_L2_TOL
        assert n_diff_bits(got_l, want_l) == 0, f"step {t}: {n_diff_bits(got_l, want_l)} logits differ from dfssm_step's"
        assert np.array_equal(got_t, want_t), (t, got_t, want_t)
        if B > 1:       # a smaller call in between leaves other contents in the shared array; tokens only (logits_dev = NULL)
            n1 = torch.full((1,), -1, dtype=torch.int32, device="cuda")
            pk.head_noalloc(hidden[B - 1:B].contiguous(), normf_w, emb, emb_s, n1, None, eps=s.norm_eps)
            torch.cuda.synchronize()
            assert int(n1.item()) == int(want_t[B - 1])
    m.close()


def test_two_calls_in_a_row_equal_the_step_path(env):
    s = ds.shape_for_config(0)                     # d_model 256, vocab 1024
    run_case(env, s, ds.make_blob(s, 0), seed=0, B=5)
    s = ds.tiny_shape(n_layers=2, d_model=96, d_inner=192, headdim=32, d_state=32, ngroups=2, lora_rank=5, vocab=101)      # ragged vocab
    run_case(env, s, ds.make_blob(s, seed=7, variant="varied"), seed=7, B=9)      # two sequence tiles of the LM head


def test_baseline_vocabulary_after_a_small_shape(env):
    """cfg 1 (vocab 50,288, d_model 768) at batch 3 = 0.6 MB of the 4 MiB array, right after calls of other shapes."""
    s = ds.shape_for_config(1)
    run_case(env, s, ds.make_blob(s, 1), seed=1, B=3, n_steps=2)


def test_zero_hidden_state(env):
    """amax = 0: codes and scale 0, every logit +0.0, token 0 (the degenerate case of the quantiser, R4)."""
    torch, pk = env["torch"], env["pk"]
    s = ds.shape_for_config(0)
    normf_w, emb, emb_s = head_weights(torch, ds.make_blob(s, 0))
    nxt = torch.full((2,), -1, dtype=torch.int32, device="cuda")
    lg = torch.full((2, s.vocab), float("nan"), device="cuda")
    pk.head_noalloc(torch.zeros(2, s.d_model, device="cuda"), normf_w, emb, emb_s, nxt, lg, eps=s.norm_eps)
    torch.cuda.synchronize()
    assert not lg.cpu().numpy().view(np.uint32).any() and not nxt.cpu().numpy().any()


def test_limit_and_argument_errors(env):
    torch, pk = env["torch"], env["pk"]
    from paper_2606_10932_b200 import binding
    vocab, d = 50288, 768
    assert pk.head_noalloc_scratch_need(20, d, vocab) <= pk.NOALLOC_SCRATCH_BYTES < pk.head_noalloc_scratch_need(21, d, vocab)
    assert pk.head_noalloc_scratch_need(3, d, vocab) == 2304 + 256 + 3 * 4 * vocab
    emb = torch.zeros(vocab, d, dtype=torch.int8, device="cuda")
    emb_s = torch.ones(vocab, device="cuda")
    w = torch.ones(d, device="cuda")
    B = 21
    with pytest.raises(binding.DfssmError) as ei:
        pk.head_noalloc(torch.ones(B, d, device="cuda"), w, emb, emb_s, torch.empty(B, dtype=torch.int32, device="cuda"))
    assert ei.value.code == -2 and "DFSSM_NOALLOC_SCRATCH_BYTES" in str(ei.value)
    L = pk.lib()
    assert L.dfssm_head_noalloc(None, w.data_ptr(), emb.data_ptr(), emb_s.data_ptr(), 1, d, vocab, 1e-5, emb_s.data_ptr(), None, None) == -1
    assert b"null" in L.dfssm_head_noalloc_error()
    x = torch.ones(1, 40, device="cuda")           # d_model not a multiple of 16
    with pytest.raises(binding.DfssmError) as ei:
        pk.head_noalloc(x, torch.ones(40, device="cuda"), torch.zeros(8, 40, dtype=torch.int8, device="cuda"), torch.ones(8, device="cuda"),
                        torch.empty(1, dtype=torch.int32, device="cuda"))
    assert ei.value.code == -1
    # the failed calls left the entry point usable
    nxt = torch.empty(20, dtype=torch.int32, device="cuda")
    pk.head_noalloc(torch.ones(20, d, device="cuda"), w, emb, emb_s, nxt)      # the largest batch that fits
    torch.cuda.synchronize()
    assert not nxt.cpu().numpy().any()             # all logits equal (0): lowest index
