"""Pins for the oracle's integer parts and the quantiser (no GPU).

Each test checks an oracle function against something other than itself: a dense +-1 float
matvec, a closed form, an invariant, a hand-computed example.  Citations: P:NN = PAPER.md line.
"""
import numpy as np
import pytest


def _unpack_pm1(sign_words):
    """[rows][W] uint32 -> dense [rows][32W] float64 of +-1; bit b (LSB=0) of word w <-> k = 32w+b."""
    rows, W = sign_words.shape
    bits = np.unpackbits(sign_words.astype("<u4").view(np.uint8).reshape(rows, W * 4), axis=1, bitorder="little")
    return bits.astype(np.float64) * 2.0 - 1.0


# ---------------------------------------------------------------- packed sign matvec (S2/S7)
@pytest.mark.parametrize("rows,K", [(1, 32), (5, 64), (17, 96), (40, 256)])
def test_sign_matvec_equals_dense_pm1(oracle_mod, rows, K):
    # BASELINE.json check 1; P:134-136 every packed bit becomes exactly +-1
    g = np.random.default_rng(rows * 1000 + K)
    sign = g.integers(0, 1 << 32, size=(rows, K // 32), dtype=np.uint32)
    xq = g.integers(-127, 128, size=K, dtype=np.int8)
    dense = _unpack_pm1(sign) @ xq.astype(np.float64)
    acc = oracle_mod.sign_matvec(sign, xq)
    assert acc.dtype == np.int32
    assert np.array_equal(acc.astype(np.float64), dense)


def test_sign_matvec_special_rows_and_bit_order(oracle_mod):
    g = np.random.default_rng(1)
    K = 128
    xq = g.integers(-127, 128, size=K, dtype=np.int8)
    sign = np.zeros((3, K // 32), np.uint32)
    sign[0, :] = 0xFFFFFFFF            # all +1 -> sum q
    sign[1, :] = 0                     # all -1 -> -sum q
    sign[2, :] = 0
    sign[2, 1] = np.uint32(1) << 5     # only element k = 32*1 + 5 is +1
    acc = oracle_mod.sign_matvec(sign, xq)
    sq = int(xq.astype(np.int64).sum())
    assert acc[0] == sq and acc[1] == -sq
    assert acc[2] == -sq + 2 * int(xq[37])          # flipping one bit changes acc by exactly 2*q_k
    # identity sum_k s_k q_k = 2*sum_{bit=1} q_k - sum_k q_k on a random row
    row = g.integers(0, 1 << 32, size=(1, K // 32), dtype=np.uint32)
    bits = np.unpackbits(row.view(np.uint8), bitorder="little").astype(bool)
    assert oracle_mod.sign_matvec(row, xq)[0] == 2 * int(xq[bits].astype(np.int64).sum()) - sq


def test_sign_matvec_extreme_magnitude(oracle_mod):
    # |acc| <= 127*K, reached when signs align with the activations
    K = 4096
    xq = np.full(K, 127, np.int8)
    xq[::2] = -127
    sign = np.zeros((1, K // 32), np.uint32)
    sign[0, :] = 0xAAAAAAAA            # bit set at odd k where xq = +127
    assert oracle_mod.sign_matvec(sign, xq)[0] == 127 * K


# ---------------------------------------------------------------- quantiser (S1/S6/S8)
def test_quantiser_invariants(oracle_mod):
    g = np.random.default_rng(2)
    d = 256
    v = (g.standard_normal(d) * 3).astype(np.float32)
    w = g.uniform(0.5, 1.5, d).astype(np.float32)
    q, s, rstd, amax = oracle_mod.norm_quant(v, w, 1e-5)
    t = v.astype(np.float64) * w.astype(np.float64)
    # rstd is 1/sqrt(mean(v^2)+eps)
    assert abs(rstd - 1.0 / np.sqrt(np.mean(v.astype(np.float64) ** 2) + 1e-5)) < 1e-6 * rstd
    assert amax == np.float32(np.abs((v * w)).max())
    # the arg-max element maps to +-127, all codes within +-127
    k = int(np.abs(v * w).argmax())
    assert abs(int(q[k])) == 127 and np.abs(q.astype(np.int32)).max() == 127
    assert np.sign(q[k]) == np.sign(t[k])
    # reconstruction error at most half a step: |t - (amax/127) q| <= (amax/127)/2
    step = float(amax) / 127.0
    assert np.max(np.abs(t - step * q.astype(np.float64))) <= 0.5 * step * (1 + 1e-5)
    # s * q ~= v * rstd * w  (what the projections consume)
    assert abs(s - step * float(rstd)) <= 1e-6 * s
    # scaling v by 2 leaves q unchanged (power of two: exact)
    q2, s2, rstd2, amax2 = oracle_mod.norm_quant(2 * v, w, 0.0)
    q1, s1, _, _ = oracle_mod.norm_quant(v, w, 0.0)
    assert np.array_equal(q2, q1) and abs(s2 - s1) <= 2e-7 * s1 and amax2 == 2 * amax
    # zero vector -> zero codes, zero scale
    qz, sz, _, az = oracle_mod.norm_quant(np.zeros(d, np.float32), w, 1e-5)
    assert not qz.any() and sz == 0.0 and az == 0.0


def test_quantiser_ties_to_even_and_sign(oracle_mod):
    # amax = 127 -> inv = 1 exactly, so the codes are rint(v): .5 ties go to the even integer
    v = np.array([127.0, 0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 3.49, -126.5, 0.0], np.float32)
    q, s, rstd, amax = oracle_mod.norm_quant(v, np.ones_like(v), 0.0)
    assert amax == 127.0
    assert q.tolist() == [127, 0, 2, 2, 0, -2, -2, 3, -126, 0]


def test_quantiser_constant_vector_closed_form(oracle_mod):
    # RMSNorm of a constant vector c: c*rstd = sign(c)/sqrt(1+eps/c^2); all codes +-127
    for c in (0.25, -3.0):
        v = np.full(64, c, np.float32)
        w = np.full(64, 1.5, np.float32)
        q, s, rstd, _ = oracle_mod.norm_quant(v, w, 1e-5)
        assert np.all(q == (127 if c > 0 else -127))
        want = 1.5 * np.sign(c) / np.sqrt(1 + 1e-5 / c ** 2)
        assert abs(float(s) * float(q[0]) - want) < 1e-6 * abs(want)


# ---------------------------------------------------------------- LoRA (S3)
def test_lora_down_equals_int_matmul(oracle_mod):
    g = np.random.default_rng(3)
    r, K = 7, 160
    A = g.integers(-127, 128, size=(r, K), dtype=np.int8)
    xq = g.integers(-127, 128, size=K, dtype=np.int8)
    t = oracle_mod.lora_down(A, xq)
    assert np.array_equal(t.astype(np.int64), A.astype(np.int64) @ xq.astype(np.int64))
    # bound |t| <= 127^2 K reached
    A[:] = 127
    xq[:] = -127
    assert oracle_mod.lora_down(A, xq)[0] == -127 * 127 * K


def test_proj_epilogue_dense_and_special_cases(oracle_mod):
    # Eq. 3: y = W_scaffold x + W_A (W_B x); here out = s_x*(w_s*acc + b_s * B.(a_s*t))
    g = np.random.default_rng(4)
    rows, r = 23, 5
    acc = g.integers(-20000, 20000, size=rows, dtype=np.int32)
    t = g.integers(-3_000_000, 3_000_000, size=r, dtype=np.int32)
    rs = (np.abs(g.standard_normal(rows)) * 0.02).astype(np.float16)
    a_s = g.uniform(5e-4, 2e-3, r).astype(np.float32)
    b_s = g.uniform(5e-4, 2e-3, rows).astype(np.float32)
    B = g.integers(-127, 128, size=(rows, r), dtype=np.int8)
    s_x = 0.0173
    out = oracle_mod.proj_epilogue(acc, t, rs, a_s, B, b_s, s_x)
    f = np.float64
    dense = f(np.float32(s_x)) * (rs.astype(f) * acc.astype(f)
                                  + b_s.astype(f) * (B.astype(f) @ (a_s.astype(f) * t.astype(f))))
    assert np.allclose(out, dense, rtol=2e-6, atol=1e-9)
    # B = 0 or t = 0 -> scaffold only
    only = f(np.float32(s_x)) * rs.astype(f) * acc.astype(f)
    assert np.allclose(oracle_mod.proj_epilogue(acc, t, rs, a_s, np.zeros_like(B), b_s, s_x), only, rtol=1e-6)
    assert np.allclose(oracle_mod.proj_epilogue(acc, np.zeros_like(t), rs, a_s, B, b_s, s_x), only, rtol=1e-6)
    # acc = 0 -> LoRA only
    lo = f(np.float32(s_x)) * b_s.astype(f) * (B.astype(f) @ (a_s.astype(f) * t.astype(f)))
    assert np.allclose(oracle_mod.proj_epilogue(np.zeros_like(acc), t, rs, a_s, B, b_s, s_x), lo, rtol=2e-6)


def test_proj_epilogue_rank1_hand_example(oracle_mod):
    # rank 1, numbers chosen to be exact in binary32: acc=8, w_s=0.5; t=4, a_s=0.25, B=[2,-3], b_s=0.5; s_x=2
    acc = np.array([8, -4], np.int32)
    out = oracle_mod.proj_epilogue(acc, np.array([4], np.int32), np.array([0.5, 0.25], np.float16),
                                   np.array([0.25], np.float32), np.array([[2], [-3]], np.int8),
                                   np.array([0.5, 0.5], np.float32), 2.0)
    # row0: 2*(0.5*8 + 0.5*(2*1)) = 10 ; row1: 2*(0.25*-4 + 0.5*(-3*1)) = -5
    assert out.tolist() == [10.0, -5.0]


# ---------------------------------------------------------------- LM head / argmax (S8), embed (S0)
def test_lm_head_dense_ties_permutation(oracle_mod):
    g = np.random.default_rng(5)
    V, d = 37, 96
    E = g.integers(-127, 128, size=(V, d), dtype=np.int8)
    e_s = (g.uniform(0.5, 1.5, V) / 127).astype(np.float32)
    hq = g.integers(-127, 128, size=d, dtype=np.int8)
    acc, logits = oracle_mod.lm_head(E, e_s, hq, 0.031)
    assert np.array_equal(acc.astype(np.int64), E.astype(np.int64) @ hq.astype(np.int64))
    want = acc.astype(np.float64) * (np.float64(np.float32(0.031)) * e_s.astype(np.float64))
    assert np.allclose(logits, want, rtol=3e-7, atol=0)
    perm = g.permutation(V)
    acc_p, logits_p = oracle_mod.lm_head(E[perm], e_s[perm], hq, 0.031)
    assert np.array_equal(acc_p, acc[perm]) and np.array_equal(logits_p, logits[perm])
    assert oracle_mod.argmax(logits) == int(np.argmax(logits))
    # ties -> lowest index
    assert oracle_mod.argmax(np.array([1.0, 3.0, 3.0, 2.0, 3.0], np.float32)) == 1
    assert oracle_mod.argmax(np.array([-0.0, 0.0, -1.0], np.float32)) == 0


def test_embed_row_scale(oracle_mod):
    row = np.array([-127, 0, 1, 64], np.int8)
    assert oracle_mod.embed(row, 0.5).tolist() == [-63.5, 0.0, 0.5, 32.0]
