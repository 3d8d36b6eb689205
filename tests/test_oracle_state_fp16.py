"""fp16 state format of the oracle (SURVEY 8(f) NEXT-2 first step, R24): pins of dfo_float_to_half against IEEE 754
binary16 (hand-worked ties, range ends, numpy's float16 conversion) and of the whole-model mode against its definition
(stored state = round(binary32 update); the step's own readout is unrounded)."""
import numpy as np

import dfssm_synth as ds
import oracle
from _parity import rel_l2


def setup_module():
    oracle.build()


def h(x):
    return int(oracle.float_to_half(np.float32(x))[0])


def test_hand_worked_codes():
    """IEEE 754-2019 3.4/3.6 binary16: 1 sign, 5 exponent (bias 15), 10 fraction bits; 4.3.1 roundTiesToEven."""
    assert h(0.0) == 0x0000 and h(-0.0) == 0x8000
    assert h(1.0) == 0x3C00 and h(-2.0) == 0xC000 and h(0.5) == 0x3800
    assert h(65504.0) == 0x7BFF                          # largest finite
    assert h(65519.996) == 0x7BFF                        # below the midpoint to 2^16: stays finite
    assert h(65520.0) == 0x7C00                          # the midpoint ties to the even neighbour = 2^16 = infinity
    assert h(1e9) == 0x7C00 and h(-1e9) == 0xFC00
    assert h(np.inf) == 0x7C00 and h(-np.inf) == 0xFC00
    assert (h(np.nan) & 0x7C00) == 0x7C00 and (h(np.nan) & 0x03FF) != 0
    # ties at 1 + k * 2^-11 (half of the last place 2^-10)
    assert h(1.0 + 2.0 ** -11) == 0x3C00                 # tie -> even (fraction 0)
    assert h(1.0 + 3 * 2.0 ** -11) == 0x3C02             # tie between fraction 1 and 2 -> 2
    assert h(1.0 + 2.0 ** -11 + 2.0 ** -23) == 0x3C01    # just above the tie
    assert h(1.0 + 3 * 2.0 ** -11 - 2.0 ** -23) == 0x3C01
    # subnormals: spacing 2^-24 below 2^-14
    assert h(2.0 ** -14) == 0x0400                       # smallest normal
    assert h(2.0 ** -24) == 0x0001                       # smallest subnormal
    assert h(2.0 ** -25) == 0x0000                       # tie between 0 and 2^-24 -> 0 (even)
    assert h(np.float32(2.0 ** -25) * np.float32(1.0000002)) == 0x0001
    assert h(3 * 2.0 ** -25) == 0x0002                   # tie between 1 and 2 -> 2
    assert h(2.0 ** -14 - 2.0 ** -25) == 0x0400          # the largest subnormal's upper tie rounds into the normal range
    assert h(-(2.0 ** -24)) == 0x8001


def test_against_numpy_float16_conversion():
    """numpy's float32 -> float16 cast is IEEE round-to-nearest-even: a library routine the oracle's bit code does not call."""
    rng = np.random.default_rng(5)
    bits = rng.integers(0, 2 ** 32, 40000, dtype=np.uint64).astype(np.uint32)       # every exponent, both signs
    x = bits.view(np.float32)
    x = x[np.isfinite(x)]
    near = (rng.standard_normal(20000) * np.exp(rng.uniform(-20, 12, 20000))).astype(np.float32)
    halves = rng.integers(0, 0x7C00, 4000, dtype=np.uint16).view(np.float16).astype(np.float32)
    ties = halves + (np.spacing(halves.astype(np.float16)).astype(np.float32) / 2)    # exact midpoints (binary32 holds them)
    for v in (x, near, halves, ties):
        with np.errstate(over="ignore"):
            want = v.astype(np.float16).view(np.uint16)
        got = oracle.float_to_half(v)
        assert np.array_equal(got, want), np.flatnonzero(got != want)[:5]


def _run(blob, toks, fp16):
    m = oracle.OracleModel(blob, 1)
    m.set_state_fp16(fp16)
    out = []
    for t in toks:
        m.step(np.array([t], np.int32))
        out.append((m.logits()[0].copy(), [m.ssm_state(l, 0).copy() for l in range(m.n_layers)]))
    return out


def test_model_mode_follows_its_definition():
    """R24: step 1 from the zero state has the same logits in both modes (the readout uses the unrounded update) and the
    stored state is round(fp32 state); every stored value is binary16-representable at every step; from step 2 on the two
    modes differ, by a small amount."""
    s = ds.tiny_shape(n_layers=3, d_model=64, d_inner=128, headdim=32, d_state=16, lora_rank=4, vocab=97)
    blob = ds.make_blob(s, seed=3, variant="varied")
    toks = ds.token_stream(s.vocab, 24, seed=3, seq_index=0)
    a, b = _run(blob, toks, False), _run(blob, toks, True)
    assert np.array_equal(a[0][0].view(np.uint32), b[0][0].view(np.uint32))
    for l in range(s.n_layers):
        with np.errstate(over="ignore"):
            want = a[0][1][l].astype(np.float16).astype(np.float32)
        assert np.array_equal(want.view(np.uint32), b[0][1][l].view(np.uint32))
        assert a[0][1][l].any()
    for lg, st in b:
        for x in st:
            assert np.array_equal(x.astype(np.float16).astype(np.float32).view(np.uint32), x.view(np.uint32))
    drift = [rel_l2(y[0], x[0]) for x, y in zip(a, b)]
    assert any(d > 0 for d in drift[1:]), "the rounding never reached the logits"
    assert max(drift) < 5e-2, drift
    print("fp16-state drift of the logits over 24 steps (rel L2 vs fp32 state):", " ".join(f"{d:.1e}" for d in drift))
