"""Weight-format variants of the oracle (R25): the 17-level scaffold of PAPER.md Eq. 1 / Eq. 3 and
the int4 LoRA of Table 4.  Pins: dense integer references built with numpy from an independent unpacking (dfssm_synth holds the
byte layout only), hand-worked codes, extreme values, and two cross-format identities that tie the variants to the already
pinned 1-bit / int8 model: a 17-level model whose levels are all +-8 IS the 1-bit model with row scales 8 x larger, and an
int4-LoRA model IS the int8-LoRA model with the same (small) entries -- logits bit for bit."""
import numpy as np
import pytest

import dfssm_synth as ds
import oracle
from dfssm_synth.weights import make_tensors


def setup_module():
    oracle.build()


def test_level_codes_are_eq1_levels():
    """Eq. 1 with K_w = 16: w_q = round(clamp((w+1)/2, 0, 1) * 16) / 16 * 2 - 1 takes exactly the 17 values (m - 8) / 8,
    m = 0..16 -- the integer level the planes hold is 8 * w_q."""
    from pathlib import Path
    txt = [l for l in (Path(__file__).parent / "golden" / "paper_eq1_levels.txt").read_text().splitlines() if l.strip() and not l.startswith("#")]
    sixteenths = [int(v) for v in txt[0].split()]
    assert len(sixteenths) == 17 and sixteenths[0] == -16 and sixteenths[-1] == 16
    w = np.linspace(-1.3, 1.3, 2001)
    m = np.round(np.clip((w + 1) / 2, 0, 1) * 16)
    wq = m / 16 * 2 - 1
    assert sorted(set(np.unique(wq))) == [v / 16 for v in sixteenths] == [(k - 8) / 8 for k in range(17)]
    lv = (m - 8).astype(np.int64)[None, :1984]                       # 1984 = 62 words
    planes = ds.pack_levels(lv)
    one_hot = np.eye(1984, dtype=np.int8)
    got = np.array([oracle.level_matvec(planes, one_hot[k])[0] for k in range(0, 1984, 37)])      # level of element k alone
    assert np.array_equal(got, lv[0, ::37])
    assert np.array_equal(got / 8.0, wq[:1984:37])


def test_level_matvec_hand_worked_planes():
    """one word: element 0 has m = 16 (plane 4 only) -> +8; element 1 has m = 0 -> -8; element 5 has m = 0b01011 = 11 -> +3;
    every other element m = 8 (plane 3) -> 0"""
    pl = np.zeros((1, 1, 5), np.uint32)
    pl[0, 0, 3] = 0xFFFFFFFF & ~((1 << 0) | (1 << 1) | (1 << 5))
    pl[0, 0, 4] = 1 << 0
    pl[0, 0, 0] = 1 << 5
    pl[0, 0, 1] = 1 << 5
    pl[0, 0, 3] |= 1 << 5
    q = np.arange(1, 33, dtype=np.int8)
    assert int(oracle.level_matvec(pl, q)[0]) == 8 * 1 - 8 * 2 + 3 * 6


@pytest.mark.parametrize("rows,K", [(1, 32), (7, 96), (33, 256), (130, 2048)])
def test_level_matvec_vs_dense_integer_matmul(rows, K):
    rng = np.random.default_rng(rows * K)
    lv = rng.integers(-8, 9, size=(rows, K))
    q = rng.integers(-127, 128, size=K).astype(np.int8)
    planes = ds.pack_levels(lv)
    assert np.array_equal(ds.unpack_levels(planes), lv)
    assert np.array_equal(oracle.level_matvec(planes, q), lv.astype(np.int64) @ q.astype(np.int64))
    # extremes: every level +8 against q = 127 and -8 against q = -127
    top = ds.pack_levels(np.full((2, K), 8))
    assert np.array_equal(oracle.level_matvec(top, np.full(K, 127, np.int8)), [8 * 127 * K] * 2)
    bot = ds.pack_levels(np.full((2, K), -8))
    assert np.array_equal(oracle.level_matvec(bot, np.full(K, -127, np.int8)), [8 * 127 * K] * 2)


def test_int4_unpack_every_byte():
    b = np.arange(256, dtype=np.uint8)[None, :]
    got = oracle.unpack_int4(b)[0]
    lo = (np.arange(256) & 15); hi = np.arange(256) >> 4
    sx = lambda n: np.where(n >= 8, n - 16, n)
    assert np.array_equal(got[0::2], sx(lo)) and np.array_equal(got[1::2], sx(hi))
    assert list(oracle.unpack_int4(np.array([[0x8F, 0x70]], np.uint8))[0]) == [-1, -8, 0, 7]
    rng = np.random.default_rng(3)
    a = rng.integers(-8, 8, size=(9, 14))
    assert np.array_equal(oracle.unpack_int4(ds.pack_int4(a)), a) and np.array_equal(ds.unpack_int4(ds.pack_int4(a)), a)


def _logits(blob, toks):
    m = oracle.OracleModel(blob, 1)
    out = []
    for t in toks:
        m.step(np.array([t], np.int32))
        out.append(m.logits()[0].copy())
    return np.stack(out)


def test_17_levels_at_plus_minus_one_are_the_1bit_model():
    s1 = ds.tiny_shape(n_layers=3, d_model=64, d_inner=128, headdim=32, d_state=16, lora_rank=4, vocab=97)
    t1 = make_tensors(s1, 5, "varied")
    s17 = s1.with_(fmt=ds.FMT_SCAFFOLD17)
    t17 = {}
    for k, v in t1.items():
        if k.endswith(".sign"):
            bits = (v[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1
            t17[k[:-5] + ".lvl"] = ds.pack_levels((bits.astype(np.int64) * 16 - 8).reshape(v.shape[0], -1))
        else:
            t17[k] = v
    for k in list(t1):
        if k.endswith("row_scale"):
            t1[k] = (t17[k].astype(np.float32) * 8).astype(np.float16)
            assert np.array_equal(t1[k].astype(np.float32), t17[k].astype(np.float32) * 8)      # exact in binary16
    toks = ds.token_stream(s1.vocab, 12, seed=2)
    a, b = _logits(ds.write_blob(s1, t1), toks), _logits(ds.write_blob(s17, t17), toks)
    assert np.array_equal(a.view(np.uint32), b.view(np.uint32)) and np.abs(a).max() > 0


def test_int4_lora_is_the_int8_model_with_the_same_entries():
    s8 = ds.tiny_shape(n_layers=3, d_model=64, d_inner=128, headdim=32, d_state=16, lora_rank=4, vocab=97)
    s4 = s8.with_(fmt=ds.FMT_LORA_INT4)
    t4 = make_tensors(s4, 6, "varied")
    t8 = {}
    for k, v in t4.items():
        if k.endswith(".A4") or k.endswith(".B4"):
            t8[k[:-1]] = ds.unpack_int4(v)
        else:
            t8[k] = v
    toks = ds.token_stream(s8.vocab, 12, seed=3)
    a, b = _logits(ds.write_blob(s8, t8), toks), _logits(ds.write_blob(s4, t4), toks)
    assert np.array_equal(a.view(np.uint32), b.view(np.uint32)) and np.abs(a).max() > 0
    # and the variant is not a no-op: the 17-level + int4 model differs from the plain one of the same seed
    c = _logits(ds.make_blob(s8, 6, "varied"), toks)
    assert not np.array_equal(a, c)


def test_loader_rejects_bad_format_words():
    s = ds.tiny_shape(fmt=3, lora_rank=4)
    blob = ds.make_blob(s, 1).copy()
    oracle.OracleModel(blob, 1)
    blob[52] = 7
    with pytest.raises(ValueError):
        oracle.OracleModel(blob, 1)
    blob[52] = 0                                   # claims the plain format: the size no longer matches the shape
    with pytest.raises(ValueError):
        oracle.OracleModel(blob, 1)
