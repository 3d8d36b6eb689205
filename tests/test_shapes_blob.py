"""Shape calculator and blob layout, pinned to the paper's size table (Table 1)."""
import numpy as np
import pytest

import dfssm_synth as S
from dfssm_synth.blob import read_header


def test_table1_scaffold_155MB():
    # P:95 "Scaffold (48 layers, in+out proj) 1-bit packed 155 MB"
    s = S.shape_for_config(2)
    assert s.d_in_proj == 8512 and s.conv_dim == 4352 and s.nheads == 64
    assert s.scaffold_bytes() == 154_927_104
    assert round(s.scaffold_bytes() / 1e6) == 155


def test_table1_lora_12MB_at_rank16():
    # P:97 "LoRA correction (48 layers, r=16) int8 12 MB"; 12.83 MB exact, printed as 12
    s = S.shape_for_config(2).with_(lora_rank=16)
    assert s.lora_bytes() == 48 * 16 * (2048 + 8512 + 4096 + 2048)
    assert 12.0e6 <= s.lora_bytes() < 13.0e6


def test_table1_embedding_103MB():
    # P:96 "Embedding + LM head (tied) int8 103 MB"
    s = S.shape_for_config(2)
    assert s.embedding_bytes() == 102_989_824
    assert round(s.embedding_bytes() / 1e6) == 103


def _golden(name):
    from pathlib import Path
    rows = {}
    for line in (Path(__file__).parent / "golden" / name).read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            rows[k] = v
    return rows


def test_table1_fixture_is_consistent_and_matches_the_shape_calculator():
    """tests/golden/paper_table1_sizes.txt = Table 1 as printed: the printed total is the sum of the printed
    components, the printed ratio is teacher / total, the printed fractions are size / total, and the three components the
    shape fixes (scaffold, tied embedding, rank-16 LoRA) come out of dfssm_synth's byte counts."""
    t = _golden("paper_table1_sizes.txt")
    size = {k: float(v[0]) for k, v in t.items()}
    parts = ("scaffold_1bit_packed", "embedding_lm_head_tied_int8", "lora_r16_int8", "other_conv_norms_ssm")
    assert sum(size[k] for k in parts) == size["total"] == 278
    assert round(size["teacher_fp16"] / size["total"], 1) == size["compression_ratio"]
    for k in parts:
        assert round(100 * size[k] / size["total"]) == int(t[k][1]), k
    s = S.shape_for_config(2)
    assert round(s.scaffold_bytes() / 1e6) == size["scaffold_1bit_packed"]
    assert round(s.embedding_bytes() / 1e6) == size["embedding_lm_head_tied_int8"]
    assert int(s.with_(lora_rank=16).lora_bytes() / 1e6) == size["lora_r16_int8"]        # 12.83 MB, printed as 12
    # the teacher: 1.3B parameters in FP16 ("A 1.3B parameter model in FP16 requires 2.7 GB")
    assert abs(size["teacher_fp16"] / 2 - 1344) < 1


def test_state_524k_elements_per_layer():
    # P:13 "fixed-size hidden state (524 KB for Mamba-2 1.3B)" = 64*64*128 elements of one layer
    c = {k: int(v[0]) for k, v in _golden("paper_constants.txt").items()}
    assert S.shape_for_config(2).ssm_state_elems_per_layer() == 524_288
    assert S.shape_for_config(2).ssm_state_elems_per_layer() // 1000 == c["state_kb_per_layer_1p3b"]
    assert S.shape_for_config(2).n_layers == c["n_layers_1p3b"]


def test_vnni_row_is_32_instructions():
    # P:138 "32 VPDPBUSD instructions per 2048-element row": 64 weights per instruction
    c = {k: int(v[0]) for k, v in _golden("paper_constants.txt").items()}
    assert S.shape_for_config(2).d_model // 64 == c["vpdpbusd_per_2048_row"]


@pytest.mark.parametrize("idx,dip,cd", [(0, 1160, 640), (1, 3352, 1792), (2, 8512, 4352), (4, 10576, 5376)])
def test_derived_widths(idx, dip, cd):
    s = S.shape_for_config(idx)
    assert (s.d_in_proj, s.conv_dim) == (dip, cd)


def test_blob_roundtrip_and_alignment():
    s = S.tiny_shape(n_layers=2)
    blob = S.make_blob(s, seed=3, variant="varied")
    assert blob.nbytes == S.blob_nbytes(s)
    hdr = read_header(blob)
    assert hdr.with_(norm_eps=s.norm_eps) == s and np.float32(hdr.norm_eps) == np.float32(s.norm_eps)
    layout, total = S.blob_layout(s)
    assert total % 64 == 0
    prev_end = S.HEADER_BYTES
    for name, (off, dt, shp) in layout.items():
        assert off % 64 == 0 and off >= prev_end
        prev_end = off + int(np.prod(shp)) * dt.itemsize
    _, v = S.blob_views(blob)
    assert v["L1.in.sign"].shape == (s.d_in_proj, s.d_model // 32) and v["L1.in.sign"].dtype == np.uint32
    assert v["G.emb"].dtype == np.int8 and v["G.emb"].min() >= -127
    # deterministic: same seed -> same bytes; another seed -> different bytes
    assert np.array_equal(blob, S.make_blob(s, seed=3, variant="varied"))
    assert not np.array_equal(blob, S.make_blob(s, seed=4, variant="varied"))


def test_baseline_distributions_cfg0():
    # BASELINE.json config 0 weight recipe
    s = S.shape_for_config(0)
    _, v = S.blob_views(S.make_blob(s, 0))
    bits = np.unpackbits(v["L0.in.sign"].view(np.uint8))
    assert abs(bits.mean() - 0.5) < 0.01
    rs = v["L0.in.row_scale"].astype(np.float64)
    assert rs.min() >= 0 and abs(rs.mean() - 0.02 * np.sqrt(2 / np.pi)) < 2e-3
    assert np.all(v["L0.in.a_s"] == np.float32(1e-3)) and np.all(v["L1.out.b_s"] == np.float32(1e-3))
    A = v["L0.in.A"]
    assert A.min() == -127 and A.max() == 127
    a = np.exp(v["L0.A_log"].astype(np.float64))
    assert a.min() >= 1 and a.max() <= 16
    dt0 = np.log1p(np.exp(v["L0.dt_bias"].astype(np.float64)))
    assert dt0.min() >= 1e-3 * 0.999 and dt0.max() <= 1e-1 * 1.001
    assert np.all(v["L0.D"] == 1) and np.all(v["L0.norm_w"] == 1) and np.all(v["L0.conv_b"] == 0)
    assert abs(v["L0.conv_w"].std() - 0.2) < 0.02
    es = v["G.emb_s"] * 127
    assert es.min() >= 0.5 and es.max() < 1.5


def test_token_streams():
    a = S.token_stream(1024, 64, seed=0)
    assert a.dtype == np.int32 and a.min() >= 0 and a.max() < 1024
    assert np.array_equal(a, S.token_stream(1024, 64, seed=0))
    tb = S.token_batch(1024, 8, seed=0, batch=3)
    assert tb.shape == (8, 3) and np.array_equal(tb[:, 0], a[:8])
    assert not np.array_equal(tb[:, 0], tb[:, 1])
