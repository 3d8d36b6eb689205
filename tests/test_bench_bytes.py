"""The roofline numerator of bench.py: algorithmic bytes per step, pinned to the paper's Table 1 sizes and to the
per-token totals derived from them in SURVEY.md section 8(a) / 8(d)."""
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))

import bench  # noqa: E402
import dfssm_synth as ds  # noqa: E402


def test_cfg2_batch1_bytes_match_the_survey_table():
    s = ds.shape_for_config(2)
    ab = bench.algorithmic_bytes(s, 1)
    assert ab["scaffold"] == 48 * (8512 * 2048 + 2048 * 4096) // 8 == 154_927_104        # "155 MB"
    assert ab["lora"] == 48 * 32 * (2048 + 8512 + 4096 + 2048)                            # rank 32: twice the "12 MB" of rank 16
    assert ab["state"] == 48 * 2 * 64 * 64 * 128 * 4 == 201_326_592                      # fp32 state read + written once
    assert ab["lm_head"] == 50288 * 2048 == 102_989_824                                   # "103 MB"
    assert ab["bj_formula"] == ab["scaffold"] + ab["lora"] + ab["state"]
    assert abs(ab["bj_formula"] / 1e6 - 381.9) < 0.1
    assert abs(ab["total"] / 1e6 - 498.6) < 0.5                                           # SURVEY 8(a) totals


@pytest.mark.parametrize("cfg_idx,batch,total_mb", [(1, 1, 93.0), (3, 4, 1117.6), (3, 16, 3593.7), (3, 64, 13498.0), (4, 1, 850.8), (4, 8, 3257.0)])
def test_other_configs_match_the_survey_table(cfg_idx, batch, total_mb):
    s = ds.shape_for_config(cfg_idx)
    ab = bench.algorithmic_bytes(s, batch)
    assert abs(ab["total"] / 1e6 - total_mb) / total_mb < 0.005, ab["total"]     # the table is rounded to 0.1 MB


def test_state_bytes_scale_with_batch_and_weights_do_not():
    s = ds.shape_for_config(3)
    a, b = bench.algorithmic_bytes(s, 1), bench.algorithmic_bytes(s, 64)
    assert b["state"] == 64 * a["state"]
    assert b["scaffold"] == a["scaffold"] and b["lora"] == a["lora"] and b["lm_head"] == a["lm_head"]
    assert b["state"] / b["total"] > 0.94                                                # "95 % of all bytes at batch 64"
