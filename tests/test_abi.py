"""CPU-side checks of the boundary: libdfssm.so builds for sm_100a, loads, and exports exactly the
symbols include/dfssm.h declares; the binding mirrors them; host-only calls behave."""
import ctypes
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def built():
    from paper_2606_10932_b200 import build
    return build.build()


def _header_functions():
    text = (ROOT / "include" / "dfssm.h").read_text()
    return sorted(set(re.findall(r"DFSSM_API[^;(]*?\b(dfssm_\w+)\s*\(", text)))


def test_header_declares_the_five_named_calls():
    names = _header_functions()
    for must in ("dfssm_create", "dfssm_load_weights", "dfssm_reset_state", "dfssm_step", "dfssm_logits"):
        assert must in names


def test_library_exports_every_declared_symbol(built):
    names = _header_functions()
    L = ctypes.CDLL(str(built))
    for n in names:
        assert hasattr(L, n), f"{n} declared in dfssm.h but not exported"
    out = subprocess.run(["nm", "-D", "--defined-only", str(built)], capture_output=True, text=True, check=True).stdout
    exported = sorted(set(re.findall(r"\bT (dfssm_\w+)", out)))
    assert exported == names, (exported, names)


def test_binding_mirrors_header(built):
    from paper_2606_10932_b200 import EXPORTED_SYMBOLS, lib
    assert sorted(EXPORTED_SYMBOLS) == _header_functions()
    L = lib()
    for n in EXPORTED_SYMBOLS:
        assert getattr(L, n).argtypes is not None


def test_library_is_sm100a_only(built):
    out = subprocess.run(["cuobjdump", "-lelf", str(built)], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out), out


def test_arena_bytes_host_only(built):
    import dfssm_synth as ds
    from paper_2606_10932_b200 import Config, dfssm_arena_bytes
    s = ds.shape_for_config(2)
    n1 = dfssm_arena_bytes(Config.from_shape(s, max_batch=1))
    n2 = dfssm_arena_bytes(Config.from_shape(s, max_batch=2))
    assert n1 > ds.blob_nbytes(s)
    # one more sequence = one more fp32 SSM state + conv ring per layer (+ small activations)
    per_seq = s.n_layers * (s.ssm_state_elems_per_layer() * 4 + s.conv_dim * 16)
    assert per_seq <= n2 - n1 <= per_seq + 4 * (s.vocab + 8 * s.d_in_proj) + 65536
    bad = Config.from_shape(s.with_(d_model=2050))
    assert dfssm_arena_bytes(bad) == 0
    assert dfssm_arena_bytes(Config.from_shape(s, max_batch=0)) == 0


def test_no_cpu_fallback_without_gpu(built):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import dfssm_synth as ds
    from paper_2606_10932_b200 import Config, DfssmError, Model
    with pytest.raises(DfssmError):
        Model(Config.from_shape(ds.shape_for_config(0)))


def test_product_does_not_import_oracle():
    for p in (ROOT / "paper_2606_10932_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            t = p.read_text()
            assert "oracle" not in t.replace("no oracle", ""), f"{p} mentions the oracle"
