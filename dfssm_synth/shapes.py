"""Model shapes of BASELINE.json's five configs (Mamba-2-shaped DF-SSM).

Derived widths follow the Mamba-2 mixer the paper builds on and
are pinned by the paper's size table (Table 1): with
``d_in_proj = 2*d_inner + 2*ngroups*d_state + nheads`` the packed 1.3B scaffold is
154.93 MB, the paper's "155 MB".
"""
from __future__ import annotations

from dataclasses import dataclass, replace


FMT_SCAFFOLD17 = 1            # 17-level scaffold {-1, -14/16, ..., 1} (Eq. 1 / Eq. 3) as five bit planes
FMT_LORA_INT4 = 2             # int4 LoRA matrices (Table 4), two values per byte


@dataclass(frozen=True)
class Shape:
    n_layers: int
    d_model: int
    d_inner: int
    headdim: int
    d_state: int
    ngroups: int
    d_conv: int
    vocab: int
    lora_rank: int
    norm_eps: float = 1e-5
    fmt: int = 0              # weight format variants: FMT_SCAFFOLD17 | FMT_LORA_INT4; 0 = 1-bit scaffold, int8 LoRA

    @property
    def nheads(self) -> int:
        return self.d_inner // self.headdim

    @property
    def d_in_proj(self) -> int:
        # z | x | B | C | dt
        return 2 * self.d_inner + 2 * self.ngroups * self.d_state + self.nheads

    @property
    def conv_dim(self) -> int:
        # x | B | C go through the depthwise conv
        return self.d_inner + 2 * self.ngroups * self.d_state

    def validate(self) -> None:
        assert self.d_conv == 4, "only the 4-tap conv of the paper's model is supported"
        assert self.d_model % 32 == 0 and self.d_inner % 32 == 0
        assert self.d_inner % self.headdim == 0
        assert self.nheads % self.ngroups == 0
        assert self.lora_rank >= 1 and self.vocab >= 1 and self.n_layers >= 0
        assert 0 <= self.fmt <= 3
        if self.fmt & FMT_LORA_INT4:
            assert self.lora_rank % 2 == 0, "int4 LoRA packs two values per byte"

    # ---- byte counts used by tests (Table 1 pins) and by bench.py's roofline ----
    def scaffold_bytes(self) -> int:
        per_layer = (self.d_in_proj * self.d_model + self.d_model * self.d_inner) // 8
        return self.n_layers * per_layer * (5 if self.fmt & FMT_SCAFFOLD17 else 1)

    def lora_bytes(self) -> int:
        r = self.lora_rank
        per_layer = r * (self.d_model + self.d_in_proj + self.d_inner + self.d_model)
        return self.n_layers * per_layer // (2 if self.fmt & FMT_LORA_INT4 else 1)

    def embedding_bytes(self) -> int:
        return self.vocab * self.d_model

    def ssm_state_elems_per_layer(self) -> int:
        return self.nheads * self.headdim * self.d_state

    def with_(self, **kw) -> "Shape":
        return replace(self, **kw)


# BASELINE.json `configs`, index -> shape.  cfg 3 shares cfg 2's shape (batch sweep).
CONFIGS = {
    0: Shape(n_layers=2, d_model=256, d_inner=512, headdim=64, d_state=64, ngroups=1,
             d_conv=4, vocab=1024, lora_rank=8),
    1: Shape(n_layers=24, d_model=768, d_inner=1536, headdim=64, d_state=128, ngroups=1,
             d_conv=4, vocab=50288, lora_rank=16),
    2: Shape(n_layers=48, d_model=2048, d_inner=4096, headdim=64, d_state=128, ngroups=1,
             d_conv=4, vocab=50288, lora_rank=32),
    3: Shape(n_layers=48, d_model=2048, d_inner=4096, headdim=64, d_state=128, ngroups=1,
             d_conv=4, vocab=50288, lora_rank=32),
    4: Shape(n_layers=64, d_model=2560, d_inner=5120, headdim=64, d_state=128, ngroups=1,
             d_conv=4, vocab=50288, lora_rank=32),
}

# name -> (config index, run recipe) as BASELINE.json states them
RUNS = {
    0: dict(name="tiny", prompt=0, decode=16, batches=(1,)),
    1: dict(name="130M", prompt=128, decode=256, batches=(1,)),
    2: dict(name="1.3B", prompt=128, decode=512, batches=(1,)),
    3: dict(name="1.3B-batch-sweep", prompt=0, decode=256, batches=(1, 4, 16, 64)),
    4: dict(name="2.7B", prompt=64, decode=512, batches=(1, 8)),
}


def shape_for_config(idx: int) -> Shape:
    s = CONFIGS[idx]
    s.validate()
    return s


def tiny_shape(**kw) -> Shape:
    """A small shape for unit tests; any field can be overridden."""
    base = dict(n_layers=1, d_model=64, d_inner=128, headdim=32, d_state=16, ngroups=1,
                d_conv=4, vocab=96, lora_rank=4)
    base.update(kw)
    s = Shape(**base)
    s.validate()
    return s
