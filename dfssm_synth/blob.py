"""Canonical DF-SSM weight blob: byte layout, writer, and numpy views.

Little-endian.  A 256-byte header, then tensors in a fixed order, every tensor
starting on a 64-byte boundary (zero padding between).  The oracle (C) and the CUDA
library (C++) each parse this layout with their own code.

Header:
    off  0  char[8]  magic "DFSSMW1\\0"
    off  8  u32      blob version (1)
    off 12  i32 x 9  n_layers, d_model, d_inner, headdim, d_state, ngroups, d_conv,
                     vocab, lora_rank
    off 48  f32      norm_eps
    off 52  u32      weight format: bit 0 = 17-level scaffold, bit 1 = int4 LoRA (0 = the paper's deployed format)
    off 56  u64      total blob bytes
    off 64..255      0

Sign matrices: row-major [rows][K/32] uint32; bit b (LSB = 0) of word w of row i is
element k = 32*w + b; bit 1 -> +1, bit 0 -> -1 (every packed bit
expands to exactly +-1).

Format variants (R25):
  17-level scaffold: instead of `sign`, `lvl` = [rows][K/32][5] uint32.  The weight of element k = 32*w + b is level/8 with
    level = m - 8 in [-8, 8] (Eq. 1 with K_w = 16: {-1, -14/16, ..., 1}); bit b of word [w][p] is bit p of m.
    `row_scale` multiplies the INTEGER accumulator sum(level * q), i.e. it holds the paper's row scale / 8.
  int4 LoRA: `A4` = [r][K/2], `B4` = [rows][r/2] uint8; element 2i is the low nibble of byte i, element 2i+1 the high
    nibble, each a two's-complement 4-bit integer in [-8, 7].
"""
from __future__ import annotations

import struct
from typing import Dict, List, Tuple

import numpy as np

from .shapes import Shape, FMT_SCAFFOLD17, FMT_LORA_INT4

BLOB_MAGIC = b"DFSSMW1\0"
BLOB_VERSION = 1
HEADER_BYTES = 256
TENSOR_ALIGN = 64

Spec = Tuple[str, np.dtype, Tuple[int, ...]]


def layer_tensor_specs(s: Shape) -> List[Spec]:
    r = s.lora_rank
    u32, f16, f32, i8, u8 = np.dtype("<u4"), np.dtype("<f2"), np.dtype("<f4"), np.dtype("i1"), np.dtype("u1")
    s17, i4 = bool(s.fmt & FMT_SCAFFOLD17), bool(s.fmt & FMT_LORA_INT4)

    def scaffold(side, rows, K):
        return (f"{side}.lvl", u32, (rows, K // 32, 5)) if s17 else (f"{side}.sign", u32, (rows, K // 32))

    def lora_a(side, K):
        return (f"{side}.A4", u8, (r, K // 2)) if i4 else (f"{side}.A", i8, (r, K))

    def lora_b(side, rows):
        return (f"{side}.B4", u8, (rows, r // 2)) if i4 else (f"{side}.B", i8, (rows, r))

    return [
        ("norm_w", f32, (s.d_model,)),
        scaffold("in", s.d_in_proj, s.d_model),
        ("in.row_scale", f16, (s.d_in_proj,)),
        lora_a("in", s.d_model),
        ("in.a_s", f32, (r,)),
        lora_b("in", s.d_in_proj),
        ("in.b_s", f32, (s.d_in_proj,)),
        ("conv_w", f32, (s.conv_dim, 4)),
        ("conv_b", f32, (s.conv_dim,)),
        ("A_log", f32, (s.nheads,)),
        ("dt_bias", f32, (s.nheads,)),
        ("D", f32, (s.nheads,)),
        ("gnorm_w", f32, (s.d_inner,)),
        scaffold("out", s.d_model, s.d_inner),
        ("out.row_scale", f16, (s.d_model,)),
        lora_a("out", s.d_inner),
        ("out.a_s", f32, (r,)),
        lora_b("out", s.d_model),
        ("out.b_s", f32, (s.d_model,)),
    ]


# ---- packing of the format variants (byte layout only) ----
def pack_levels(levels: np.ndarray) -> np.ndarray:
    """int levels in [-8, 8], [rows][K] -> uint32 [rows][K/32][5] bit planes of m = level + 8"""
    lv = np.asarray(levels).astype(np.int64)
    assert lv.ndim == 2 and lv.shape[1] % 32 == 0 and lv.min() >= -8 and lv.max() <= 8
    m = (lv + 8).reshape(lv.shape[0], -1, 32).astype(np.uint64)
    w = (np.uint64(1) << np.arange(32, dtype=np.uint64))
    planes = [(((m >> np.uint64(p)) & np.uint64(1)) * w).sum(-1) for p in range(5)]
    return np.stack(planes, -1).astype("<u4")


def unpack_levels(lvl: np.ndarray) -> np.ndarray:
    """uint32 [rows][K/32][5] -> int8 levels [rows][K]"""
    lvl = np.asarray(lvl, dtype=np.uint32)
    bits = (lvl[:, :, None, :] >> np.arange(32, dtype=np.uint32)[None, None, :, None]) & 1       # [rows][W][32][5]
    m = (bits.astype(np.int64) << np.arange(5)[None, None, None, :]).sum(-1)
    return (m - 8).reshape(lvl.shape[0], -1).astype(np.int8)


def pack_int4(a: np.ndarray) -> np.ndarray:
    """int values in [-8, 7], [n][m] (m even) -> uint8 [n][m/2]: element 2i = low nibble of byte i"""
    a = np.asarray(a).astype(np.int64)
    assert a.ndim == 2 and a.shape[1] % 2 == 0 and a.min() >= -8 and a.max() <= 7
    n = (a & 0xF).astype(np.uint8)
    return (n[:, 0::2] | (n[:, 1::2] << 4)).astype(np.uint8)


def unpack_int4(b: np.ndarray) -> np.ndarray:
    b = np.asarray(b, dtype=np.uint8)
    out = np.empty((b.shape[0], 2 * b.shape[1]), np.int16)
    out[:, 0::2] = b & 0xF
    out[:, 1::2] = b >> 4
    return ((out ^ 8) - 8).astype(np.int8)


def global_tensor_specs(s: Shape) -> List[Spec]:
    f32, i8 = np.dtype("<f4"), np.dtype("i1")
    return [
        ("emb", i8, (s.vocab, s.d_model)),
        ("emb_s", f32, (s.vocab,)),
        ("normf_w", f32, (s.d_model,)),
    ]


def _align(x: int) -> int:
    return (x + TENSOR_ALIGN - 1) // TENSOR_ALIGN * TENSOR_ALIGN


def blob_layout(s: Shape) -> Tuple[Dict[str, Tuple[int, np.dtype, Tuple[int, ...]]], int]:
    """name -> (byte offset, dtype, shape); names are 'L{l}.{tensor}' and 'G.{tensor}'."""
    off = HEADER_BYTES
    out: Dict[str, Tuple[int, np.dtype, Tuple[int, ...]]] = {}
    for l in range(s.n_layers):
        for name, dt, shp in layer_tensor_specs(s):
            off = _align(off)
            out[f"L{l}.{name}"] = (off, dt, shp)
            off += int(np.prod(shp)) * dt.itemsize
    for name, dt, shp in global_tensor_specs(s):
        off = _align(off)
        out[f"G.{name}"] = (off, dt, shp)
        off += int(np.prod(shp)) * dt.itemsize
    return out, _align(off)


def blob_nbytes(s: Shape) -> int:
    return blob_layout(s)[1]


def _header(s: Shape, total: int) -> bytes:
    h = bytearray(HEADER_BYTES)
    h[0:8] = BLOB_MAGIC
    struct.pack_into("<I9ifIQ", h, 8, BLOB_VERSION, s.n_layers, s.d_model, s.d_inner, s.headdim,
                     s.d_state, s.ngroups, s.d_conv, s.vocab, s.lora_rank, float(s.norm_eps), int(s.fmt), total)
    return bytes(h)


def write_blob(s: Shape, tensors: Dict[str, np.ndarray]) -> np.ndarray:
    """Pack named tensors into one uint8 array in the canonical layout."""
    s.validate()
    layout, total = blob_layout(s)
    buf = np.zeros(total, dtype=np.uint8)
    buf[:HEADER_BYTES] = np.frombuffer(_header(s, total), dtype=np.uint8)
    missing = set(layout) - set(tensors)
    assert not missing, f"missing tensors: {sorted(missing)[:4]}..."
    for name, (off, dt, shp) in layout.items():
        a = np.ascontiguousarray(tensors[name])
        assert a.shape == tuple(shp), (name, a.shape, shp)
        assert a.dtype == dt, (name, a.dtype, dt)
        buf[off:off + a.nbytes] = a.reshape(-1).view(np.uint8)
    return buf


def read_header(blob: np.ndarray) -> Shape:
    raw = bytes(blob[:HEADER_BYTES])
    assert raw[0:8] == BLOB_MAGIC, "bad magic"
    ver, nl, dm, di, hd, ds, ng, dc, vo, r, eps, fmt, total = struct.unpack_from("<I9ifIQ", raw, 8)
    assert ver == BLOB_VERSION
    assert total == blob.nbytes, (total, blob.nbytes)
    return Shape(nl, dm, di, hd, ds, ng, dc, vo, r, eps, fmt)


def blob_views(blob: np.ndarray) -> Tuple[Shape, Dict[str, np.ndarray]]:
    """Zero-copy numpy views of every tensor in a blob (tests build dense references from these)."""
    s = read_header(blob)
    layout, total = blob_layout(s)
    assert total == blob.nbytes
    views = {}
    for name, (off, dt, shp) in layout.items():
        n = int(np.prod(shp)) * dt.itemsize
        views[name] = blob[off:off + n].view(dt).reshape(shp)
    return s, views
