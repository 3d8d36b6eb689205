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
    off 52  u32      0
    off 56  u64      total blob bytes
    off 64..255      0

Sign matrices: row-major [rows][K/32] uint32; bit b (LSB = 0) of word w of row i is
element k = 32*w + b; bit 1 -> +1, bit 0 -> -1 (every packed bit
expands to exactly +-1).
"""
from __future__ import annotations

import struct
from typing import Dict, List, Tuple

import numpy as np

from .shapes import Shape

BLOB_MAGIC = b"DFSSMW1\0"
BLOB_VERSION = 1
HEADER_BYTES = 256
TENSOR_ALIGN = 64

Spec = Tuple[str, np.dtype, Tuple[int, ...]]


def layer_tensor_specs(s: Shape) -> List[Spec]:
    r = s.lora_rank
    u32, f16, f32, i8 = np.dtype("<u4"), np.dtype("<f2"), np.dtype("<f4"), np.dtype("i1")
    return [
        ("norm_w", f32, (s.d_model,)),
        ("in.sign", u32, (s.d_in_proj, s.d_model // 32)),
        ("in.row_scale", f16, (s.d_in_proj,)),
        ("in.A", i8, (r, s.d_model)),
        ("in.a_s", f32, (r,)),
        ("in.B", i8, (s.d_in_proj, r)),
        ("in.b_s", f32, (s.d_in_proj,)),
        ("conv_w", f32, (s.conv_dim, 4)),
        ("conv_b", f32, (s.conv_dim,)),
        ("A_log", f32, (s.nheads,)),
        ("dt_bias", f32, (s.nheads,)),
        ("D", f32, (s.nheads,)),
        ("gnorm_w", f32, (s.d_inner,)),
        ("out.sign", u32, (s.d_model, s.d_inner // 32)),
        ("out.row_scale", f16, (s.d_model,)),
        ("out.A", i8, (r, s.d_inner)),
        ("out.a_s", f32, (r,)),
        ("out.B", i8, (s.d_model, r)),
        ("out.b_s", f32, (s.d_model,)),
    ]


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
                     s.d_state, s.ngroups, s.d_conv, s.vocab, s.lora_rank, float(s.norm_eps), 0, total)
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
    ver, nl, dm, di, hd, ds, ng, dc, vo, r, eps, _z, total = struct.unpack_from("<I9ifIQ", raw, 8)
    assert ver == BLOB_VERSION
    assert total == blob.nbytes, (total, blob.nbytes)
    return Shape(nl, dm, di, hd, ds, ng, dc, vo, r, eps)


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
