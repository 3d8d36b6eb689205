"""Seeded synthetic inputs for DF-SSM (arxiv/paper_2606_10932): shapes, weight blobs, token streams.

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_10932_b200/``).  It holds none of the method's arithmetic: it only
knows tensor shapes, the canonical weight-blob byte layout, and the
random distributions BASELINE.json's configs prescribe.  The blob bytes -- not the
RNG -- are the contract shared by the two sides.
"""
from .shapes import Shape, CONFIGS, shape_for_config, tiny_shape, FMT_SCAFFOLD17, FMT_LORA_INT4
from .blob import (BLOB_MAGIC, BLOB_VERSION, HEADER_BYTES, TENSOR_ALIGN,
                   layer_tensor_specs, global_tensor_specs, blob_layout, blob_nbytes,
                   write_blob, blob_views, pack_levels, unpack_levels, pack_int4, unpack_int4)
from .weights import make_blob
from .tokens import token_stream, token_batch

__all__ = [
    "Shape", "CONFIGS", "shape_for_config", "tiny_shape",
    "BLOB_MAGIC", "BLOB_VERSION", "HEADER_BYTES", "TENSOR_ALIGN",
    "layer_tensor_specs", "global_tensor_specs", "blob_layout", "blob_nbytes",
    "write_blob", "blob_views", "make_blob", "token_stream", "token_batch",
    "FMT_SCAFFOLD17", "FMT_LORA_INT4", "pack_levels", "unpack_levels", "pack_int4", "unpack_int4",
]
