"""Seeded token streams: ids uniform over the vocabulary (BASELINE.json config 0: "token ids
uniform over the vocab"); sequence i of a batch has its own sub-seeded stream."""
from __future__ import annotations

import numpy as np


def token_stream(vocab: int, n_tokens: int, seed: int, seq_index: int = 0) -> np.ndarray:
    g = np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(seed), 7919, int(seq_index)])))
    return g.integers(0, vocab, size=n_tokens, dtype=np.int32)


def token_batch(vocab: int, n_tokens: int, seed: int, batch: int) -> np.ndarray:
    """[n_tokens][batch] int32 -- row t is the batch of tokens fed at step t."""
    cols = [token_stream(vocab, n_tokens, seed, i) for i in range(batch)]
    return np.ascontiguousarray(np.stack(cols, axis=1))
