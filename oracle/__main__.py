"""Diagnostic of the oracle's arithmetic contract:

    python -m oracle [--config 1] [--steps 64] [--layers N] [--vocab V]

runs the same seeded model three times -- contract mode, contract mode with every binary64 reduction summed in
reversed order, and the "float64 everything" mode -- and prints, for the two variants, the first step whose hidden
state is not bit-identical to the contract mode and the rel-L2 distance at every step after it.  Expected: the
reversed order never departs; float64-everything departs within a few steps and stays at the quantisation-noise floor.
TEST INFRASTRUCTURE: nothing of the product path runs here.
"""
from __future__ import annotations

import argparse
import sys
from pathlib import Path

import numpy as np

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))
import dfssm_synth as ds  # noqa: E402
import oracle  # noqa: E402


def run(blob, toks, mode):
    oracle.set_mode(mode)
    try:
        m = oracle.OracleModel(blob, 1)
        out = []
        for t in range(len(toks)):
            m.step(toks[t:t + 1])
            out.append((m.hidden()[0].copy(), m.logits()[0].copy()))
        m.close()
        return out
    finally:
        oracle.set_mode(oracle.MODE_CONTRACT)


def first_departure(ref, other):
    rels = []
    first = None
    for t, ((h0, _), (h1, _)) in enumerate(zip(ref, other)):
        same = np.array_equal(h0.view(np.uint32), h1.view(np.uint32))
        if not same and first is None:
            first = t
        den = np.linalg.norm(h0.astype(np.float64))
        rels.append(float(np.linalg.norm(h0.astype(np.float64) - h1.astype(np.float64)) / max(den, 1e-300)))
    return first, rels


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--steps", type=int, default=64)
    ap.add_argument("--layers", type=int, default=0, help="override n_layers (0: the config's)")
    ap.add_argument("--vocab", type=int, default=4096, help="cut the vocabulary (0: the config's)")
    a = ap.parse_args()
    s = ds.shape_for_config(a.config)
    kw = {}
    if a.layers:
        kw["n_layers"] = a.layers
    if a.vocab:
        kw["vocab"] = a.vocab
    if kw:
        import dataclasses
        s = dataclasses.replace(s, **kw)
    blob = ds.make_blob(s, a.config)
    toks = ds.token_stream(s.vocab, a.steps, seed=a.config, seq_index=0)
    ref = run(blob, toks, oracle.MODE_CONTRACT)
    for name, mode in (("reversed reduction order", oracle.MODE_REVERSED), ("float64 everything", oracle.MODE_F64)):
        first, rels = first_departure(ref, run(blob, toks, mode))
        if first is None:
            print(f"{name}: bit-identical to the contract mode for all {a.steps} steps")
        else:
            print(f"{name}: first departs at step {first}; rel-L2(hidden) before {max(rels[:first], default=0.0):.2e}, "
                  f"at it {rels[first]:.2e}, max after {max(rels[first:]):.2e}")


if __name__ == "__main__":
    main()
