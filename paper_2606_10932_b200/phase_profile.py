"""Phase profile of the persistent step kernel (k_mega) from its in-kernel stamps (DFSSM_FLAG_PROF / dfssm_debug_profile).

    python -m paper_2606_10932_b200.phase_profile [--config 2] [--steps 200]

Prints, for the worker CTAs and the service CTAs, the mean SM clocks between consecutive phase stamps of a layer (mean over
CTAs and layers; and the mean over layers of the slowest CTA), and a cross-CTA timeline from the %globaltimer stamps.
A tracing aid: the profiler instantiation of the kernel is slower than the production one (the stamps cost time).
"""
from __future__ import annotations

import argparse
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

WORKER_PHASES = [("wait for the pipeline stage", 0, 1), ("z|x sign rows", 1, 2), ("gather t_in + scale, barrier", 2, 3),
                 ("in_proj epilogue (own rows + all B|C rows, polls their accumulators)", 3, 4), ("state update + gate", 4, 24),
                 ("fence + partial sums + barrier", 24, 26), ("publish G", 26, 27), ("resets + state write-back issue", 27, 5),
                 ("gather G", 5, 6), ("quantise: amax + barrier 1", 6, 17), ("quantise: 127/amax, codes", 17, 18),
                 ("quantise: barrier 2", 18, 7), ("out_proj sign rows", 7, 8), ("gather T, barrier", 8, 9),
                 ("out_proj epilogue + residual + publish U", 9, 10), ("gather U", 10, 11), ("quantise: amax + barrier 1", 11, 21),
                 ("quantise: 127/amax, codes", 21, 22), ("quantise: barrier 2 + ring refill", 22, 12), ("LAYER", 0, 12)]
SERVICE_PHASES = [("wait for the pipeline stage", 0, 1), ("LoRA-down + B|C|dt sign rows, publish A", 1, 2), ("gather G", 2, 6),
                  ("quantise", 6, 7), ("out_proj LoRA-down partial tasks, publish T", 7, 8), ("resets + barrier", 8, 10),
                  ("gather U", 10, 11), ("quantise", 11, 12), ("LAYER", 0, 12)]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--steps", type=int, default=200)
    a = ap.parse_args()
    import torch
    import dfssm_synth as ds
    import paper_2606_10932_b200 as pk
    from paper_2606_10932_b200 import binding, build
    build.build()
    s = ds.shape_for_config(a.config)
    blob = ds.make_blob(s, a.config)
    m = pk.Model(pk.Config.from_shape(s, max_batch=1, flags=binding.FLAG_PROF), blob)
    toks = ds.token_stream(s.vocab, 8, seed=a.config, seq_index=0)
    for t in range(8):
        m.step(torch.from_numpy(toks[t:t + 1].astype(np.int32)).cuda())
    nxt = m.next_tokens()[:1]
    for _ in range(32):
        m.step(nxt)
    m.sync()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(m.stream)
    for _ in range(a.steps):
        m.step(nxt)
    e1.record(m.stream)
    m.sync()
    print(f"config {a.config}, profiler instantiation: {e0.elapsed_time(e1) / a.steps * 1000:.1f} us/step")
    p = m.debug_profile().astype(np.int64)          # [CTAs][layers + 1][stamps]
    G, L1, _ = p.shape
    L = L1 - 1
    lay = slice(2, L)                               # skip the first layers (pipeline fill)
    # workers: the CTAs that stamp phase 4 (service CTAs never do)
    is_worker = p[:, 2, 4] != 0
    W, S = np.flatnonzero(is_worker), np.flatnonzero(~is_worker)
    for name, rows, phases in (("WORKER CTAs", W, WORKER_PHASES), ("SERVICE CTAs", S[1:], SERVICE_PHASES)):
        print(f"{name} ({len(rows)}): clocks, mean over CTAs and layers | mean over layers of the slowest CTA")
        for label, a_, b_ in phases:
            d = p[rows][:, lay, b_] - p[rows][:, lay, a_]
            print(f"  {label:72s} {d.mean():8.0f} {d.max(axis=0).mean():8.0f}")
    lm = p[:, L, 1] - p[:, L, 0]
    print(f"LM head: {lm.mean():.0f} clocks mean, {lm.max()} max")
    # cross-CTA timeline (%globaltimer, ns): slot 28 = gather U of layer l done, 29 = A published (service) / t_in gathered (worker),
    # 30 = worker z|x rows done
    gU, gA, gZ = p[:, :L, 28], p[:, :L, 29], p[:, :L, 30]
    ref = gU[W][:, 2:L - 1].min(axis=0)             # the first worker that has all of U(l-1)
    print("timeline per layer, ns after the first worker holds the whole residual vector (mean over layers):")
    print(f"  last worker holds it          {(gU[W][:, 2:L - 1].max(axis=0) - ref).mean():7.0f}")
    print(f"  last service CTA holds it     {(gU[S][:, 2:L - 1].max(axis=0) - ref).mean():7.0f}")
    print(f"  last service CTA published A  {(gA[S[1:]][:, 3:L].max(axis=0) - ref).mean():7.0f}")
    print(f"  workers done with z|x rows    {(gZ[W][:, 3:L].mean(axis=0) - ref).mean():7.0f} (mean)")
    print(f"  workers hold t_in + scale     {(gA[W][:, 3:L].mean(axis=0) - ref).mean():7.0f} (mean)")
    m.close()


if __name__ == "__main__":
    main()
