"""ctypes binding of include/dfssm.h -- same names, argument marshalling only.

`Model` owns a torch uint8 CUDA tensor (the arena) and a torch stream and hands their raw
pointers to the library; everything else happens inside libdfssm.so.  If the library is not
built, or the device is not a B200-class GPU, this raises: there is no fallback.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from pathlib import Path
from typing import Optional

import numpy as np

_HERE = Path(__file__).resolve().parent

ABI_VERSION = 1
FLAG_TAPS = 1
FLAG_NO_GRAPH = 2
FLAG_NO_MEGA = 4
FLAG_PROF = 8
FLAG_NO_MMA = 16
FLAG_STATE_FP16 = 64
FLAG_SCAFFOLD17 = 128      # 17-level scaffold blob (format word bit 0)
FLAG_LORA_INT4 = 256       # int4 LoRA blob (format word bit 1)

TAPS = dict(XQ_IN=0, S_IN=1, ACC_IN=2, T_IN=3, ZXBCDT=4, XBC_CONV=5, DT=6, Y=7, G=8, GQ=9,
            S_G=10, ACC_OUT=11, T_OUT=12, HIDDEN=13)
_TAP_DTYPES = {0: np.int8, 1: np.float32, 2: np.int32, 3: np.int32, 4: np.float32, 5: np.float32,
               6: np.float32, 7: np.float32, 8: np.float32, 9: np.int8, 10: np.float32, 11: np.int32,
               12: np.int32, 13: np.float32}
KCLASSES = ("embed", "normquant", "proj_in", "ssm", "proj_out", "epi_out", "lmhead", "argmax", "mega")

# every symbol include/dfssm.h declares (tests check the .so exports exactly these)
EXPORTED_SYMBOLS = (
    "dfssm_arena_bytes", "dfssm_create", "dfssm_load_weights", "dfssm_reset_state", "dfssm_step", "dfssm_prefill", "dfssm_sample",
    "dfssm_step_host", "dfssm_logits", "dfssm_next_tokens", "dfssm_hidden", "dfssm_debug_tensor",
    "dfssm_get_state", "dfssm_set_state", "dfssm_debug_profile", "dfssm_sync", "dfssm_launches_per_step",
    "dfssm_time_kernels", "dfssm_last_error", "dfssm_destroy",
    "dfssm_head_noalloc_scratch_need", "dfssm_head_noalloc", "dfssm_head_noalloc_error",
    "dfssm_sched_create", "dfssm_sched_submit", "dfssm_sched_iterate", "dfssm_sched_run", "dfssm_sched_result", "dfssm_sched_stats",
    "dfssm_sched_last_error", "dfssm_sched_destroy", "dfssm_sched_set_sampling", "dfssm_sched_uniform",
)

_ERR = {0: "OK", -1: "E_ARG", -2: "E_SIZE", -3: "E_STATE", -4: "E_CUDA", -5: "E_ARCH", -6: "E_TOKEN"}


class DfssmError(RuntimeError):
    def __init__(self, code: int, text: str = ""):
        self.code = code
        super().__init__(f"dfssm: {_ERR.get(code, code)} {text}".strip())


class _CConfig(C.Structure):
    _fields_ = [("abi_version", C.c_uint32), ("n_layers", C.c_int32), ("d_model", C.c_int32),
                ("d_inner", C.c_int32), ("headdim", C.c_int32), ("d_state", C.c_int32),
                ("ngroups", C.c_int32), ("d_conv", C.c_int32), ("vocab", C.c_int32),
                ("lora_rank", C.c_int32), ("max_batch", C.c_int32), ("norm_eps", C.c_float),
                ("flags", C.c_uint32)]


@dataclass(frozen=True)
class Config:
    n_layers: int
    d_model: int
    d_inner: int
    headdim: int
    d_state: int
    ngroups: int
    d_conv: int
    vocab: int
    lora_rank: int
    max_batch: int = 1
    norm_eps: float = 1e-5
    flags: int = 0

    @classmethod
    def from_shape(cls, s, max_batch: int = 1, flags: int = 0) -> "Config":
        """`s` is anything with the shape attributes (e.g. dfssm_synth.Shape); its weight format (`fmt`, if it has one) sets
        FLAG_SCAFFOLD17 / FLAG_LORA_INT4."""
        fmt = int(getattr(s, "fmt", 0))
        flags |= (FLAG_SCAFFOLD17 if fmt & 1 else 0) | (FLAG_LORA_INT4 if fmt & 2 else 0)
        return cls(s.n_layers, s.d_model, s.d_inner, s.headdim, s.d_state, s.ngroups, s.d_conv, s.vocab,
                   s.lora_rank, max_batch, float(s.norm_eps), flags)

    def c(self) -> _CConfig:
        return _CConfig(ABI_VERSION, self.n_layers, self.d_model, self.d_inner, self.headdim, self.d_state,
                        self.ngroups, self.d_conv, self.vocab, self.lora_rank, self.max_batch, self.norm_eps,
                        self.flags)

    @property
    def nheads(self) -> int:
        return self.d_inner // self.headdim

    @property
    def d_in_proj(self) -> int:
        return 2 * self.d_inner + 2 * self.ngroups * self.d_state + self.nheads

    @property
    def conv_dim(self) -> int:
        return self.d_inner + 2 * self.ngroups * self.d_state


def lib_path() -> Path:
    return _HERE / "libdfssm.so"


_lib = None


def lib() -> C.CDLL:
    """Load libdfssm.so (never builds it: see paper_2606_10932_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    p = lib_path()
    if not p.exists():
        raise DfssmError(-3, f"{p} is missing: run `python -m paper_2606_10932_b200.build` "
                             "(there is no CPU fallback)")
    L = C.CDLL(str(p))
    vp, i32p, f32p = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_float)
    cfgp = C.POINTER(_CConfig)
    sig = {
        "dfssm_arena_bytes": (C.c_size_t, [cfgp]),
        "dfssm_create": (C.c_int, [cfgp, vp, C.c_size_t, vp, C.POINTER(vp)]),
        "dfssm_load_weights": (C.c_int, [vp, vp, C.c_size_t]),
        "dfssm_reset_state": (C.c_int, [vp, C.c_int]),
        "dfssm_step": (C.c_int, [vp, vp, C.c_int]),
        "dfssm_prefill": (C.c_int, [vp, vp, C.c_int, C.c_int]),
        "dfssm_sample": (C.c_int, [vp, C.c_int, C.c_float, C.c_int, vp]),
        "dfssm_step_host": (C.c_int, [vp, i32p, C.c_int, i32p, f32p]),
        "dfssm_logits": (C.c_int, [vp, C.POINTER(vp)]),
        "dfssm_next_tokens": (C.c_int, [vp, C.POINTER(vp)]),
        "dfssm_hidden": (C.c_int, [vp, C.POINTER(vp)]),
        "dfssm_debug_tensor": (C.c_int, [vp, C.c_int, C.c_int, C.c_int, C.POINTER(vp), C.POINTER(C.c_size_t)]),
        "dfssm_get_state": (C.c_int, [vp, C.c_int, C.c_int, f32p, C.c_size_t, f32p, C.c_size_t]),
        "dfssm_set_state": (C.c_int, [vp, C.c_int, C.c_int, f32p, C.c_size_t, f32p, C.c_size_t]),
        "dfssm_debug_profile": (C.c_int, [vp, C.POINTER(C.c_uint64), C.c_size_t, i32p]),
        "dfssm_sync": (C.c_int, [vp]),
        "dfssm_launches_per_step": (C.c_int, [vp, C.c_int]),
        "dfssm_time_kernels": (C.c_int, [vp, vp, C.c_int, C.c_int, f32p]),
        "dfssm_last_error": (C.c_char_p, [vp]),
        "dfssm_destroy": (None, [vp]),
        "dfssm_head_noalloc_scratch_need": (C.c_size_t, [C.c_int, C.c_int, C.c_int]),
        "dfssm_head_noalloc": (C.c_int, [vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, C.c_float, vp, vp, vp]),
        "dfssm_head_noalloc_error": (C.c_char_p, []),
        "dfssm_sched_create": (C.c_int, [vp, C.c_int, vp, C.c_size_t, vp, C.POINTER(vp)]),
        "dfssm_sched_submit": (C.c_int, [vp, i32p, C.c_int, C.c_int, i32p]),
        "dfssm_sched_iterate": (C.c_int, [vp, i32p]),
        "dfssm_sched_run": (C.c_int, [vp]),
        "dfssm_sched_result": (C.c_int, [vp, C.c_int, i32p, C.c_int, i32p, i32p]),
        "dfssm_sched_stats": (C.c_int, [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]),
        "dfssm_sched_last_error": (C.c_char_p, [vp]),
        "dfssm_sched_destroy": (None, [vp]),
        "dfssm_sched_set_sampling": (C.c_int, [vp, C.c_float, C.c_int, C.c_ulonglong]),
        "dfssm_sched_uniform": (C.c_float, [C.c_ulonglong, C.c_int]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def dfssm_arena_bytes(cfg: Config) -> int:
    c = cfg.c()
    return int(lib().dfssm_arena_bytes(C.byref(c)))


NOALLOC_SCRATCH_BYTES = 4 << 20


def head_noalloc_scratch_need(batch: int, d_model: int, vocab: int) -> int:
    return int(lib().dfssm_head_noalloc_scratch_need(int(batch), int(d_model), int(vocab)))


def head_noalloc(hidden, normf_w, emb, emb_scale, next_out, logits_out=None, eps: float = 1e-5, stream=None):
    """dfssm_head_noalloc: S8 (final norm + quantiser, tied int8 LM head, greedy argmax) with the intermediates in the
    library's static device array: no allocation, no context, no arena.  All arguments are torch CUDA tensors of the caller
    (hidden float32 [batch][d_model], normf_w float32 [d_model], emb int8 [vocab][d_model], emb_scale float32 [vocab],
    next_out int32 [batch], logits_out float32 [batch][vocab] or None); enqueued on `stream` (default: torch's current one)."""
    import torch
    batch, d_model = hidden.shape
    vocab = emb.shape[0]
    for t_, dt in ((hidden, torch.float32), (normf_w, torch.float32), (emb, torch.int8), (emb_scale, torch.float32),
                   (next_out, torch.int32)) + (((logits_out, torch.float32),) if logits_out is not None else ()):
        if not (t_.is_cuda and t_.is_contiguous() and t_.dtype == dt):
            raise DfssmError(-1, "head_noalloc: contiguous CUDA tensors of the documented dtypes are required")
    if emb.shape[1] != d_model or normf_w.numel() != d_model or emb_scale.numel() != vocab or next_out.numel() < batch or \
            (logits_out is not None and logits_out.numel() < batch * vocab):
        raise DfssmError(-1, "head_noalloc: shapes do not match")
    st = stream if stream is not None else torch.cuda.current_stream(hidden.device)
    L = lib()
    with torch.cuda.device(hidden.device):
        rc = L.dfssm_head_noalloc(hidden.data_ptr(), normf_w.data_ptr(), emb.data_ptr(), emb_scale.data_ptr(), int(batch), int(d_model),
                                  int(vocab), float(eps), next_out.data_ptr(), logits_out.data_ptr() if logits_out is not None else None,
                                  st.cuda_stream)
    if rc != 0:
        raise DfssmError(rc, L.dfssm_head_noalloc_error().decode())


def _f32p(a: Optional[np.ndarray]):
    return a.ctypes.data_as(C.POINTER(C.c_float)) if a is not None else None


class Model:
    """One dfssm_ctx plus the torch-owned arena and stream behind it."""

    def __init__(self, cfg: Config, blob: Optional[np.ndarray] = None, device: str = "cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise DfssmError(-5, "no CUDA device: the DF-SSM step runs only on the GPU (no CPU fallback)")
        self._L = lib()
        self._torch = torch
        self.cfg = cfg
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        nbytes = dfssm_arena_bytes(cfg)
        if nbytes == 0:
            raise DfssmError(-1, "invalid config")
        self.arena = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        assert self.arena.data_ptr() % 256 == 0
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        self._h = C.c_void_p()
        c = cfg.c()
        rc = self._L.dfssm_create(C.byref(c), C.c_void_p(self.arena.data_ptr()), nbytes,
                                  C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        self._check(rc)
        self.batch = 0
        if blob is not None:
            self.load_weights(blob)

    # ---- plumbing ----
    def _check(self, rc: int):
        if rc != 0:
            text = ""
            if self._h:
                text = (self._L.dfssm_last_error(self._h) or b"").decode(errors="replace")
            raise DfssmError(rc, text)

    def close(self):
        if getattr(self, "_h", None):
            self._L.dfssm_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _view(self, ptr: int, nbytes: int):
        """torch uint8 view of `nbytes` of the arena starting at device address `ptr`."""
        off = ptr - self.arena.data_ptr()
        assert 0 <= off and off + nbytes <= self.arena.numel()
        return self.arena[off:off + nbytes]

    # ---- the C ABI, one method per call ----
    def load_weights(self, blob: np.ndarray):
        blob = np.ascontiguousarray(blob, dtype=np.uint8)
        self._check(self._L.dfssm_load_weights(self._h, C.c_void_p(blob.ctypes.data), blob.nbytes))

    def reset_state(self, seq: int = -1):
        self._check(self._L.dfssm_reset_state(self._h, int(seq)))

    def step(self, tokens_dev, batch: Optional[int] = None):
        """tokens_dev: torch int32 CUDA tensor [batch] (or a raw device pointer with `batch`)."""
        if isinstance(tokens_dev, int):
            ptr, n = tokens_dev, int(batch)
        else:
            assert tokens_dev.dtype == self._torch.int32 and tokens_dev.is_cuda and tokens_dev.is_contiguous()
            ptr, n = tokens_dev.data_ptr(), (int(batch) if batch is not None else tokens_dev.numel())
            a0 = self.arena.data_ptr()
            if not (a0 <= ptr < a0 + self.arena.numel()):
                # a caller tensor made on torch's current stream: the library copies it on ITS stream, so order that stream
                # behind the producer and keep the block from being reused before the copy has run
                self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
                tokens_dev.record_stream(self.stream)
        self._check(self._L.dfssm_step(self._h, C.c_void_p(ptr), n))
        self.batch = n

    def prefill(self, tokens_dev, seq: int = 0):
        """tokens_dev: torch int32 CUDA tensor [n_tokens] of sequence `seq` (dfssm_prefill)."""
        assert tokens_dev.dtype == self._torch.int32 and tokens_dev.is_cuda and tokens_dev.is_contiguous()
        self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
        tokens_dev.record_stream(self.stream)
        self._check(self._L.dfssm_prefill(self._h, C.c_void_p(tokens_dev.data_ptr()), tokens_dev.numel(), int(seq)))
        self.batch = max(self.batch, int(seq) + 1)

    def sample(self, temperature: float, top_k: int, uniform_dev, batch: Optional[int] = None):
        """uniform_dev: torch float32 CUDA tensor [batch] in [0, 1) (dfssm_sample); the result replaces next_tokens()."""
        assert uniform_dev.dtype == self._torch.float32 and uniform_dev.is_cuda and uniform_dev.is_contiguous()
        n = int(batch) if batch is not None else uniform_dev.numel()
        self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
        uniform_dev.record_stream(self.stream)
        self._check(self._L.dfssm_sample(self._h, n, float(temperature), int(top_k), C.c_void_p(uniform_dev.data_ptr())))

    def step_host(self, tokens_host: np.ndarray, next_host: np.ndarray, logits_host: Optional[np.ndarray] = None):
        assert tokens_host.dtype == np.int32 and next_host.dtype == np.int32
        n = tokens_host.size
        assert next_host.size >= n
        if logits_host is not None:
            assert logits_host.dtype == np.float32 and logits_host.size >= n * self.cfg.vocab
        self._check(self._L.dfssm_step_host(self._h, tokens_host.ctypes.data_as(C.POINTER(C.c_int32)), n,
                                            next_host.ctypes.data_as(C.POINTER(C.c_int32)), _f32p(logits_host)))
        self.batch = n

    def next_tokens_ptr(self) -> int:
        p = C.c_void_p()
        self._check(self._L.dfssm_next_tokens(self._h, C.byref(p)))
        return int(p.value)

    def next_tokens(self):
        """Borrowed torch int32 view [max_batch] of the greedy tokens (device)."""
        return self._view(self.next_tokens_ptr(), 4 * self.cfg.max_batch).view(self._torch.int32)

    def logits(self):
        p = C.c_void_p()
        self._check(self._L.dfssm_logits(self._h, C.byref(p)))
        return self._view(int(p.value), 4 * self.cfg.max_batch * self.cfg.vocab).view(self._torch.float32).view(
            self.cfg.max_batch, self.cfg.vocab)

    def hidden(self):
        p = C.c_void_p()
        self._check(self._L.dfssm_hidden(self._h, C.byref(p)))
        return self._view(int(p.value), 4 * self.cfg.max_batch * self.cfg.d_model).view(self._torch.float32).view(
            self.cfg.max_batch, self.cfg.d_model)

    def debug_tensor(self, layer: int, which, seq: int = 0) -> np.ndarray:
        which = TAPS[which] if isinstance(which, str) else int(which)
        p, n = C.c_void_p(), C.c_size_t()
        self._check(self._L.dfssm_debug_tensor(self._h, int(layer), which, int(seq), C.byref(p), C.byref(n)))
        self.sync()
        raw = self._view(int(p.value), int(n.value)).cpu().numpy()
        return raw.view(_TAP_DTYPES[which]).copy()

    def get_state(self, layer: int, seq: int = 0):
        c = self.cfg
        ssm = np.empty((c.nheads, c.headdim, c.d_state), np.float32)
        conv = np.empty((c.conv_dim, 3), np.float32)
        self._check(self._L.dfssm_get_state(self._h, int(layer), int(seq), _f32p(ssm), ssm.nbytes, _f32p(conv), conv.nbytes))
        return ssm, conv

    def set_state(self, layer: int, seq: int, ssm: Optional[np.ndarray], conv: Optional[np.ndarray]):
        ssm = np.ascontiguousarray(ssm, np.float32) if ssm is not None else None
        conv = np.ascontiguousarray(conv, np.float32) if conv is not None else None
        self._check(self._L.dfssm_set_state(self._h, int(layer), int(seq), _f32p(ssm), ssm.nbytes if ssm is not None else 0,
                                            _f32p(conv), conv.nbytes if conv is not None else 0))

    def debug_profile(self) -> np.ndarray:
        """uint64 [CTAs][layers + 1][stamps] phase stamps of the last persistent-kernel step (FLAG_PROF)."""
        dims = (C.c_int32 * 3)()
        self._check(self._L.dfssm_debug_profile(self._h, None, 0, dims))
        out = np.zeros(tuple(int(d) for d in dims), np.uint64)
        self._check(self._L.dfssm_debug_profile(self._h, out.ctypes.data_as(C.POINTER(C.c_uint64)), out.nbytes, dims))
        return out

    def sync(self):
        self._check(self._L.dfssm_sync(self._h))

    def launches_per_step(self, batch: int = 1) -> int:
        return int(self._L.dfssm_launches_per_step(self._h, int(batch)))

    def time_kernels(self, tokens_dev, iters: int = 4) -> dict:
        out = np.zeros(len(KCLASSES), np.float32)
        self._check(self._L.dfssm_time_kernels(self._h, C.c_void_p(tokens_dev.data_ptr()), tokens_dev.numel(), int(iters),
                                               _f32p(out)))
        return dict(zip(KCLASSES, (float(x) for x in out)))


class Scheduler:
    """dfssm_sched_*: continuous-batching greedy generation over one Model (argument marshalling only)."""

    def __init__(self, model: "Model", max_batch: Optional[int] = None, max_prompt: int = 4096):
        import torch
        self._m, self._L = model, model._L
        nb = int(max_batch or model.cfg.max_batch)
        self._scratch = torch.empty(max_prompt + nb, dtype=torch.int32, device=model.device)       # one prompt + nb uniforms
        h = C.c_void_p()
        rc = self._L.dfssm_sched_create(model._h, nb, self._scratch.data_ptr(), 4 * (max_prompt + nb),
                                        model.stream.cuda_stream, C.byref(h))
        self._h = h
        self._check(rc)

    def _check(self, rc: int):
        if rc != 0:
            raise DfssmError(rc, self._L.dfssm_sched_last_error(self._h).decode() if self._h else "")

    def submit(self, prompt, max_new_tokens: int) -> int:
        p = np.ascontiguousarray(prompt, np.int32)
        rid = C.c_int32()
        self._check(self._L.dfssm_sched_submit(self._h, p.ctypes.data_as(C.POINTER(C.c_int32)), p.size, int(max_new_tokens), C.byref(rid)))
        return int(rid.value)

    def set_sampling(self, temperature: float, top_k: int, seed: int = 0):
        self._check(self._L.dfssm_sched_set_sampling(self._h, float(temperature), int(top_k), int(seed)))

    def iterate(self) -> int:
        n = C.c_int32()
        self._check(self._L.dfssm_sched_iterate(self._h, C.byref(n)))
        return int(n.value)

    def run(self):
        self._check(self._L.dfssm_sched_run(self._h))

    def result(self, rid: int):
        n, done = C.c_int32(), C.c_int32()
        self._check(self._L.dfssm_sched_result(self._h, int(rid), None, 0, C.byref(n), C.byref(done)))
        out = np.empty(int(n.value), np.int32)
        self._check(self._L.dfssm_sched_result(self._h, int(rid), out.ctypes.data_as(C.POINTER(C.c_int32)), out.size, C.byref(n), C.byref(done)))
        return out, bool(done.value)

    def stats(self) -> dict:
        a, b, c = C.c_longlong(), C.c_longlong(), C.c_longlong()
        self._check(self._L.dfssm_sched_stats(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return dict(steps=int(a.value), slot_steps_used=int(b.value), slot_steps_run=int(c.value))

    def close(self):
        if getattr(self, "_h", None):
            self._L.dfssm_sched_destroy(self._h)
            self._h = None

    __del__ = close
