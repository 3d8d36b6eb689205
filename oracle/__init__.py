"""ctypes driver for the CPU oracle (oracle/dfssm_oracle.c).

TEST INFRASTRUCTURE ONLY.  Importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs -- never from paper_2606_10932_b200/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libdfssm_oracle.so"
_SRC = _HERE / "dfssm_oracle.c"
_HDR = _HERE / "dfssm_oracle.h"

# the arithmetic contract needs: no contraction, no fast-math.  -O2, no -march: plain code.
CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fno-math-errno",
          "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra"]

TAPS = dict(XQ_IN=0, S_IN=1, ACC_IN=2, T_IN=3, ZXBCDT=4, XBC_CONV=5, DT=6, Y=7, G=8, GQ=9,
            S_G=10, ACC_OUT=11, T_OUT=12, HIDDEN=13)


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc if the .so is missing or older than its sources."""
    if not force and _SO.exists() and _SO.stat().st_mtime >= max(_SRC.stat().st_mtime, _HDR.stat().st_mtime):
        return _SO
    tmp = _SO.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.run(["gcc", *CFLAGS, str(_SRC), "-o", str(tmp), "-lm"], check=True)
    os.replace(tmp, _SO)
    return _SO


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(str(build()))
    f32p, i8p, i32p, u32p, u16p = (C.POINTER(C.c_float), C.POINTER(C.c_int8), C.POINTER(C.c_int32),
                                   C.POINTER(C.c_uint32), C.POINTER(C.c_uint16))
    sig = {
        "dfo_sp_expf": (C.c_float, [C.c_float]),
        "dfo_sp_log1pf": (C.c_float, [C.c_float]),
        "dfo_sp_softplusf": (C.c_float, [C.c_float]),
        "dfo_siluf": (C.c_float, [C.c_float]),
        "dfo_half_to_float": (C.c_float, [C.c_uint16]),
        "dfo_embed": (None, [i8p, C.c_float, C.c_int, f32p]),
        "dfo_norm_quant": (None, [f32p, f32p, C.c_int, C.c_float, i8p, f32p, f32p, f32p]),
        "dfo_sign_matvec": (None, [u32p, C.c_int, C.c_int, i8p, i32p]),
        "dfo_lora_down": (None, [i8p, C.c_int, C.c_int, i8p, i32p]),
        "dfo_level_matvec": (None, [u32p, C.c_int, C.c_int, i8p, i32p]),
        "dfo_unpack_int4": (None, [C.POINTER(C.c_uint8), C.c_int, C.c_int, i8p]),
        "dfo_proj_epilogue": (None, [i32p, i32p, u16p, f32p, i8p, f32p, C.c_int, C.c_int, C.c_float, f32p]),
        "dfo_conv_step": (None, [f32p, f32p, f32p, f32p, C.c_int, f32p]),
        "dfo_ssm_step": (None, [f32p, f32p, f32p, f32p, f32p, f32p, f32p, C.c_int, C.c_int, C.c_int, C.c_int, f32p]),
        "dfo_gate": (None, [f32p, f32p, C.c_int, f32p]),
        "dfo_lm_head": (None, [i8p, f32p, C.c_int, C.c_int, i8p, C.c_float, i32p, f32p]),
        "dfo_argmax": (C.c_int, [f32p, C.c_int]),
        "dfo_float_to_half": (C.c_uint16, [C.c_float]),
        "dfo_set_state_fp16": (None, [C.c_void_p, C.c_int]),
        "dfo_sample": (C.c_int, [f32p, C.c_int, C.c_float, C.c_int, C.c_float]),
        "dfo_load": (C.c_void_p, [C.c_void_p, C.c_size_t, C.c_int, C.c_char_p, C.c_size_t]),
        "dfo_free": (None, [C.c_void_p]),
        "dfo_set_threads": (None, [C.c_int]),
        "dfo_get_threads": (C.c_int, []),
        "dfo_set_mode": (None, [C.c_int]),
        "dfo_get_mode": (C.c_int, []),
        "dfo_enable_taps": (None, [C.c_void_p, C.c_int]),
        "dfo_reset": (None, [C.c_void_p, C.c_int]),
        "dfo_step": (C.c_int, [C.c_void_p, i32p, C.c_int]),
        "dfo_logits": (f32p, [C.c_void_p]),
        "dfo_next_tokens": (i32p, [C.c_void_p]),
        "dfo_hidden": (f32p, [C.c_void_p]),
        "dfo_tap": (C.c_void_p, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_size_t)]),
        "dfo_ssm_state": (f32p, [C.c_void_p, C.c_int, C.c_int]),
        "dfo_conv_state": (f32p, [C.c_void_p, C.c_int, C.c_int]),
        "dfo_shape": (C.c_int, [C.c_void_p, i32p]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def _p(a: np.ndarray, ctype):
    return a.ctypes.data_as(C.POINTER(ctype))


def _c(a, dtype) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


# ------------------------- function-level wrappers (numpy in, numpy out) -------------------------
def sp_expf(x):
    L = lib()
    return np.array([L.dfo_sp_expf(float(v)) for v in np.asarray(x, np.float32).ravel()], np.float32).reshape(np.shape(x))


def sp_log1pf(x):
    L = lib()
    return np.array([L.dfo_sp_log1pf(float(v)) for v in np.asarray(x, np.float32).ravel()], np.float32).reshape(np.shape(x))


def sp_softplusf(x):
    L = lib()
    return np.array([L.dfo_sp_softplusf(float(v)) for v in np.asarray(x, np.float32).ravel()], np.float32).reshape(np.shape(x))


def siluf(x):
    L = lib()
    return np.array([L.dfo_siluf(float(v)) for v in np.asarray(x, np.float32).ravel()], np.float32).reshape(np.shape(x))


def half_to_float(h):
    L = lib()
    return np.array([L.dfo_half_to_float(int(v)) for v in np.asarray(h, np.uint16).ravel()], np.float32).reshape(np.shape(h))


def embed(E_row, e_s):
    E_row = _c(E_row, np.int8)
    u = np.empty(E_row.size, np.float32)
    lib().dfo_embed(_p(E_row, C.c_int8), float(e_s), E_row.size, _p(u, C.c_float))
    return u


def norm_quant(v, w, eps=1e-5):
    v, w = _c(v, np.float32), _c(w, np.float32)
    q = np.empty(v.size, np.int8)
    s, rstd, amax = C.c_float(), C.c_float(), C.c_float()
    lib().dfo_norm_quant(_p(v, C.c_float), _p(w, C.c_float), v.size, float(eps), _p(q, C.c_int8),
                         C.byref(s), C.byref(rstd), C.byref(amax))
    return q, np.float32(s.value), np.float32(rstd.value), np.float32(amax.value)


def sign_matvec(sign, xq):
    sign, xq = _c(sign, np.uint32), _c(xq, np.int8)
    rows, W = sign.shape
    assert xq.size == 32 * W
    acc = np.empty(rows, np.int32)
    lib().dfo_sign_matvec(_p(sign, C.c_uint32), rows, 32 * W, _p(xq, C.c_int8), _p(acc, C.c_int32))
    return acc


def level_matvec(lvl, xq):
    """17-level scaffold (five bit planes [rows][K/32][5]): acc_i = sum_k level_ik * q_k (R25)"""
    lvl, xq = _c(lvl, np.uint32), _c(xq, np.int8)
    rows, W, five = lvl.shape
    assert five == 5 and xq.size == 32 * W
    acc = np.empty(rows, np.int32)
    lib().dfo_level_matvec(_p(lvl, C.c_uint32), rows, 32 * W, _p(xq, C.c_int8), _p(acc, C.c_int32))
    return acc


def unpack_int4(packed):
    packed = _c(packed, np.uint8)
    rows, half = packed.shape
    out = np.empty((rows, 2 * half), np.int8)
    lib().dfo_unpack_int4(_p(packed, C.c_uint8), rows, 2 * half, _p(out, C.c_int8))
    return out


def lora_down(A, xq):
    A, xq = _c(A, np.int8), _c(xq, np.int8)
    r, K = A.shape
    t = np.empty(r, np.int32)
    lib().dfo_lora_down(_p(A, C.c_int8), r, K, _p(xq, C.c_int8), _p(t, C.c_int32))
    return t


def proj_epilogue(acc, t, row_scale_f16, a_s, B, b_s, s_x):
    acc, t = _c(acc, np.int32), _c(t, np.int32)
    rs = _c(row_scale_f16, np.float16).view(np.uint16)
    a_s, B, b_s = _c(a_s, np.float32), _c(B, np.int8), _c(b_s, np.float32)
    rows, r = B.shape
    out = np.empty(rows, np.float32)
    lib().dfo_proj_epilogue(_p(acc, C.c_int32), _p(t, C.c_int32), _p(rs, C.c_uint16), _p(a_s, C.c_float),
                            _p(B, C.c_int8), _p(b_s, C.c_float), rows, r, float(s_x), _p(out, C.c_float))
    return out


def conv_step(state, w, bias, xin):
    """state [C][3] is updated in place (must be a contiguous float32 array)."""
    assert state.dtype == np.float32 and state.flags.c_contiguous
    w, bias, xin = _c(w, np.float32), _c(bias, np.float32), _c(xin, np.float32)
    Cn = xin.size
    out = np.empty(Cn, np.float32)
    lib().dfo_conv_step(_p(state, C.c_float), _p(w, C.c_float), _p(bias, C.c_float), _p(xin, C.c_float), Cn,
                        _p(out, C.c_float))
    return out


def ssm_step(H, x, Bv, Cv, dt, A, D, ngroups=1):
    """H [nheads][headdim][d_state] is updated in place; dt is post-softplus, A negative."""
    assert H.dtype == np.float32 and H.flags.c_contiguous
    nheads, headdim, d_state = H.shape
    x, Bv, Cv = _c(x, np.float32), _c(Bv, np.float32), _c(Cv, np.float32)
    dt, A, D = _c(dt, np.float32), _c(A, np.float32), _c(D, np.float32)
    y = np.empty(nheads * headdim, np.float32)
    lib().dfo_ssm_step(_p(H, C.c_float), _p(x, C.c_float), _p(Bv, C.c_float), _p(Cv, C.c_float),
                       _p(dt, C.c_float), _p(A, C.c_float), _p(D, C.c_float), nheads, headdim, d_state,
                       ngroups, _p(y, C.c_float))
    return y


def gate(y, z):
    y, z = _c(y, np.float32), _c(z, np.float32)
    g = np.empty(y.size, np.float32)
    lib().dfo_gate(_p(y, C.c_float), _p(z, C.c_float), y.size, _p(g, C.c_float))
    return g


def lm_head(E, e_s, hq, s_h):
    E, e_s, hq = _c(E, np.int8), _c(e_s, np.float32), _c(hq, np.int8)
    vocab, d = E.shape
    acc = np.empty(vocab, np.int32)
    logits = np.empty(vocab, np.float32)
    lib().dfo_lm_head(_p(E, C.c_int8), _p(e_s, C.c_float), vocab, d, _p(hq, C.c_int8), float(s_h),
                      _p(acc, C.c_int32), _p(logits, C.c_float))
    return acc, logits


def argmax(logits):
    logits = _c(logits, np.float32)
    return int(lib().dfo_argmax(_p(logits, C.c_float), logits.size))


def float_to_half(x) -> np.ndarray:
    """binary32 -> binary16 bit patterns (RN-even), element by element through dfo_float_to_half"""
    a = np.atleast_1d(np.asarray(x, np.float32))
    L = lib()
    return np.array([L.dfo_float_to_half(float(v)) for v in a.ravel()], np.uint16).reshape(a.shape)


def sample(logits, temperature: float, top_k: int, u: float) -> int:
    lg = _c(logits, np.float32)
    return int(lib().dfo_sample(_p(lg, C.c_float), lg.size, float(temperature), int(top_k), float(u)))


def set_threads(n: int) -> int:
    lib().dfo_set_threads(int(n))
    return int(lib().dfo_get_threads())


# TEST-ONLY arithmetic modes of the oracle (dfssm_oracle.c): the default is the contract of DESIGN.md section 5
MODE_CONTRACT, MODE_REVERSED, MODE_F64 = 0, 1, 2


def set_mode(mode: int) -> None:
    """MODE_REVERSED: every binary64 reduction summed in reversed order (must not change a bit);
    MODE_F64: the "float64 everything" diagnostic (departs from the contract within a few steps)."""
    lib().dfo_set_mode(int(mode))


def get_mode() -> int:
    return int(lib().dfo_get_mode())


def get_threads() -> int:
    return int(lib().dfo_get_threads())


# ------------------------------------ whole-model wrapper ------------------------------------
class OracleModel:
    _TAP_DTYPES = {0: np.int8, 1: np.float32, 2: np.int32, 3: np.int32, 4: np.float32, 5: np.float32,
                   6: np.float32, 7: np.float32, 8: np.float32, 9: np.int8, 10: np.float32, 11: np.int32,
                   12: np.int32, 13: np.float32}

    def __init__(self, blob: np.ndarray, max_batch: int = 1, taps: bool = False):
        self._L = lib()
        blob = np.ascontiguousarray(blob, dtype=np.uint8)
        err = C.create_string_buffer(256)
        self._h = self._L.dfo_load(blob.ctypes.data, blob.nbytes, int(max_batch), err, 256)
        if not self._h:
            raise ValueError("oracle: " + err.value.decode())
        shp = (C.c_int32 * 12)()
        self._L.dfo_shape(self._h, shp)
        (self.n_layers, self.d_model, self.d_inner, self.headdim, self.d_state, self.ngroups, self.d_conv,
         self.vocab, self.lora_rank, self.nheads, self.d_in_proj, self.conv_dim) = [int(v) for v in shp]
        self.max_batch = int(max_batch)
        self.batch = 0
        if taps:
            self._L.dfo_enable_taps(self._h, 1)
        self._tap_len = {0: self.d_model, 1: 1, 2: self.d_in_proj, 3: self.lora_rank, 4: self.d_in_proj,
                         5: self.conv_dim, 6: self.nheads, 7: self.d_inner, 8: self.d_inner, 9: self.d_inner,
                         10: 1, 11: self.d_model, 12: self.lora_rank, 13: self.d_model}

    def set_state_fp16(self, on: bool = True):
        """DESIGN.md R24: store the SSM state as binary16 between steps (rounded after every step)."""
        self._L.dfo_set_state_fp16(self._h, 1 if on else 0)

    def close(self):
        if getattr(self, "_h", None):
            self._L.dfo_free(self._h)
            self._h = None

    __del__ = close

    def reset(self, seq: int = -1):
        self._L.dfo_reset(self._h, int(seq))

    def step(self, tokens):
        tokens = np.ascontiguousarray(tokens, dtype=np.int32).ravel()
        rc = self._L.dfo_step(self._h, _p(tokens, C.c_int32), tokens.size)
        if rc != 0:
            raise ValueError(f"oracle step failed: {rc}")
        self.batch = tokens.size

    def logits(self) -> np.ndarray:
        p = self._L.dfo_logits(self._h)
        return np.ctypeslib.as_array(p, shape=(self.max_batch, self.vocab))[: self.batch].copy()

    def next_tokens(self) -> np.ndarray:
        p = self._L.dfo_next_tokens(self._h)
        return np.ctypeslib.as_array(p, shape=(self.max_batch,))[: self.batch].copy()

    def hidden(self) -> np.ndarray:
        p = self._L.dfo_hidden(self._h)
        return np.ctypeslib.as_array(p, shape=(self.max_batch, self.d_model))[: self.batch].copy()

    def tap(self, layer: int, which, seq: int = 0) -> np.ndarray:
        which = TAPS[which] if isinstance(which, str) else int(which)
        n = C.c_size_t()
        ptr = self._L.dfo_tap(self._h, int(layer), which, int(seq), C.byref(n))
        if not ptr:
            raise ValueError("taps not enabled or bad index")
        dt = np.dtype(self._TAP_DTYPES[which])
        cnt = self._tap_len[which]
        buf = (C.c_uint8 * (cnt * dt.itemsize)).from_address(ptr)
        return np.frombuffer(buf, dtype=dt, count=cnt).copy()

    def ssm_state(self, layer: int, seq: int = 0) -> np.ndarray:
        """Live view (writes go through) of [nheads][headdim][d_state]."""
        p = self._L.dfo_ssm_state(self._h, int(layer), int(seq))
        return np.ctypeslib.as_array(p, shape=(self.nheads, self.headdim, self.d_state))

    def conv_state(self, layer: int, seq: int = 0) -> np.ndarray:
        p = self._L.dfo_conv_state(self._h, int(layer), int(seq))
        return np.ctypeslib.as_array(p, shape=(self.conv_dim, 3))
