"""Thin ctypes mirror of include/metronome.h (+ the aids of include/metronome_measure.h) -- argument marshalling only.

Every step of the path runs in libmetronome.so's CUDA kernels; torch is used by callers for device
memory and streams.  There is NO fallback: if the library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_float, c_int, c_int32, c_int64, c_size_t, c_uint32, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmetronome.so")

FLAG_POISON_ON_FREE = 0x1
FLAG_BOOKKEEPING_ONLY = 0x2
FLAG_UNBOUNDED = 0x4
FLAG_KV_FP8 = 0x8

ERR_NAMES = {0: "OK", 1: "INVALID_ARG", 2: "INVALID_SESSION", 3: "DUPLICATE_SESSION", 4: "SESSIONS_FULL",
             5: "POOL_EXHAUSTED", 6: "CHUNK_TOO_LARGE", 7: "QLEN_EXCEEDS_LAST_APPEND", 8: "LAYER_SEQUENCE",
             9: "LEN_OVERFLOW", 10: "CUDA", 11: "UNSUPPORTED", 12: "OUT_OF_MEMORY", 13: "SCRATCH_EXCEEDED"}
STATIC_SCRATCH_BYTES = 16 << 20      # METRONOME_STATIC_SCRATCH_BYTES

# every symbol include/metronome.h and include/metronome_measure.h declare
EXPORTS = ["metronome_abi_version", "metronome_strerror", "metronome_last_cuda_error",
           "metronome_kv_storage_bytes", "metronome_max_blocks_per_session", "metronome_pool_create",
           "metronome_pool_destroy", "metronome_session_open", "metronome_session_close",
           "metronome_append_kv", "metronome_attend_frame", "metronome_attend_frame_static", "metronome_append_attend", "metronome_step_host", "metronome_step_host_async", "metronome_step_host_wait",
           "metronome_session_query", "metronome_pool_query", "metronome_read_kv", "metronome_pool_stats",
           "metronome_pool_set_tuning", "metronome_pool_sm_speeds", "metronome_pool_debug_fail_next", "metronome_pool_debug_read_flags", "metronome_pool_set_profiling", "metronome_pool_read_profile", "metronome_pool_read_stamps",
           "metronome_gate_create", "metronome_gate_destroy", "metronome_gate_observe", "metronome_gate_admit",
           "metronome_stream_read_gbs"]


class MetronomeError(RuntimeError):
    def __init__(self, status: int, detail: str = ""):
        self.status = status
        self.code = ERR_NAMES.get(status, f"UNKNOWN_{status}")
        super().__init__(f"{self.code}" + (f": {detail}" if detail else ""))


class PoolConfig(ctypes.Structure):
    _fields_ = [("n_layers", c_int32), ("n_q_heads", c_int32), ("n_kv_heads", c_int32), ("head_dim", c_int32),
                ("block_size", c_int32), ("n_sinks", c_int32), ("window", c_int32), ("max_sessions", c_int32),
                ("max_new_tokens", c_int32), ("n_blocks", c_int32), ("softmax_scale", c_float), ("flags", c_uint32),
                ("max_session_len", c_int64), ("kv_storage", c_void_p), ("kv_storage_bytes", c_size_t)]


_lib = None


def load():
    """Loads libmetronome.so; fails loudly if it has not been built (no CPU fallback exists)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2607_02640_b200.build` "
                          "(or __graft_entry__.build()). There is no fallback path.")
    lib = ctypes.CDLL(LIB_PATH)
    i32p = POINTER(c_int32)
    lib.metronome_abi_version.restype = c_int
    lib.metronome_strerror.restype = c_char_p
    lib.metronome_strerror.argtypes = [c_int]
    lib.metronome_last_cuda_error.restype = c_char_p
    lib.metronome_last_cuda_error.argtypes = [c_void_p]
    lib.metronome_kv_storage_bytes.restype = c_size_t
    lib.metronome_kv_storage_bytes.argtypes = [POINTER(PoolConfig)]
    lib.metronome_max_blocks_per_session.restype = c_int32
    lib.metronome_max_blocks_per_session.argtypes = [c_int32] * 4
    lib.metronome_pool_create.argtypes = [POINTER(PoolConfig), POINTER(c_void_p)]
    lib.metronome_pool_destroy.argtypes = [c_void_p]
    lib.metronome_session_open.argtypes = [c_void_p, i32p]
    lib.metronome_session_close.argtypes = [c_void_p, c_int32, c_void_p]
    lib.metronome_append_kv.argtypes = [c_void_p, c_int32, c_int32, i32p, i32p, c_void_p, c_void_p, c_void_p]
    lib.metronome_attend_frame.argtypes = [c_void_p, c_int32, c_int32, i32p, i32p, c_void_p, c_void_p, c_void_p]
    lib.metronome_attend_frame_static.argtypes = [c_void_p, c_int32, c_int32, i32p, i32p, c_void_p, c_void_p, c_void_p]
    lib.metronome_append_attend.argtypes = [c_void_p, c_int32, c_int32, i32p, i32p, c_void_p, c_void_p, c_void_p,
                                            c_void_p, c_void_p]
    lib.metronome_step_host.argtypes = [c_void_p, c_int32, c_int32, i32p, i32p, c_void_p, c_void_p, c_void_p,
                                        c_void_p, c_void_p]
    lib.metronome_step_host_async.argtypes = lib.metronome_step_host.argtypes
    lib.metronome_step_host_wait.argtypes = [c_void_p, c_int32]
    lib.metronome_session_query.argtypes = [c_void_p, c_int32, c_void_p, POINTER(c_int64), i32p, i32p, i32p]
    lib.metronome_pool_query.argtypes = [c_void_p, c_void_p, i32p, i32p]
    lib.metronome_read_kv.argtypes = [c_void_p, c_int32, c_int32, c_int64, c_int32, c_void_p, c_void_p, c_void_p]
    lib.metronome_pool_stats.argtypes = [c_void_p, POINTER(c_int64), POINTER(c_int64), POINTER(c_int64)]
    lib.metronome_pool_set_tuning.argtypes = [c_void_p, c_int32, c_int32, c_int32, c_int32]
    lib.metronome_pool_sm_speeds.argtypes = [c_void_p, i32p, i32p, POINTER(ctypes.c_double)]
    lib.metronome_pool_debug_fail_next.argtypes = [c_void_p, c_int32]
    lib.metronome_pool_debug_read_flags.argtypes = [c_void_p, c_void_p, i32p]
    lib.metronome_pool_set_profiling.argtypes = [c_void_p, c_int32]
    lib.metronome_pool_read_stamps.argtypes = [c_void_p, c_int32, i32p, POINTER(ctypes.c_double), POINTER(ctypes.c_double), i32p]
    lib.metronome_pool_read_profile.argtypes = [c_void_p, POINTER(ctypes.c_double), POINTER(c_int64), c_int32]
    lib.metronome_gate_create.argtypes = [c_void_p, POINTER(c_void_p)]
    lib.metronome_gate_destroy.argtypes = [c_void_p]
    lib.metronome_gate_observe.argtypes = [c_void_p, c_float, POINTER(c_float)]
    lib.metronome_gate_admit.argtypes = [c_void_p, c_int32, i32p]
    lib.metronome_stream_read_gbs.argtypes = [c_size_t, c_int32, c_void_p, POINTER(ctypes.c_double)]
    _lib = lib
    return lib


def max_blocks_per_session(S: int, W: int, B: int, max_new_tokens: int) -> int:
    return int(load().metronome_max_blocks_per_session(S, W, B, max_new_tokens))


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(POINTER(c_int32))


def _ptr(t):
    """torch tensor (device or pinned host) or raw integer address -> c_void_p."""
    if t is None:
        return None
    if isinstance(t, int):
        return c_void_p(t)
    return c_void_p(t.data_ptr())


class Pool:
    """metronome_pool_t with the header's entry points (same names, same argument order)."""

    def __init__(self, *, n_q_heads, n_kv_heads, head_dim, n_sinks, window, n_blocks, max_sessions,
                 max_new_tokens, n_layers=1, block_size=16, softmax_scale=0.0, flags=0, max_session_len=0,
                 kv_storage=None, kv_storage_bytes=0):
        self._lib = load()
        self._h = c_void_p()
        self.cfg = PoolConfig(n_layers, n_q_heads, n_kv_heads, head_dim, block_size, n_sinks, window, max_sessions,
                              max_new_tokens, n_blocks, softmax_scale, flags, max_session_len,
                              kv_storage, kv_storage_bytes)
        self._check(self._lib.metronome_pool_create(byref(self.cfg), byref(self._h)))
        if flags & FLAG_UNBOUNDED:
            self.max_blocks = (max_session_len + block_size - 1) // block_size + 1
        else:
            self.max_blocks = max_blocks_per_session(n_sinks, window, block_size, max_new_tokens)

    def _check(self, status):
        if status != 0:
            detail = ""
            if status in (10, 13) and self._h:
                detail = self._lib.metronome_last_cuda_error(self._h).decode()
            raise MetronomeError(status, detail)

    def kv_storage_bytes(self) -> int:
        return int(self._lib.metronome_kv_storage_bytes(byref(self.cfg)))

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.metronome_pool_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def session_open(self) -> int:
        sid = c_int32(-1)
        self._check(self._lib.metronome_session_open(self._h, byref(sid)))
        return sid.value

    def session_close(self, sid: int, stream=0):
        self._check(self._lib.metronome_session_close(self._h, sid, c_void_p(stream)))

    def append_kv(self, layer, sids, n_new, k_new, v_new, stream=0):
        s, sp = _i32(sids)
        n, np_ = _i32(n_new)
        self._check(self._lib.metronome_append_kv(self._h, layer, len(s), sp, np_, _ptr(k_new), _ptr(v_new),
                                                  c_void_p(stream)))

    def attend_frame(self, layer, sids, q_lens, q, out, stream=0):
        s, sp = _i32(sids)
        n, np_ = _i32(q_lens)
        self._check(self._lib.metronome_attend_frame(self._h, layer, len(s), sp, np_, _ptr(q), _ptr(out),
                                                     c_void_p(stream)))

    def attend_frame_static(self, layer, sids, q_lens, q, out, stream=0):
        """attend_frame that allocates nothing: split-KV partials in the library's fixed scratch array."""
        s, sp = _i32(sids)
        n, np_ = _i32(q_lens)
        self._check(self._lib.metronome_attend_frame_static(self._h, layer, len(s), sp, np_, _ptr(q), _ptr(out),
                                                            c_void_p(stream)))

    def append_attend(self, layer, sids, n_new, k_new, v_new, q, out, stream=0):
        s, sp = _i32(sids)
        n, np_ = _i32(n_new)
        self._check(self._lib.metronome_append_attend(self._h, layer, len(s), sp, np_, _ptr(k_new), _ptr(v_new),
                                                      _ptr(q), _ptr(out), c_void_p(stream)))

    def step_host(self, layer, sids, n_new, k_host, v_host, q_host, out_host, stream=0):
        s, sp = _i32(sids)
        n, np_ = _i32(n_new)
        self._check(self._lib.metronome_step_host(self._h, layer, len(s), sp, np_, _ptr(k_host), _ptr(v_host),
                                                  _ptr(q_host), _ptr(out_host), c_void_p(stream)))

    def step_host_async(self, layer, sids, n_new, k_host, v_host, q_host, out_host, stream=0):
        s, sp = _i32(sids)
        n, np_ = _i32(n_new)
        self._check(self._lib.metronome_step_host_async(self._h, layer, len(s), sp, np_, _ptr(k_host), _ptr(v_host),
                                                        _ptr(q_host), _ptr(out_host), c_void_p(stream)))

    def step_host_wait(self, keep=0):
        self._check(self._lib.metronome_step_host_wait(self._h, keep))

    def session_query(self, sid, stream=0):
        """-> (len, first_live_block, [physical block ids in logical order])"""
        ln, fl, nb = c_int64(), c_int32(), c_int32()
        ids = (c_int32 * max(1, self.max_blocks))()
        self._check(self._lib.metronome_session_query(self._h, sid, c_void_p(stream), byref(ln), byref(fl),
                                                      byref(nb), ids))
        return ln.value, fl.value, [ids[i] for i in range(nb.value)]

    def pool_query(self, stream=0, want_ids=True):
        """-> (n_free, [free ids in pop order])"""
        nf = c_int32()
        ids = (c_int32 * max(1, self.cfg.n_blocks))() if want_ids else None
        self._check(self._lib.metronome_pool_query(self._h, c_void_p(stream), byref(nf), ids))
        return nf.value, ([ids[i] for i in range(nf.value)] if want_ids else None)

    def read_kv(self, layer, sid, pos0, n, k_out, v_out, stream=0):
        self._check(self._lib.metronome_read_kv(self._h, layer, sid, pos0, n, _ptr(k_out), _ptr(v_out),
                                                c_void_p(stream)))

    def stats(self):
        a, b, c = c_int64(), c_int64(), c_int64()
        self._check(self._lib.metronome_pool_stats(self._h, byref(a), byref(b), byref(c)))
        return {"kernel_launches": a.value, "append_calls": b.value, "attend_calls": c.value}

    def set_tuning(self, split_tokens=0, kernel_family=0, gqa_dynamic=0, fused_step=0):
        self._check(self._lib.metronome_pool_set_tuning(self._h, split_tokens, kernel_family, gqa_dynamic, fused_step))

    def sm_speeds(self):
        """-> (SMs, slow SMs, their relative speed) as measured at pool creation."""
        n, ns, r = c_int32(), c_int32(), ctypes.c_double()
        self._check(self._lib.metronome_pool_sm_speeds(self._h, byref(n), byref(ns), byref(r)))
        return n.value, ns.value, r.value

    def debug_fail_next(self, stage: int):
        self._check(self._lib.metronome_pool_debug_fail_next(self._h, stage))

    def debug_read_flags(self, stream=0):
        buf = (c_int32 * 16)()
        self._check(self._lib.metronome_pool_debug_read_flags(self._h, c_void_p(stream), buf))
        return list(buf)

    def set_profiling(self, mode):
        """0 off, 1 (or True) event brackets, 2 in-kernel %globaltimer stamps (launches unchanged)."""
        self._check(self._lib.metronome_pool_set_profiling(self._h, int(mode)))

    def read_stamps(self, max_launches=1 << 15):
        """-> (kinds, span_ms, start_ms) numpy arrays, one entry per stamped attention launch; clears them."""
        kinds = np.zeros(max_launches, np.int32)
        span = np.zeros(max_launches, np.float64)
        start = np.zeros(max_launches, np.float64)
        n = c_int32()
        self._check(self._lib.metronome_pool_read_stamps(
            self._h, max_launches, kinds.ctypes.data_as(POINTER(c_int32)), span.ctypes.data_as(POINTER(ctypes.c_double)),
            start.ctypes.data_as(POINTER(ctypes.c_double)), byref(n)))
        return kinds[:n.value], span[:n.value], start[:n.value]

    def read_profile(self, reset=True):
        """-> (summed attention-kernel milliseconds, bracketed launches)"""
        ms, n = ctypes.c_double(), c_int64()
        self._check(self._lib.metronome_pool_read_profile(self._h, byref(ms), byref(n), int(reset)))
        return ms.value, n.value


def stream_read_gbs(n_bytes: int = 4 << 30, reps: int = 5, stream=0) -> float:
    """Read-only HBM stream microbenchmark (best of `reps`), GB/s."""
    out = ctypes.c_double()
    st = load().metronome_stream_read_gbs(n_bytes, reps, c_void_p(stream), byref(out))
    if st:
        raise MetronomeError(st)
    return out.value


class GateConfig(ctypes.Structure):
    _fields_ = [("budget_ms", c_float), ("target_frac", c_float), ("add_step", c_float), ("mult_factor", c_float),
                ("cap_min", c_float), ("cap_max", c_float), ("cap_init", c_float)]


class Gate:
    """metronome_gate_t: the AIMD admission gate of PAPER.md:L105-111 (NEXT row f3).  Host-only."""

    def __init__(self, *, budget_ms, target_frac, add_step, mult_factor, cap_min, cap_max, cap_init):
        self._lib = load()
        self._h = c_void_p()
        cfg = GateConfig(budget_ms, target_frac, add_step, mult_factor, cap_min, cap_max, cap_init)
        st = self._lib.metronome_gate_create(byref(cfg), byref(self._h))
        if st:
            raise MetronomeError(st)

    def observe(self, frame_latency_ms: float) -> float:
        cap = c_float()
        st = self._lib.metronome_gate_observe(self._h, c_float(frame_latency_ms), byref(cap))
        if st:
            raise MetronomeError(st)
        return cap.value

    def admit(self, n_live: int) -> bool:
        out = c_int32()
        st = self._lib.metronome_gate_admit(self._h, n_live, byref(out))
        if st:
            raise MetronomeError(st)
        return bool(out.value)

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.metronome_gate_destroy(self._h)
            self._h = None
