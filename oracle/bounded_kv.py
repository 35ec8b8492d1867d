"""oracle/bounded_kv.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain CPU oracle for Metronome's bounded per-session KV cache (sec. 4.1, App. A).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It shares no code with paper_2607_02640_b200/ and never imports it.

Two layers, so that bookkeeping and arithmetic are pinned separately:

  DefinitionOracle  keeps every session's ENTIRE unpaged K/V history and evaluates
                    admit(j,t) = j<=t and (j<S or t-j<W) directly over positions 0..len-1
                    ("[0,S) U [t-W,t]", L258 "OR-term k < S").
  PagedOracle       simulates the fixed block pool (L60), the per-session block list with a pinned
                    head and a freed middle (L256 "frees blocks that fall entirely behind the
                    window", L258 "pins each request's first ceil(S/block) blocks"), stores K/V
                    ONLY in simulated blocks, NaN-poisons freed blocks (L258 "freed blocks
                    NaN-poisoned") and evaluates attention ONLY through the block table.

Both call the same float32 routine (oracle/attention_ref.c) with keys in ascending position, so
they must agree bit for bit: that proves residency >= admitted set.

Free-list discipline (LIFO, two-phase append, batch order) is NOT fixed by the paper; it is
DESIGN.md reading R6 -- "parity unpinned" by the paper for that convention alone; everything the
paper does fix (which blocks are resident, which keys are attended) is pinned in tests/.

bf16 values travel as numpy uint16 bit patterns.
"""
from __future__ import annotations

import ctypes
import math
import os
from dataclasses import dataclass, field

import numpy as np

from .build import LIB, build_oracle

BF16_NAN = np.uint16(0x7FC0)

# ----------------------------------------------------------------------------- error vocabulary


class OracleError(Exception):
    """Raised with the same symbolic name the C-ABI uses (include/metronome.h)."""

    def __init__(self, code: str, msg: str = ""):
        super().__init__(f"{code}: {msg}")
        self.code = code


# ----------------------------------------------------------------------------- C routine loader

_lib = None


def _load():
    global _lib
    if _lib is None:
        build_oracle()
        lib = ctypes.CDLL(LIB)
        u16p = ctypes.POINTER(ctypes.c_uint16)
        i64p = ctypes.POINTER(ctypes.c_int64)
        f32p = ctypes.POINTER(ctypes.c_float)
        for name in ("oracle_attend_f32", "oracle_attend_f64", "oracle_attend_kvf32_f32", "oracle_attend_kvf32_f64"):
            fn = getattr(lib, name)
            kvp = f32p if "kvf32" in name else u16p
            fn.restype = ctypes.c_int
            fn.argtypes = [u16p, i64p, ctypes.c_int64, kvp, kvp, i64p, ctypes.c_int64,
                           ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int64,
                           ctypes.c_int64, ctypes.c_double, f32p, f32p, ctypes.c_int32]
        lib.oracle_admit.restype = ctypes.c_int
        lib.oracle_admit.argtypes = [ctypes.c_int64] * 4
        lib.oracle_max_threads.restype = ctypes.c_int32
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def admit(j: int, t: int, S: int, W: int) -> bool:
    """admit(j,t) = j<=t and (j<S or t-j<W); reading R1 (W keys incl. t)."""
    return bool(_load().oracle_admit(j, t, S, W))


def attend(q, q_pos, k, v, k_pos, S, W, scale=None, precision="f32", want_weights=False,
           n_threads=1):
    """Masked softmax attention for ONE session (definition in attention_ref.c's header).

    q [n_q,Hq,D] uint16(bf16), q_pos [n_q] absolute positions; k,v [n_k,Hkv,D] uint16(bf16) -- or float32 VALUES
    (the fp8 KV arm: dequantised rows) --, k_pos [n_k] ascending.  Returns float32 out [n_q,Hq,D] (and weights
    [n_q,Hq,n_k] if asked)."""
    lib = _load()
    q = np.ascontiguousarray(q, dtype=np.uint16)
    kv_f32 = np.asarray(k).dtype == np.float32
    k = np.ascontiguousarray(k, dtype=np.float32 if kv_f32 else np.uint16)
    v = np.ascontiguousarray(v, dtype=np.float32 if kv_f32 else np.uint16)
    q_pos = np.ascontiguousarray(q_pos, dtype=np.int64)
    k_pos = np.ascontiguousarray(k_pos, dtype=np.int64)
    n_q, Hq, D = q.shape
    n_k, Hkv, D2 = k.shape
    assert D2 == D and v.shape == k.shape and q_pos.shape == (n_q,) and k_pos.shape == (n_k,)
    assert np.all(np.diff(k_pos) > 0), "keys must be in ascending position"
    if scale is None:
        scale = 1.0 / math.sqrt(D)  # reading R7
    out = np.empty((n_q, Hq, D), dtype=np.float32)
    weights = np.empty((n_q, Hq, n_k), dtype=np.float32) if want_weights else None
    fn = getattr(lib, ("oracle_attend_kvf32_" if kv_f32 else "oracle_attend_") + ("f32" if precision == "f32" else "f64"))
    u16p = ctypes.POINTER(ctypes.c_uint16)
    i64p = ctypes.POINTER(ctypes.c_int64)
    f32p = ctypes.POINTER(ctypes.c_float)
    rc = fn(q.ctypes.data_as(u16p), q_pos.ctypes.data_as(i64p), n_q,
            k.ctypes.data_as(f32p if kv_f32 else u16p), v.ctypes.data_as(f32p if kv_f32 else u16p), k_pos.ctypes.data_as(i64p), n_k,
            Hq, Hkv, D, int(S), int(W), float(scale),
            out.ctypes.data_as(f32p),
            weights.ctypes.data_as(f32p) if want_weights else None, int(n_threads))
    if rc != 0:
        raise RuntimeError("oracle_attend failed")
    return (out, weights) if want_weights else out


# ----------------------------------------------------------------------------- shared config


@dataclass
class PoolConfig:
    """Names follow the paper: S sinks, W window, block = KV block of 16 tokens (L149, L145)."""
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    S: int
    W: int
    n_blocks: int
    block_size: int = 16
    max_sessions: int = 512
    max_new_tokens: int = 32
    n_layers: int = 1
    scale: float | None = None
    max_session_len: int = 2**31 - 1 - 4096
    unbounded: bool = False  # the paper's vanilla arm: nothing is ever freed, full causal mask
    kv_fp8: bool = False     # K / V rows are stored as e4m3 codes + one scale per (token, KV head): oracle/kv_fp8.py

    @property
    def n_sink(self) -> int:  # ceil(S / block)
        return -(-self.S // self.block_size)

    @property
    def W_eff(self) -> int:
        return 2**62 if self.unbounded else self.W


def max_blocks_per_session(S: int, W: int, B: int, max_new_tokens: int) -> int:
    """Worst-case resident blocks of one session, by brute force over every phase of the ring
    (the closed form n_sink + floor((W+n_max-1)/B) + 2 lives in the product; this is its check).
    PAPER.md:L258 "the per-request admission cap counts the pinned blocks"."""
    n_sink = -(-S // B)
    worst = 0
    # resident after an append of n tokens to a session of length L0 (old enough that the ring
    # is in steady state, and every alignment of L0 modulo B)
    base = (n_sink + (W // B) + 4) * B
    for L0 in range(0, base + 2 * B):
        for n in range(1, max_new_tokens + 1):
            L1 = L0 + n
            first = max(n_sink, max(0, L0 - W + 1) // B)
            nblk = -(-L1 // B)
            resident = min(n_sink, nblk) + max(0, nblk - first)
            worst = max(worst, resident)
    return worst


# ----------------------------------------------------------------------------- layer 1


class DefinitionOracle:
    """Layer 1: whole unpaged history per session, formula applied directly."""

    def __init__(self, cfg: PoolConfig):
        self.cfg = cfg
        # [layer][sid] -> (K [len,Hkv,D] uint16, V)
        self.hist: list[dict[int, list[np.ndarray]]] = [dict() for _ in range(cfg.n_layers)]
        self.length: dict[int, int] = {}
        self.last_n: dict[int, int] = {}

    def session_open(self) -> int:
        sid = 0
        while sid in self.length:
            sid += 1
        if sid >= self.cfg.max_sessions:
            raise OracleError("SESSIONS_FULL")
        self.length[sid] = 0
        self.last_n[sid] = 0
        c = self.cfg
        dt = np.float32 if c.kv_fp8 else np.uint16
        for layer in range(c.n_layers):
            self.hist[layer][sid] = [np.zeros((0, c.n_kv_heads, c.head_dim), dt),
                                     np.zeros((0, c.n_kv_heads, c.head_dim), dt)]
        return sid

    def session_close(self, sid: int) -> None:
        if sid not in self.length:
            raise OracleError("INVALID_SESSION")
        del self.length[sid], self.last_n[sid]
        for layer in range(self.cfg.n_layers):
            del self.hist[layer][sid]

    def append_kv(self, layer: int, sids, n_new, k_new, v_new) -> None:
        """k_new/v_new: [sum n_new, Hkv, D] uint16 in batch order (PAPER.md:L46 'prefill the new chunk').
        In the fp8 arm every row is replaced by what its stored form decodes to (kv_fp8.roundtrip)."""
        if self.cfg.kv_fp8:
            from . import kv_fp8
            k_new, v_new = kv_fp8.roundtrip(k_new), kv_fp8.roundtrip(v_new)
        row = 0
        for sid, n in zip(sids, n_new):
            if sid not in self.length:
                raise OracleError("INVALID_SESSION")
            h = self.hist[layer][sid]
            h[0] = np.concatenate([h[0], k_new[row:row + n]], axis=0)
            h[1] = np.concatenate([h[1], v_new[row:row + n]], axis=0)
            row += n
            if layer == 0:
                self.length[sid] += n
                self.last_n[sid] = n

    def attend_frame(self, layer: int, sids, q_lens, q, precision="f32", want_weights=False,
                     n_threads=1):
        """Queries are the LAST q_lens[i] positions of session i (decode: 1; chunk: n)."""
        c = self.cfg
        outs, weights = [], []
        row = 0
        for sid, ql in zip(sids, q_lens):
            K, V = self.hist[layer][sid]
            L = K.shape[0]
            q_pos = np.arange(L - ql, L, dtype=np.int64)
            r = attend(q[row:row + ql], q_pos, K, V, np.arange(L, dtype=np.int64), c.S, c.W_eff,
                       c.scale, precision, want_weights, n_threads)
            if want_weights:
                outs.append(r[0]); weights.append(r[1])
            else:
                outs.append(r)
            row += ql
        out = np.concatenate(outs, axis=0) if outs else np.zeros((0, c.n_q_heads, c.head_dim), np.float32)
        return (out, weights) if want_weights else out


# ----------------------------------------------------------------------------- layer 2


@dataclass
class _Session:
    length: int = 0
    first_live: int = 0          # first logical NON-sink block still resident
    last_n: int = 0
    table: dict = field(default_factory=dict)   # logical block -> physical block id


class PagedOracle:
    """Layer 2: block pool + free list + block tables, attention only through the tables.

    Bookkeeping rules:
      1. pool ids 0..n_blocks-1; the free list is a LIFO stack whose initial pop order is 0,1,2,...
      2. session_open: lowest free slot id; len=0; first_live=n_sink; no blocks.
      3. append_kv(layer 0) over the batch, in batch order:
           phase 1 (frees)   new_first = max(first_live, n_sink, floor(max(0, L0-W+1)/B));
                             push logical blocks [first_live, new_first) ascending.
                             (block b is freed iff b>=n_sink and (b+1)*B <= L0-W+1: every key in it
                             is outside the window of position L0, the oldest query of this frame:
                             PAPER.md:L256 "frees blocks that fall entirely behind the window")
           check             free + sum(frees) >= sum(allocs), else POOL_EXHAUSTED, nothing changes
                             (PAPER.md:L60 is the stall this replaces)
           phase 2 (allocs)  pop ceil(L1/B)-ceil(L0/B) blocks per session, ascending; len=L1.
      4. token p lives in logical block p//B, row p%B; logical blocks < n_sink are never freed
         ("pins each request's first ceil(S/block) blocks instead of freeing them").
      5. session_close: push sink blocks then live window blocks, ascending; release the slot.
    """

    def __init__(self, cfg: PoolConfig, poison_on_free: bool = True, store_kv: bool = True):
        self.cfg = cfg
        self.poison = poison_on_free
        self.store_kv = store_kv
        self.free = list(range(cfg.n_blocks - 1, -1, -1))  # pop() from the end => 0,1,2,...
        self.sessions: dict[int, _Session] = {}
        self.kv = None
        if store_kv:
            shape = (cfg.n_layers, 2, cfg.n_blocks, cfg.block_size, cfg.n_kv_heads, cfg.head_dim)
            self.kv = np.full(shape, BF16_NAN, dtype=np.uint16)  # never-written storage is poison too
        self.last_batch = None
        self.layer_done = [0] * cfg.n_layers
        self.epoch = 0

    # -- sessions
    def session_open(self) -> int:
        sid = 0
        while sid in self.sessions:
            sid += 1
        if sid >= self.cfg.max_sessions:
            raise OracleError("SESSIONS_FULL")
        self.sessions[sid] = _Session(first_live=self.cfg.n_sink)
        return sid

    def session_close(self, sid: int) -> None:
        if sid not in self.sessions:
            raise OracleError("INVALID_SESSION")
        s = self.sessions[sid]
        for b in sorted(s.table):  # sinks (ascending) then live window blocks (ascending)
            self._free_block(s.table[b])
        del self.sessions[sid]

    def _free_block(self, phys: int) -> None:
        if self.poison and self.kv is not None:
            self.kv[:, :, phys] = BF16_NAN
        self.free.append(phys)

    # -- append
    def plan_append(self, sids, n_new):
        """Counts of an append, without changing anything (frees, allocs per session)."""
        c = self.cfg
        B = c.block_size
        if len(set(sids)) != len(sids):
            raise OracleError("DUPLICATE_SESSION")
        plan = []
        for sid, n in zip(sids, n_new):
            if sid not in self.sessions:
                raise OracleError("INVALID_SESSION")
            if n < 0:
                raise OracleError("INVALID_ARG")
            if n > c.max_new_tokens:
                raise OracleError("CHUNK_TOO_LARGE")
            s = self.sessions[sid]
            L0, L1 = s.length, s.length + n
            if L1 > c.max_session_len:
                raise OracleError("LEN_OVERFLOW")
            new_first = max(s.first_live, c.n_sink, max(0, L0 - c.W_eff + 1) // B)
            n_alloc = -(-L1 // B) - (-(-L0 // B))
            plan.append((sid, n, L0, L1, new_first, n_alloc))
        return plan

    def append_kv(self, layer: int, sids, n_new, k_new=None, v_new=None) -> None:
        c = self.cfg
        B = c.block_size
        sids = [int(x) for x in sids]
        n_new = [int(x) for x in n_new]
        if not (0 <= layer < c.n_layers):
            raise OracleError("INVALID_ARG")
        if layer == 0:
            plan = self.plan_append(sids, n_new)
            total_free = 0
            for sid, n, L0, L1, new_first, n_alloc in plan:
                s = self.sessions[sid]
                total_free += sum(1 for b in range(s.first_live, new_first) if b in s.table)
            total_alloc = sum(p[5] for p in plan)
            if len(self.free) + total_free < total_alloc:
                raise OracleError("POOL_EXHAUSTED")      # nothing has changed
            # phase 1: all frees, batch order
            for sid, n, L0, L1, new_first, n_alloc in plan:
                s = self.sessions[sid]
                for b in range(s.first_live, new_first):
                    if b in s.table:
                        self._free_block(s.table.pop(b))
                s.first_live = new_first
            # phase 2: all allocations, batch order
            for sid, n, L0, L1, new_first, n_alloc in plan:
                s = self.sessions[sid]
                for b in range(-(-L0 // B), -(-L1 // B)):
                    s.table[b] = self.free.pop()
                s.length = L1
                s.last_n = n
            self.epoch += 1
            self.layer_done[0] = self.epoch
            self.last_batch = (list(sids), list(n_new))
        else:
            if self.last_batch is None or self.last_batch != (list(sids), list(n_new)) \
                    or self.layer_done[layer] >= self.epoch:
                raise OracleError("LAYER_SEQUENCE")
            self.layer_done[layer] = self.epoch
        # K/V rows go to their paged slots (rule 4)
        if self.store_kv and k_new is not None:
            row = 0
            for sid, n in zip(sids, n_new):
                s = self.sessions[sid]
                for i in range(n):
                    p = s.length - n + i
                    phys = s.table[p // B]
                    self.kv[layer, 0, phys, p % B] = k_new[row]
                    self.kv[layer, 1, phys, p % B] = v_new[row]
                    row += 1

    # -- attention through the table only
    def resident_positions(self, sid: int) -> np.ndarray:
        s = self.sessions[sid]
        B = self.cfg.block_size
        pos = []
        for b in sorted(s.table):
            lo, hi = b * B, min((b + 1) * B, s.length)
            pos.extend(range(lo, hi))
        return np.asarray(pos, dtype=np.int64)

    def attend_frame(self, layer: int, sids, q_lens, q, precision="f32", want_weights=False):
        c = self.cfg
        if c.kv_fp8:       # (the fp8 KV arm is stated at the definition layer only; this layer then checks bookkeeping)
            raise OracleError("PagedOracle has no fp8 arm: attend through DefinitionOracle")
        B = c.block_size
        outs, weights = [], []
        row = 0
        for sid, ql in zip(sids, q_lens):
            if sid not in self.sessions:
                raise OracleError("INVALID_SESSION")
            s = self.sessions[sid]
            if ql > s.last_n:
                raise OracleError("QLEN_EXCEEDS_LAST_APPEND")
            pos = self.resident_positions(sid)
            phys = np.asarray([s.table[p // B] for p in pos], dtype=np.int64)
            K = self.kv[layer, 0, phys, pos % B]
            V = self.kv[layer, 1, phys, pos % B]
            q_pos = np.arange(s.length - ql, s.length, dtype=np.int64)
            r = attend(q[row:row + ql], q_pos, K, V, pos, c.S, c.W_eff, c.scale, precision,
                       want_weights)
            if want_weights:
                outs.append(r[0]); weights.append(r[1])
            else:
                outs.append(r)
            row += ql
        out = np.concatenate(outs, axis=0) if outs else np.zeros((0, c.n_q_heads, c.head_dim), np.float32)
        return (out, weights) if want_weights else out

    # -- introspection (mirrors metronome_session_query / metronome_pool_query)
    def session_query(self, sid: int):
        s = self.sessions[sid]
        blocks = [s.table[b] for b in sorted(s.table)]
        return s.length, s.first_live, blocks

    def pool_query(self):
        """Free ids in POP order (next allocation first)."""
        return list(reversed(self.free))

    def occupancy(self) -> float:
        """rho = fraction of the pool in use (Eq. 1, Fig. 5)."""
        return 1.0 - len(self.free) / self.cfg.n_blocks
