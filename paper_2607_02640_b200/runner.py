"""Drives a workload schedule (workloads.py) through the C-ABI library (binding.py).

Plumbing only: it opens sessions, generates each step's seeded K/V/Q rows on the device with
synth.rows(), and issues append_kv / attend_frame.  Used by bench.py, the GPU tests and smoke().
Every row's coordinates (session uid, absolute position) are exposed so that a test can regenerate
the same bf16 values on the CPU for the oracle.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

from . import binding, synth
from .workloads import Workload


@dataclass
class Step:
    """One batched append+attend: rows are in batch order, session after session."""
    local: np.ndarray        # workload-local session index per batch item
    sids: np.ndarray         # library session ids per batch item
    n_new: np.ndarray        # tokens per batch item
    uid_rows: np.ndarray     # per row: session uid (synth coordinate)
    pos_rows: np.ndarray     # per row: absolute position
    timed: bool
    frame: int


class Runner:
    def __init__(self, w: Workload, n_layers: int = 1, flags: int = 0, device: str = "cuda",
                 softmax_scale: float = 0.0, uid_base: int = 0, max_session_len: int = 0):
        self.w = w
        self.n_layers = n_layers
        self.device = torch.device(device)
        self.pool = binding.Pool(n_q_heads=w.n_q_heads, n_kv_heads=w.n_kv_heads, head_dim=w.head_dim,
                                 n_sinks=w.S, window=w.W, n_blocks=w.n_blocks, max_sessions=w.slots,
                                 max_new_tokens=w.max_new_tokens, n_layers=n_layers,
                                 block_size=w.block_size, softmax_scale=softmax_scale, flags=flags,
                                 max_session_len=max_session_len)
        self.sid = {}            # local index -> library sid
        self.uid = {}            # local index -> unique session uid (fresh on every open)
        self.length = {}         # local index -> tokens so far
        self._next_uid = uid_base    # replicas draw different inputs (replicas.uid_base)
        oc = w.outlier_channels()
        self.outliers = torch.from_numpy(oc).to(self.device) if oc.size else None

    # -- session events
    def open(self, i: int):
        self.sid[i] = self.pool.session_open()
        self.uid[i] = self._next_uid
        self._next_uid += 1
        self.length[i] = 0

    def close(self, i: int, stream=0):
        self.pool.session_close(self.sid.pop(i), stream)
        del self.uid[i], self.length[i]

    # -- steps
    def make_step(self, ev) -> Step:
        """Resolves a ("step", idx, n_new, timed, frame) event and advances the host-side lengths."""
        _, idx, n_new, timed, frame = ev
        uid_rows = np.repeat(np.asarray([self.uid[int(i)] for i in idx], np.int64), n_new)
        pos_rows = np.concatenate([np.arange(self.length[int(i)], self.length[int(i)] + int(n), dtype=np.int64)
                                   for i, n in zip(idx, n_new)]) if len(idx) else np.zeros(0, np.int64)
        for i, n in zip(idx, n_new):
            self.length[int(i)] += int(n)
        sids = np.asarray([self.sid[int(i)] for i in idx], np.int32)
        return Step(np.asarray(idx, np.int32), sids, np.asarray(n_new, np.int32), uid_rows, pos_rows, timed, frame)

    def rows(self, stream_tag: int, layer: int, uid_rows, pos_rows, device=None) -> torch.Tensor:
        dev = self.device if device is None else torch.device(device)
        heads = self.w.n_q_heads if stream_tag == synth.STREAM_Q else self.w.n_kv_heads
        out_ch = None
        if stream_tag != synth.STREAM_Q and self.outliers is not None:
            out_ch = self.outliers.to(dev)
        return synth.rows(self.w.seed, stream_tag, layer, torch.from_numpy(np.asarray(uid_rows)).to(dev),
                          torch.from_numpy(np.asarray(pos_rows)).to(dev), heads, self.w.head_dim,
                          out_ch, self.w.outlier_scale)

    def append(self, st: Step, layer: int, k=None, v=None, stream=0):
        if k is None:
            k = self.rows(synth.STREAM_K, layer, st.uid_rows, st.pos_rows)
            v = self.rows(synth.STREAM_V, layer, st.uid_rows, st.pos_rows)
        self.pool.append_kv(layer, st.sids, st.n_new, k, v, stream)
        return k, v

    def attend(self, st: Step, layer: int, q=None, out=None, stream=0):
        if q is None:
            q = self.rows(synth.STREAM_Q, layer, st.uid_rows, st.pos_rows)
        if out is None:
            out = torch.empty_like(q)
        self.pool.attend_frame(layer, st.sids, st.n_new, q, out, stream)
        return out

    def step(self, st: Step, layer: int, k=None, v=None, q=None, out=None, stream=0):
        """append + attend of one sub-step in ONE call (metronome_append_attend)."""
        if k is None:
            k = self.rows(synth.STREAM_K, layer, st.uid_rows, st.pos_rows)
            v = self.rows(synth.STREAM_V, layer, st.uid_rows, st.pos_rows)
        if q is None:
            q = self.rows(synth.STREAM_Q, layer, st.uid_rows, st.pos_rows)
        if out is None:
            out = torch.empty_like(q)
        self.pool.append_attend(layer, st.sids, st.n_new, k, v, q, out, stream)
        return out

    def run_history(self, events, rows_per_batch: int = 16384):
        """Executes the untimed prefix of a schedule (opens, closes, history appends on every layer)
        and returns the remaining events.  K/V rows of many steps are generated in one go, then
        issued step by step, layer by layer (layers > 0 repeat layer 0's batch, reading R16)."""
        pending: list[Step] = []
        n_rows = 0
        k = 0

        def flush():
            nonlocal pending, n_rows
            if not pending:
                return
            uid = np.concatenate([s.uid_rows for s in pending])
            pos = np.concatenate([s.pos_rows for s in pending])
            KV = [(self.rows(synth.STREAM_K, layer, uid, pos), self.rows(synth.STREAM_V, layer, uid, pos))
                  for layer in range(self.n_layers)]
            r = 0
            for s in pending:
                m = int(s.n_new.sum())
                for layer in range(self.n_layers):
                    self.pool.append_kv(layer, s.sids, s.n_new, KV[layer][0][r:r + m], KV[layer][1][r:r + m])
                r += m
            pending, n_rows = [], 0

        while k < len(events):
            ev = events[k]
            if ev[0] == "step" and ev[3]:
                break
            if ev[0] == "open":
                self.open(ev[1])
            elif ev[0] == "close":
                flush()
                self.close(ev[1])
            else:
                st = self.make_step(ev)
                pending.append(st)
                n_rows += len(st.uid_rows)
                if n_rows >= rows_per_batch:
                    flush()
            k += 1
        flush()
        return events[k:]
