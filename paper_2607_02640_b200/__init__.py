"""paper_2607_02640_b200 -- B200-native (sm_100a) bounded-window paged attention, the data-parallel
hot path of Metronome's per-frame serving step (arxiv/paper_2607_02640, sec. 4.1, App. A).

The product is the C-ABI library libmetronome.so (include/metronome.h) built from csrc/;
`binding` is its thin ctypes mirror.  Submodules are imported lazily so that `synth` and
`workloads` (pure input recipes) can be used without loading the CUDA library.
"""
__all__ = ["binding", "synth", "workloads", "build", "runner"]
