"""B200-native DepthWeave-KV decode-attention hot path (arxiv/paper_2607_06523).

`binding` is the thin ctypes layer over the C-ABI library libdwkv.so (include/dwkv.h); `harness` fills caches from the
seeded generators in `gen/`. Importing `binding` fails loudly if the CUDA library has not been built.
"""
from . import build as build_lib  # noqa: F401


def load():
    from . import binding
    return binding
