"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/dwkv.h declares.
No compute calls (no GPU here)."""
import os
import re

import __graft_entry__ as entry

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_build_and_exports_match_header():
    entry.build()
    from paper_2607_06523_b200 import binding
    header = open(os.path.join(ROOT, "include", "dwkv.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(dwkv_[a-z_]+)\s*\(", header))
    assert declared, "no declarations parsed"
    for name in declared:
        assert hasattr(binding.lib, name), f"{name} declared in dwkv.h but not exported"
    assert declared == set(binding.EXPORTED)


def test_config_struct_layout_matches_header():
    from paper_2607_06523_b200 import binding
    import ctypes as C
    f = binding.dwkv_config
    assert f.max_tokens_per_seq.offset == 48 and f.softmax_scale.offset == 56 and f.arena.offset == 64
    assert C.sizeof(f) == 80


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2607_06523_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in src.replace("no oracle", ""), f"{fn} mentions the oracle"
