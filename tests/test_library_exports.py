"""CPU: the C-ABI library builds/loads and exports every symbol include/promoe.h declares (no compute calls)."""
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_header_symbols_are_exported():
    from paper_2410_22134_b200.build import build
    build()
    from paper_2410_22134_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "promoe.h")).read()
    declared = sorted(set(re.findall(r"PROMOE_API [\w\s\*]*?(promoe_\w+)\(", hdr)))
    assert len(declared) >= 16
    L = binding.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert sorted(binding.EXPORTS) == declared
    # measurement hooks used by bench.py only: a header of their own, not part of the product API
    bhdr = open(os.path.join(ROOT, "include", "promoe_bench.h")).read()
    bdecl = sorted(set(re.findall(r"PROMOE_API [\w\s\*]*?(promoe_\w+)\(", bhdr)))
    assert bdecl == sorted(binding.BENCH_EXPORTS) and not set(bdecl) & set(declared)
    for name in bdecl:
        assert hasattr(L, name), name


def test_struct_layouts_match_header():
    import ctypes
    from paper_2410_22134_b200 import binding as B
    # sizes computed from the header's field lists (all int32/float/uint64/double/pointers, natural alignment)
    assert ctypes.sizeof(B.promoe_shape_t) == 17 * 4 + 2 * 4
    assert ctypes.sizeof(B.promoe_opts_t) == 64
    assert ctypes.sizeof(B.promoe_dense_t) == 15 * 8
    assert ctypes.sizeof(B.promoe_stats_t) == 27 * 8 + 3 * 8 + 8
