"""CPU: the C-ABI library loads and exports every symbol include/mss.h declares; host-side argument checks
(no compute calls without a GPU)."""
import ctypes as C

import pytest

import paper_1403_2136_b200 as mss
from paper_1403_2136_b200 import build as mss_build
from paper_1403_2136_b200.binding import _Scoring


@pytest.fixture(scope="module")
def L():
    mss_build.build()
    return mss.lib()


def test_every_declared_symbol_is_exported(L):
    names = mss.declared_symbols()
    assert {"mss_genome_load", "mss_map_reads", "mss_nw_align"} <= set(names) and len(names) >= 15
    for n in names:
        assert hasattr(L, n), n


def test_strerror_and_version(L):
    assert L.mss_version() >= 100
    assert b"argument" in L.mss_strerror(-1) and b"range" in L.mss_strerror(-2)
    assert b"workspace" in L.mss_strerror(-3) and b"CUDA" in L.mss_strerror(-4) and L.mss_strerror(0) == b"ok"


def test_host_side_argument_checks(L):
    assert L.mss_genome_workspace_bytes(0, 100, -1) == 0
    assert L.mss_genome_workspace_bytes(1000, 0, -1) == 0
    assert L.mss_genome_workspace_bytes(1000, 100, -2) == 0
    n = L.mss_genome_workspace_bytes(4_600_000, 4096, -1)
    assert 4_600_000 // 4 + 4_600_000 // 8 <= n < 2_000_000
    h = C.c_void_p()
    assert L.mss_genome_load(None, None, 1000, 100, -1, None, 0, None, C.byref(h)) == -1
    assert L.mss_genome_load(C.c_void_p(256), None, 1000, 100, -1, C.c_void_p(512), 16, None, C.byref(h)) == -3
    assert L.mss_genome_load(C.c_void_p(256), None, 1000, 1 << 25, -1, C.c_void_p(512), 1 << 30, None, C.byref(h)) == -2
    assert L.mss_map_workspace_bytes(None, 10, 100, 3) == 0
    sc = _Scoring(5, -4, -26)
    assert L.mss_map_reads(None, None, None, 7, None, 10, 100, sc, 3, None, 0, None, None) == -1
    assert L.mss_nw_align(None, None, None, 7, None, 10, 100, None, sc, 30, None, 0, None, None, None, None, 10, None) == -1
    assert L.mss_mapq_filter(None, 4, 15.2, None, None, None) == -1
    assert L.mss_mapq_filter(None, 0, 15.2, None, None, None) == 0
    assert L.mss_set_scan_variant(99) == -1 and L.mss_set_scan_variant(0) == 0
    assert L.mss_genome_free(None) == -1


def test_tuning_switches_and_static_entry_point_check_their_arguments(L):
    """Host-only: the round-2 additions reject bad values before touching a device."""
    assert L.mss_set_scan_variant(13) == 0 and L.mss_set_scan_variant(14) == -1 and L.mss_set_scan_variant(0) == 0
    for q, t, a, want in ((0, 0, -1, 0), (4, 4096, 2, 0), (2, 1024, 10, 0), (1, 0, 16, 0), (3, 0, -1, -1), (1, 1023, -1, -1),
                          (1, -2, -1, -1), (1, 0, 3, -1), (1, 0, 12, -1), (1, 0, 20, -1), (1, 0, -2, -1), (0, 0, -1, 0)):
        assert L.mss_set_pass1_geometry(q, t, a) == want, (q, t, a)
    assert L.mss_set_two_pass_chunk_bytes(12345) == 0 and L.mss_set_two_pass_chunk_bytes(0) == 0
    assert L.mss_static_scratch_bytes() == 32 << 20
    assert b"static" in L.mss_strerror(-5)
    sc = _Scoring(5, -4, -26)
    assert L.mss_map_reads_static(None, None, None, 7, None, 10, 100, sc, 3, None, None) == -1
    assert L.mss_map_reads_bounds_pssm(None, None, None, 7, None, 10, 100, None, 100, sc, 3, None, None, None) == -1


def test_product_does_not_import_the_oracle():
    import os
    import re
    root = os.path.dirname(os.path.abspath(mss.__file__))
    for dirpath, _, files in os.walk(root):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "maxss_oracle" not in text and "liboracle" not in text, f
