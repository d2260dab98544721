"""-m gpu: the CUDA MaxSS scan (through the C ABI) against the CPU oracle, element by element (bit-exact)."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tiny():
    cfg = gen.config(1)
    g, _ = cfg.genome()
    return cfg, g, cfg.reads(g)


def _cmp(got, want, ctx=""):
    bad = np.where((got != want).any(axis=(1, 2)))[0]
    assert bad.size == 0, f"{ctx}: {bad.size} reads differ, first {bad[0]}: got {got[bad[0]].tolist()} want {want[bad[0]].tolist()}"


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5, 6, 7])
def test_tiny_config_every_variant(oracle_mod, tiny, variant):
    from gpu_util import load_genome, map_reads
    cfg, g, r = tiny
    want = oracle_mod.map_reads_parallel(g, cfg.frag_len, cfg.overlap, r["reads"], r["lens"], strands=cfg.strands)
    G = load_genome(g, cfg.frag_len, cfg.overlap)
    got = map_reads(G, r["reads"], r["lens"], strands=cfg.strands, variant=variant)
    _cmp(got, want, f"tiny variant {variant}")


@pytest.mark.parametrize("strands", [1, 2, 3])
@pytest.mark.parametrize("F,V", [(1000, 0), (1000, -1), (1000, 17), (4096, -1), (700, 30), (300, -1), (5000, 50), (50_000, -1), (60_000, 0)])
def test_tiny_geometries(oracle_mod, tiny, F, V, strands):
    from gpu_util import load_genome, map_reads
    cfg, g, r = tiny
    reads, lens = r["reads"][:40], r["lens"][:40]
    want = oracle_mod.map_reads_parallel(g, F, V, reads, lens, strands=strands)
    G = load_genome(g, F, V)
    got = map_reads(G, reads, lens, strands=strands)
    _cmp(got, want, f"F={F} V={V} strands={strands}")
