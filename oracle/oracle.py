"""ctypes binding of oracle/maxss_oracle.c (plain C, gcc).  Test infrastructure only.

Two builds of the same source are kept: -O2 (`liboracle_O2.so`, the default) and -O3 -march=native
(`liboracle_O3.so`, used where many cells must be checked); tests require them to agree.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ProcessPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "maxss_oracle.c")
_LIBS: dict[str, C.CDLL] = {}
_FLAGS = {"O2": ["-O2"], "O3": ["-O3", "-march=native"]}


def _path(opt: str) -> str:
    return os.path.join(_HERE, f"liboracle_{opt}.so")


def build(force: bool = False) -> None:
    """Compile both oracle builds (gcc).  Building the checker is not using it."""
    for opt, flags in _FLAGS.items():
        out = _path(opt)
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
            tmp = out + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-std=c11", "-shared", "-fPIC", *flags, "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, out)


def _lib(opt: str = "O2") -> C.CDLL:
    if opt not in _LIBS:
        build()
        lib = C.CDLL(_path(opt))
        u8p, i32p, i64p, u32p, vp = (C.POINTER(C.c_uint8), C.POINTER(C.c_int32), C.POINTER(C.c_int64),
                                     C.POINTER(C.c_uint32), C.c_void_p)
        lib.oracle_map_reads.argtypes = [u8p, C.c_int64, C.c_int32, C.c_int32, u8p, C.c_int32, i32p, C.c_int32,
                                         C.c_int32, C.c_int32, C.c_int32, vp]
        lib.oracle_map_reads.restype = None
        lib.oracle_fragment_scores.argtypes = [u8p, C.c_int64, C.c_int32, C.c_int32, u8p, C.c_int32, C.c_int32,
                                               C.c_int32, C.c_int32, i32p, i32p]
        lib.oracle_fragment_scores.restype = None
        lib.oracle_diagonal_score.argtypes = [u8p, C.c_int64, C.c_int32, C.c_int32, C.c_int64, u8p, C.c_int32,
                                              C.c_int32, C.c_int32]
        lib.oracle_diagonal_score.restype = C.c_int32
        lib.oracle_nw_align.argtypes = [u8p, C.c_int64, C.c_int32, C.c_int32, u8p, C.c_int32, i32p, C.c_int32, vp,
                                        C.c_int32, C.c_int32, C.c_int32, C.c_int32, i32p, i64p, u32p, C.c_int32, i32p]
        lib.oracle_nw_align.restype = None
        lib.oracle_map_reads_fast.argtypes = lib.oracle_map_reads.argtypes
        lib.oracle_map_reads_fast.restype = None
        lib.oracle_pssm_from_phred.argtypes = [u8p, C.c_int64, C.c_int32, C.c_int32, C.c_int32, i32p, i32p]
        lib.oracle_pssm_from_phred.restype = None
        lib.oracle_map_reads_pssm.argtypes = [u8p, C.c_int64, C.c_int32, C.c_int32, u8p, C.c_int32, i32p, C.c_int32,
                                              i32p, i32p, C.c_int32, vp]
        lib.oracle_map_reads_pssm.restype = None
        lib.oracle_nw_align_pssm.argtypes = [u8p, C.c_int64, C.c_int32, C.c_int32, u8p, C.c_int32, i32p, C.c_int32, vp,
                                             i32p, i32p, C.c_int32, C.c_int32, i32p, i64p, u32p, C.c_int32, i32p]
        lib.oracle_nw_align_pssm.restype = None
        lib.oracle_mapq_filter.argtypes = [vp, C.c_int32, C.c_double, u8p, C.POINTER(C.c_double)]
        lib.oracle_mapq_filter.restype = None
        _LIBS[opt] = lib
    return _LIBS[opt]


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def map_reads(genome, frag_len, overlap, reads, lens, match=5, mismatch=-4, strands=3, opt="O2", fast=False):
    """-> int32 array (n_reads, 2, 4): [best|second][frag, diag, score, strand].  fast=True: MaxSSmap_fast."""
    genome = np.ascontiguousarray(genome, dtype=np.uint8)
    reads = np.ascontiguousarray(reads, dtype=np.uint8)
    if reads.ndim == 1:
        reads = reads[None, :]
    lens = np.ascontiguousarray(lens, dtype=np.int32).reshape(-1)
    n = reads.shape[0]
    out = np.zeros((n, 2, 4), dtype=np.int32)
    fn = _lib(opt).oracle_map_reads_fast if fast else _lib(opt).oracle_map_reads
    fn(_p(genome, C.c_uint8), genome.size, frag_len, overlap, _p(reads, C.c_uint8),
       reads.shape[1], _p(lens, C.c_int32), n, match, mismatch, strands, out.ctypes.data_as(C.c_void_p))
    return out


def _map_chunk(args):
    return map_reads(*args[:-2], opt=args[-2], fast=args[-1])


def map_reads_parallel(genome, frag_len, overlap, reads, lens, match=5, mismatch=-4, strands=3, opt="O3",
                       workers=None, fast=False):
    """Same result as map_reads; reads fanned out over host processes (each runs the single-threaded oracle)."""
    workers = workers or os.cpu_count() or 1
    n = reads.shape[0]
    if n == 0:
        return np.zeros((0, 2, 4), dtype=np.int32)
    workers = max(1, min(workers, n))
    build()
    bounds = np.linspace(0, n, workers + 1).astype(int)
    jobs = [(genome, frag_len, overlap, reads[a:b], lens[a:b], match, mismatch, strands, opt, fast)
            for a, b in zip(bounds[:-1], bounds[1:]) if b > a]
    if len(jobs) == 1:
        return _map_chunk(jobs[0])
    with ProcessPoolExecutor(max_workers=len(jobs)) as ex:
        parts = list(ex.map(_map_chunk, jobs))
    return np.concatenate(parts)


def fragment_scores(genome, frag_len, overlap, read, match=5, mismatch=-4, strand=0, opt="O2"):
    genome = np.ascontiguousarray(genome, dtype=np.uint8)
    read = np.ascontiguousarray(read, dtype=np.uint8)
    nfrag = -(-genome.size // frag_len)
    sc = np.zeros(nfrag, dtype=np.int32)
    dg = np.zeros(nfrag, dtype=np.int32)
    _lib(opt).oracle_fragment_scores(_p(genome, C.c_uint8), genome.size, frag_len, overlap, _p(read, C.c_uint8),
                                     read.size, match, mismatch, strand, _p(sc, C.c_int32), _p(dg, C.c_int32))
    return sc, dg


def diagonal_score(genome, frag_len, overlap, g, read, match=5, mismatch=-4, opt="O2"):
    genome = np.ascontiguousarray(genome, dtype=np.uint8)
    read = np.ascontiguousarray(read, dtype=np.uint8)
    return int(_lib(opt).oracle_diagonal_score(_p(genome, C.c_uint8), genome.size, frag_len, overlap, int(g),
                                               _p(read, C.c_uint8), read.size, match, mismatch))


def nw_align(genome, frag_len, overlap, reads, lens, top2, match=5, mismatch=-4, gap=-26, pad=30,
             cigar_stride=None, opt="O2"):
    """-> (score int32[n], ref_pos int64[n], cigar uint32[n, stride], n_cigar int32[n])."""
    genome = np.ascontiguousarray(genome, dtype=np.uint8)
    reads = np.ascontiguousarray(reads, dtype=np.uint8)
    lens = np.ascontiguousarray(lens, dtype=np.int32).reshape(-1)
    top2 = np.ascontiguousarray(top2, dtype=np.int32)
    n = reads.shape[0]
    stride = cigar_stride or (2 * reads.shape[1] + 1)
    score = np.zeros(n, dtype=np.int32)
    pos = np.zeros(n, dtype=np.int64)
    cig = np.zeros((n, stride), dtype=np.uint32)
    ncig = np.zeros(n, dtype=np.int32)
    _lib(opt).oracle_nw_align(_p(genome, C.c_uint8), genome.size, frag_len, overlap, _p(reads, C.c_uint8),
                              reads.shape[1], _p(lens, C.c_int32), n, top2.ctypes.data_as(C.c_void_p),
                              match, mismatch, gap, pad, _p(score, C.c_int32), _p(pos, C.c_int64),
                              _p(cig, C.c_uint32), stride, _p(ncig, C.c_int32))
    return score, pos, cig, ncig


def pssm_from_phred(qual, match=5, mismatch=-4, scale=16, opt="O2"):
    """phred qualities (uint8 array, any shape) -> (pmatch, pmismatch) int32 arrays of the same shape."""
    qual = np.ascontiguousarray(qual, dtype=np.uint8)
    pm = np.zeros(qual.shape, dtype=np.int32)
    pmm = np.zeros(qual.shape, dtype=np.int32)
    _lib(opt).oracle_pssm_from_phred(_p(qual, C.c_uint8), qual.size, match, mismatch, scale, _p(pm, C.c_int32),
                                     _p(pmm, C.c_int32))
    return pm, pmm


def map_reads_pssm(genome, frag_len, overlap, reads, lens, pmatch, pmismatch, strands=3, opt="O2"):
    """First phase with per-read position-specific (match, mismatch) scores; rows of pmatch/pmismatch align with reads."""
    genome = np.ascontiguousarray(genome, dtype=np.uint8)
    reads = np.ascontiguousarray(reads, dtype=np.uint8)
    if reads.ndim == 1:
        reads = reads[None, :]
    lens = np.ascontiguousarray(lens, dtype=np.int32).reshape(-1)
    pm = np.ascontiguousarray(pmatch, dtype=np.int32).reshape(reads.shape)
    pmm = np.ascontiguousarray(pmismatch, dtype=np.int32).reshape(reads.shape)
    n = reads.shape[0]
    out = np.zeros((n, 2, 4), dtype=np.int32)
    _lib(opt).oracle_map_reads_pssm(_p(genome, C.c_uint8), genome.size, frag_len, overlap, _p(reads, C.c_uint8),
                                    reads.shape[1], _p(lens, C.c_int32), n, _p(pm, C.c_int32), _p(pmm, C.c_int32),
                                    strands, out.ctypes.data_as(C.c_void_p))
    return out


def _map_pssm_chunk(args):
    return map_reads_pssm(*args[:-1], opt=args[-1])


def map_reads_pssm_parallel(genome, frag_len, overlap, reads, lens, pmatch, pmismatch, strands=3, opt="O3", workers=None):
    workers = workers or os.cpu_count() or 1
    n = reads.shape[0]
    if n == 0:
        return np.zeros((0, 2, 4), dtype=np.int32)
    workers = max(1, min(workers, n))
    build()
    bounds = np.linspace(0, n, workers + 1).astype(int)
    jobs = [(genome, frag_len, overlap, reads[a:b], lens[a:b], pmatch[a:b], pmismatch[a:b], strands, opt)
            for a, b in zip(bounds[:-1], bounds[1:]) if b > a]
    if len(jobs) == 1:
        return _map_pssm_chunk(jobs[0])
    with ProcessPoolExecutor(max_workers=len(jobs)) as ex:
        parts = list(ex.map(_map_pssm_chunk, jobs))
    return np.concatenate(parts)


def nw_align_pssm(genome, frag_len, overlap, reads, lens, top2, pmatch, pmismatch, gap, pad=30, cigar_stride=None, opt="O2"):
    """Second phase with position-specific scores; gap in the same fixed-point units."""
    genome = np.ascontiguousarray(genome, dtype=np.uint8)
    reads = np.ascontiguousarray(reads, dtype=np.uint8)
    lens = np.ascontiguousarray(lens, dtype=np.int32).reshape(-1)
    top2 = np.ascontiguousarray(top2, dtype=np.int32)
    pm = np.ascontiguousarray(pmatch, dtype=np.int32).reshape(reads.shape)
    pmm = np.ascontiguousarray(pmismatch, dtype=np.int32).reshape(reads.shape)
    n = reads.shape[0]
    stride = cigar_stride or (2 * reads.shape[1] + 1)
    score = np.zeros(n, dtype=np.int32)
    pos = np.zeros(n, dtype=np.int64)
    cig = np.zeros((n, stride), dtype=np.uint32)
    ncig = np.zeros(n, dtype=np.int32)
    _lib(opt).oracle_nw_align_pssm(_p(genome, C.c_uint8), genome.size, frag_len, overlap, _p(reads, C.c_uint8),
                                   reads.shape[1], _p(lens, C.c_int32), n, top2.ctypes.data_as(C.c_void_p),
                                   _p(pm, C.c_int32), _p(pmm, C.c_int32), gap, pad, _p(score, C.c_int32),
                                   _p(pos, C.c_int64), _p(cig, C.c_uint32), stride, _p(ncig, C.c_int32))
    return score, pos, cig, ncig


def mapq_filter(top2, threshold=-1.0, opt="O2"):
    """Repeat filter + MAPQ on top-2 records -> (mapped uint8[n], mapq float64[n]).
    threshold < 0: the paper's default "ratio below .9" decided on integers; >= 0: mapped iff MAPQ > threshold."""
    top2 = np.ascontiguousarray(top2, dtype=np.int32).reshape(-1, 2, 4)
    n = top2.shape[0]
    mapped = np.zeros(n, dtype=np.uint8)
    mapq = np.zeros(n, dtype=np.float64)
    _lib(opt).oracle_mapq_filter(top2.ctypes.data_as(C.c_void_p), n, float(threshold), _p(mapped, C.c_uint8),
                                 _p(mapq, C.c_double))
    return mapped, mapq
