"""ctypes binding of include/mss.h.  Same names as the C entry points; argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
import re
from dataclasses import dataclass

HERE = os.path.dirname(os.path.abspath(__file__))
HEADER = os.path.join(HERE, "..", "include", "mss.h")
MSS_FWD, MSS_REV, MSS_BOTH = 1, 2, 3
MSS_OVERLAP_PAPER = -1

_lib = None


class MssError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: status {status} ({mss_strerror(status)})")


class _Scoring(C.Structure):
    _fields_ = [("match", C.c_int32), ("mismatch", C.c_int32), ("gap", C.c_int32)]


class _LaunchInfo(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("variant", "grid", "block", "smem_bytes", "reads_per_block", "tile_diagonals",
                                         "launches", "pass1_kernel")]


@dataclass(frozen=True)
class Scoring:
    """Paper defaults: match 5, mismatch -4, gap -26."""
    match: int = 5
    mismatch: int = -4
    gap: int = -26

    def c(self) -> _Scoring:
        return _Scoring(self.match, self.mismatch, self.gap)


def lib_path() -> str:
    return os.path.join(HERE, "libmss.so")


def declared_symbols() -> list[str]:
    """Every function include/mss.h declares (used by the CPU test that the library exports them all)."""
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mss_[a-z0-9_]+)\s*\(", text)))


def lib() -> C.CDLL:
    """Load libmss.so; fails loudly when the CUDA extension has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: build it with `python -m paper_1403_2136_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(path)
    vp, sz, i32, i64 = C.c_void_p, C.c_size_t, C.c_int32, C.c_int64
    L.mss_genome_workspace_bytes.argtypes = [i64, i32, i32]; L.mss_genome_workspace_bytes.restype = sz
    L.mss_genome_load.argtypes = [vp, vp, i64, i32, i32, vp, sz, vp, C.POINTER(vp)]; L.mss_genome_load.restype = C.c_int
    L.mss_genome_free.argtypes = [vp]; L.mss_genome_free.restype = C.c_int
    L.mss_genome_num_fragments.argtypes = [vp]; L.mss_genome_num_fragments.restype = i32
    L.mss_genome_num_bases.argtypes = [vp]; L.mss_genome_num_bases.restype = i64
    L.mss_map_workspace_bytes.argtypes = [vp, i32, i32, i32]; L.mss_map_workspace_bytes.restype = sz
    L.mss_map_reads.argtypes = [vp, vp, vp, i32, vp, i32, i32, _Scoring, i32, vp, sz, vp, vp]; L.mss_map_reads.restype = C.c_int
    L.mss_map_host_workspace_bytes.argtypes = [vp, i32, i32, i32, i32]; L.mss_map_host_workspace_bytes.restype = sz
    L.mss_map_reads_host.argtypes = [vp, vp, vp, i32, vp, i32, i32, _Scoring, i32, vp, sz, vp, vp]
    L.mss_map_reads_host.restype = C.c_int
    L.mss_map_align_host_workspace_bytes.argtypes = [vp, i32, i32, i32, i32, _Scoring, i32, i32]
    L.mss_map_align_host_workspace_bytes.restype = sz
    L.mss_map_align_host.argtypes = [vp, vp, vp, i32, vp, i32, i32, _Scoring, i32, i32, vp, sz, vp, vp, vp, vp, vp, i32, vp]
    L.mss_map_align_host.restype = C.c_int
    L.mss_nw_workspace_bytes.argtypes = [vp, i32, i32, _Scoring, i32]; L.mss_nw_workspace_bytes.restype = sz
    L.mss_nw_align.argtypes = [vp, vp, vp, i32, vp, i32, i32, vp, _Scoring, i32, vp, sz, vp, vp, vp, vp, i32, vp]
    L.mss_nw_align.restype = C.c_int
    L.mss_mapq_filter.argtypes = [vp, i32, C.c_double, vp, vp, vp]; L.mss_mapq_filter.restype = C.c_int
    L.mss_set_two_pass_chunk_bytes.argtypes = [C.c_int64]; L.mss_set_two_pass_chunk_bytes.restype = C.c_int
    L.mss_set_pass_timing.argtypes = [C.c_int]; L.mss_set_pass_timing.restype = C.c_int
    L.mss_set_pass1_geometry.argtypes = [i32, i32, i32]; L.mss_set_pass1_geometry.restype = C.c_int
    L.mss_get_pass_times.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_float)]; L.mss_get_pass_times.restype = C.c_int
    L.mss_map_reads_bounds.argtypes = [vp, vp, vp, i32, vp, i32, i32, _Scoring, i32, i32, vp, vp, C.POINTER(i32)]
    L.mss_map_reads_bounds.restype = C.c_int
    L.mss_map_reads_bounds_pssm.argtypes = [vp, vp, vp, i32, vp, i32, i32, vp, i32, _Scoring, i32, vp, vp, C.POINTER(i32)]
    L.mss_map_reads_bounds_pssm.restype = C.c_int
    L.mss_map_reads_fast.argtypes = L.mss_map_reads.argtypes; L.mss_map_reads_fast.restype = C.c_int
    L.mss_pssm_build.argtypes = [vp, i32, vp, i32, _Scoring, i32, vp, vp, i32]; L.mss_pssm_build.restype = C.c_int
    L.mss_map_reads_pssm.argtypes = [vp, vp, vp, i32, vp, i32, i32, vp, i32, _Scoring, i32, vp, sz, vp, vp]
    L.mss_map_reads_pssm.restype = C.c_int
    L.mss_nw_align_pssm.argtypes = [vp, vp, vp, i32, vp, i32, i32, vp, vp, i32, _Scoring, i32, vp, sz, vp, vp, vp, vp, i32, vp]
    L.mss_nw_align_pssm.restype = C.c_int
    L.mss_static_scratch_bytes.argtypes = []; L.mss_static_scratch_bytes.restype = C.c_size_t
    L.mss_static_init.argtypes = []; L.mss_static_init.restype = C.c_int
    L.mss_map_reads_static.argtypes = [vp, vp, vp, i32, vp, i32, i32, _Scoring, i32, vp, vp]; L.mss_map_reads_static.restype = C.c_int
    L.mss_strerror.argtypes = [C.c_int]; L.mss_strerror.restype = C.c_char_p
    L.mss_last_cuda_error.argtypes = []; L.mss_last_cuda_error.restype = C.c_int
    L.mss_version.argtypes = []; L.mss_version.restype = C.c_int
    L.mss_set_scan_variant.argtypes = [C.c_int]; L.mss_set_scan_variant.restype = C.c_int
    L.mss_get_last_launch.argtypes = [C.POINTER(_LaunchInfo)]; L.mss_get_last_launch.restype = C.c_int
    L.mss_probe_dpx_peak.argtypes = [i32, vp, C.POINTER(C.c_double), C.POINTER(C.c_float)]; L.mss_probe_dpx_peak.restype = C.c_int
    L.mss_probe_pipe.argtypes = [i32, i32, vp, C.POINTER(C.c_double)]; L.mss_probe_pipe.restype = C.c_int
    _lib = L
    return L


def mss_strerror(status: int) -> str:
    try:
        return lib().mss_strerror(status).decode()
    except Exception:  # library missing: still give a readable message
        return "libmss.so not loaded"


def _check(status: int, what: str):
    if status != 0:
        extra = ""
        if status == -4:
            extra = f" [cudaError {lib().mss_last_cuda_error()}]"
        raise MssError(status, what + extra)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1403_2136_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _stream(stream=None):
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Genome:
    """Owner of the device buffers behind an mss_genome_t handle (packed genome, N mask, derived workspace)."""

    def __init__(self, handle, packed, nmask, workspace, n_bases, frag_len, overlap):
        self.handle, self.packed, self.nmask, self.workspace = handle, packed, nmask, workspace
        self.n_bases, self.frag_len, self.overlap = n_bases, frag_len, overlap
        self.n_frag = lib().mss_genome_num_fragments(handle)
        self._scratch = {}

    def scratch(self, nbytes: int, key: str = "ws"):
        """A cached device byte buffer of at least nbytes (torch memory; the library allocates none)."""
        torch = _torch()
        buf = self._scratch.get(key)
        if buf is None or buf.numel() < nbytes:
            buf = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=self.packed.device)
            self._scratch[key] = buf
        return buf

    def close(self):
        if self.handle:
            lib().mss_genome_free(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def mss_genome_load(d_packed, d_nmask, n_bases: int, frag_len: int, overlap: int = MSS_OVERLAP_PAPER, stream=None) -> Genome:
    """d_packed / d_nmask: CUDA int32/uint32 tensors in the wire format of include/mss.h (d_nmask may be None)."""
    torch = _torch()
    L = lib()
    nbytes = L.mss_genome_workspace_bytes(n_bases, frag_len, overlap)
    if nbytes == 0:
        raise MssError(-1, "mss_genome_workspace_bytes")
    ws = torch.empty(nbytes, dtype=torch.uint8, device=d_packed.device)
    h = C.c_void_p()
    _check(L.mss_genome_load(_ptr(d_packed), _ptr(d_nmask), n_bases, frag_len, overlap, _ptr(ws), nbytes, _stream(stream),
                             C.byref(h)), "mss_genome_load")
    return Genome(h, d_packed, d_nmask, ws, n_bases, frag_len, overlap)


def mss_map_reads(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, scoring: Scoring = Scoring(),
                  strands: int = MSS_BOTH, stream=None, out=None):
    """-> CUDA int32 tensor (n_reads, 2, 4): [best|second][frag, diag, score, strand] (mss_top2_t records)."""
    torch = _torch()
    L = lib()
    n = int(d_lens.numel())
    stride = int(d_reads.shape[1]) if d_reads.dim() == 2 else int(d_reads.numel() // max(n, 1))
    if out is None:
        out = torch.empty((n, 2, 4), dtype=torch.int32, device=d_lens.device)
    nbytes = L.mss_map_workspace_bytes(g.handle, n, max_len, strands)
    if nbytes == 0:
        raise MssError(-1, "mss_map_workspace_bytes")
    ws = g.scratch(nbytes, "map")
    _check(L.mss_map_reads(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), stride, _ptr(d_lens), n, max_len, scoring.c(),
                           strands, _ptr(ws), ws.numel(), _stream(stream), _ptr(out)), "mss_map_reads")
    return out


def mss_map_reads_fast(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, scoring: Scoring = Scoring(),
                       strands: int = MSS_BOTH, stream=None, out=None):
    """MaxSSmap_fast: as mss_map_reads, scoring every other read nucleotide."""
    torch = _torch()
    L = lib()
    n = int(d_lens.numel())
    stride = int(d_reads.shape[1]) if d_reads.dim() == 2 else int(d_reads.numel() // max(n, 1))
    if out is None:
        out = torch.empty((n, 2, 4), dtype=torch.int32, device=d_lens.device)
    nbytes = L.mss_map_workspace_bytes(g.handle, n, max_len, strands)
    if nbytes == 0:
        raise MssError(-1, "mss_map_workspace_bytes")
    ws = g.scratch(nbytes, "map")
    _check(L.mss_map_reads_fast(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), stride, _ptr(d_lens), n, max_len, scoring.c(),
                                strands, _ptr(ws), ws.numel(), _stream(stream), _ptr(out)), "mss_map_reads_fast")
    return out


def mss_map_reads_bounds(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, scoring: Scoring = Scoring(),
                         strands: int = MSS_BOTH, every_other: bool = False, stream=None):
    """Pass 1 of the two-pass scan: -> (CUDA int16 tensor (n_reads, n_strands, n_frag) holding uint16 bounds, delta)."""
    torch = _torch()
    n = int(d_lens.numel())
    stride = int(d_reads.shape[1])
    ns = 2 if strands == MSS_BOTH else 1
    out = torch.empty((n, ns, g.n_frag), dtype=torch.int16, device=d_lens.device)
    delta = C.c_int32()
    _check(lib().mss_map_reads_bounds(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), stride, _ptr(d_lens), n, max_len,
                                      scoring.c(), strands, 1 if every_other else 0, _stream(stream), _ptr(out),
                                      C.byref(delta)), "mss_map_reads_bounds")
    return out, delta.value


def mss_map_reads_bounds_pssm(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, d_pssm, bound: Scoring,
                              strands: int = MSS_BOTH, stream=None):
    """Pass 1 of the two-pass scan under base-quality scoring: -> (uint16 bounds as an int16 tensor, delta)."""
    torch = _torch()
    n = int(d_lens.numel())
    ns = 2 if strands == MSS_BOTH else 1
    out = torch.empty((n, ns, g.n_frag), dtype=torch.int16, device=d_lens.device)
    delta = C.c_int32()
    _check(lib().mss_map_reads_bounds_pssm(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), int(d_reads.shape[1]), _ptr(d_lens), n,
                                           max_len, _ptr(d_pssm), int(d_pssm.shape[1]), bound.c(), strands, _stream(stream),
                                           _ptr(out), C.byref(delta)), "mss_map_reads_bounds_pssm")
    return out, delta.value


def pssm_bound(scoring: Scoring, scale: int) -> Scoring:
    """The range of a table built by mss_pssm_build(scoring, scale): pmatch <= scale*match, and pmismatch =
    round(scale*mismatch*x/3) with x <= 1 >= -ceil(scale*|mismatch|/3); the gap is scale*gap.  The tight
    mismatch bound matters: the slack of the two-pass scan's bounds is min(PM, -PMM) - PMM."""
    return Scoring(scale * scoring.match, -((scale * -scoring.mismatch + 2) // 3), scale * scoring.gap)


def mss_pssm_build(d_qual, d_lens, scoring: Scoring = Scoring(), scale: int = 16, pssm_stride: int | None = None, stream=None):
    """phred qualities (CUDA uint8 tensor (n, qual_stride)) -> CUDA int32 tensor (n, pssm_stride) of packed
    (int16 pmatch | int16 pmismatch << 16) entries."""
    torch = _torch()
    n = int(d_lens.numel())
    qs = int(d_qual.shape[1])
    ps = pssm_stride or qs
    out = torch.empty((n, ps), dtype=torch.int32, device=d_lens.device)
    _check(lib().mss_pssm_build(_ptr(d_qual), qs, _ptr(d_lens), n, scoring.c(), int(scale), _stream(stream), _ptr(out), ps),
           "mss_pssm_build")
    return out


def mss_map_reads_pssm(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, d_pssm, bound: Scoring,
                       strands: int = MSS_BOTH, stream=None, out=None):
    """mss_map_reads with per-read position-specific scores (d_pssm from mss_pssm_build; bound = pssm_bound(...))."""
    torch = _torch()
    L = lib()
    n = int(d_lens.numel())
    stride = int(d_reads.shape[1])
    if out is None:
        out = torch.empty((n, 2, 4), dtype=torch.int32, device=d_lens.device)
    nbytes = L.mss_map_workspace_bytes(g.handle, n, max_len, strands)
    if nbytes == 0:
        raise MssError(-1, "mss_map_workspace_bytes")
    ws = g.scratch(nbytes, "map")
    _check(L.mss_map_reads_pssm(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), stride, _ptr(d_lens), n, max_len, _ptr(d_pssm),
                                int(d_pssm.shape[1]), bound.c(), strands, _ptr(ws), ws.numel(), _stream(stream), _ptr(out)),
           "mss_map_reads_pssm")
    return out


def mss_nw_align_pssm(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, d_hits, d_pssm, bound: Scoring, pad: int = 30,
                      cigar_stride: int | None = None, stream=None):
    """mss_nw_align with per-read position-specific scores; bound.gap = the gap cost in the table's units."""
    torch = _torch()
    L = lib()
    n = int(d_lens.numel())
    stride = int(d_reads.shape[1])
    cs = cigar_stride or (2 * max_len + 1)
    dev = d_lens.device
    score = torch.empty(n, dtype=torch.int32, device=dev)
    pos = torch.empty(n, dtype=torch.int64, device=dev)
    cigar = torch.zeros((n, cs), dtype=torch.int32, device=dev)
    ncig = torch.empty(n, dtype=torch.int32, device=dev)
    nbytes = L.mss_nw_workspace_bytes(g.handle, n, max_len, bound.c(), pad)
    if nbytes == 0:
        raise MssError(-1, "mss_nw_workspace_bytes")
    ws = g.scratch(nbytes, "nw")
    _check(L.mss_nw_align_pssm(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), stride, _ptr(d_lens), n, max_len, _ptr(d_hits),
                               _ptr(d_pssm), int(d_pssm.shape[1]), bound.c(), pad, _ptr(ws), ws.numel(), _stream(stream),
                               _ptr(score), _ptr(pos), _ptr(cigar), cs, _ptr(ncig)), "mss_nw_align_pssm")
    return score, pos, cigar, ncig


def mss_map_reads_host(g: Genome, h_reads, h_reads_nmask, h_lens, max_len: int, scoring: Scoring = Scoring(),
                       strands: int = MSS_BOTH, stream=None, out=None):
    """Host (pinned) tensors in, host tensor out; copies are inside the call (the e2e path of bench.py)."""
    torch = _torch()
    L = lib()
    n = int(h_lens.numel())
    stride = int(h_reads.shape[1])
    if out is None:
        out = torch.empty((n, 2, 4), dtype=torch.int32).pin_memory()
    nbytes = L.mss_map_host_workspace_bytes(g.handle, n, max_len, stride, strands)
    if nbytes == 0:
        raise MssError(-1, "mss_map_host_workspace_bytes")
    ws = g.scratch(nbytes, "maphost")
    _check(L.mss_map_reads_host(g.handle, _ptr(h_reads), _ptr(h_reads_nmask), stride, _ptr(h_lens), n, max_len, scoring.c(),
                                strands, _ptr(ws), ws.numel(), _stream(stream), _ptr(out)), "mss_map_reads_host")
    return out


def mss_map_align_host(g: Genome, h_reads, h_reads_nmask, h_lens, max_len: int, scoring: Scoring = Scoring(),
                       strands: int = MSS_BOTH, pad: int = 30, cigar_stride: int = 16, stream=None, out=None):
    """Both phases, host (pinned) tensors in and out.  -> dict(top2, score, ref_pos, cigar, n_cigar) of host tensors."""
    torch = _torch()
    L = lib()
    n = int(h_lens.numel())
    stride = int(h_reads.shape[1])
    if out is None:
        out = dict(top2=torch.empty((n, 2, 4), dtype=torch.int32).pin_memory(),
                   score=torch.empty(n, dtype=torch.int32).pin_memory(),
                   ref_pos=torch.empty(n, dtype=torch.int64).pin_memory(),
                   cigar=torch.empty((n, cigar_stride), dtype=torch.int32).pin_memory(),
                   n_cigar=torch.empty(n, dtype=torch.int32).pin_memory())
    nbytes = L.mss_map_align_host_workspace_bytes(g.handle, n, max_len, stride, strands, scoring.c(), pad, cigar_stride)
    if nbytes == 0:
        raise MssError(-1, "mss_map_align_host_workspace_bytes")
    ws = g.scratch(nbytes, "e2e")
    _check(L.mss_map_align_host(g.handle, _ptr(h_reads), _ptr(h_reads_nmask), stride, _ptr(h_lens), n, max_len, scoring.c(),
                                strands, pad, _ptr(ws), ws.numel(), _stream(stream), _ptr(out["top2"]), _ptr(out["score"]),
                                _ptr(out["ref_pos"]), _ptr(out["cigar"]), cigar_stride, _ptr(out["n_cigar"])),
           "mss_map_align_host")
    return out


def mss_nw_align(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, d_hits, scoring: Scoring = Scoring(), pad: int = 30,
                 cigar_stride: int | None = None, stream=None):
    """-> (score int32[n], ref_pos int64[n], cigar int32[n, cigar_stride] (len<<4|op), n_cigar int32[n]) on the device."""
    torch = _torch()
    L = lib()
    n = int(d_lens.numel())
    stride = int(d_reads.shape[1])
    cs = cigar_stride or (2 * max_len + 1)
    dev = d_lens.device
    score = torch.empty(n, dtype=torch.int32, device=dev)
    pos = torch.empty(n, dtype=torch.int64, device=dev)
    cigar = torch.zeros((n, cs), dtype=torch.int32, device=dev)
    ncig = torch.empty(n, dtype=torch.int32, device=dev)
    nbytes = L.mss_nw_workspace_bytes(g.handle, n, max_len, scoring.c(), pad)
    if nbytes == 0:
        raise MssError(-1, "mss_nw_workspace_bytes")
    ws = g.scratch(nbytes, "nw")
    _check(L.mss_nw_align(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), stride, _ptr(d_lens), n, max_len, _ptr(d_hits),
                          scoring.c(), pad, _ptr(ws), ws.numel(), _stream(stream), _ptr(score), _ptr(pos), _ptr(cigar), cs,
                          _ptr(ncig)), "mss_nw_align")
    return score, pos, cigar, ncig


def mss_mapq_filter(d_hits, mapq_threshold: float = -1.0, stream=None):
    """-> (mapped uint8[n], mapq float32[n]); mapq_threshold < 0 (default) = the paper's "ratio below .9" on integers
    (PAPER.md:57); >= 0 = mapped iff MAPQ > threshold."""
    torch = _torch()
    n = int(d_hits.shape[0])
    mapped = torch.empty(n, dtype=torch.uint8, device=d_hits.device)
    mapq = torch.empty(n, dtype=torch.float32, device=d_hits.device)
    _check(lib().mss_mapq_filter(_ptr(d_hits), n, float(mapq_threshold), _stream(stream), _ptr(mapped), _ptr(mapq)),
           "mss_mapq_filter")
    return mapped, mapq


MSS_ERR_STATIC_LIMIT = -5


def mss_static_scratch_bytes() -> int:
    return int(lib().mss_static_scratch_bytes())


def mss_static_init() -> None:
    """Resolve the static scratch array on the current device (once per device; before graph capture)."""
    _check(lib().mss_static_init(), "mss_static_init")


def mss_map_reads_static(g: Genome, d_reads, d_reads_nmask, d_lens, max_len: int, out, scoring: Scoring = Scoring(),
                         strands: int = MSS_BOTH, stream=None):
    """mss_map_reads into the caller's `out` (CUDA int32 tensor (n, 2, 4)) with the scan's scratch in the library's static
    device array: the call allocates nothing.  Raises MssError(status MSS_ERR_STATIC_LIMIT) when the batch needs more scratch
    than mss_static_scratch_bytes()."""
    n = int(d_lens.numel())
    _check(lib().mss_map_reads_static(g.handle, _ptr(d_reads), _ptr(d_reads_nmask), int(d_reads.shape[1]), _ptr(d_lens), n,
                                      int(max_len), scoring.c(), strands, _stream(stream), _ptr(out)), "mss_map_reads_static")
    return out


def mss_set_two_pass_chunk_bytes(nbytes: int) -> None:
    _check(lib().mss_set_two_pass_chunk_bytes(int(nbytes)), "mss_set_two_pass_chunk_bytes")


def mss_set_pass1_geometry(query_sets: int = 0, tile_window_starts: int = 0, arithmetic: int = -1) -> None:
    _check(lib().mss_set_pass1_geometry(int(query_sets), int(tile_window_starts), int(arithmetic)), "mss_set_pass1_geometry")


def mss_set_pass_timing(on: bool) -> None:
    _check(lib().mss_set_pass_timing(1 if on else 0), "mss_set_pass_timing")


def mss_get_pass_times():
    """-> (pass 1 ms, pass 2 ms) of the latest two-pass scan on this thread (waits for it)."""
    a, b = C.c_float(), C.c_float()
    _check(lib().mss_get_pass_times(C.byref(a), C.byref(b)), "mss_get_pass_times")
    return a.value, b.value


def mss_set_scan_variant(variant: int) -> None:
    _check(lib().mss_set_scan_variant(int(variant)), "mss_set_scan_variant")


def mss_get_last_launch() -> dict:
    info = _LaunchInfo()
    _check(lib().mss_get_last_launch(C.byref(info)), "mss_get_last_launch")
    return {n: getattr(info, n) for n, _ in _LaunchInfo._fields_}


def mss_probe_dpx_peak(iters: int = 4096, stream=None):
    """-> (thread-instructions per second of the 2:1 VIADDMNMX/VIMNMX3 mix, elapsed ms)."""
    rate, ms = C.c_double(), C.c_float()
    _check(lib().mss_probe_dpx_peak(iters, _stream(stream), C.byref(rate), C.byref(ms)), "mss_probe_dpx_peak")
    return rate.value, ms.value


PROBE_NAMES = ["VIADDMNMX.S16x2.RELU", "VIMNMX3.S16x2", "DPX mix 2:1 (relu : max3)", "LDS.32 (conflict-free)",
               "scan mix: LDS.32 + VIADDMNMX /2 cells + VIMNMX3 /4 cells  [cells]"]


def mss_probe_pipe(which: int, iters: int = 2000, stream=None) -> float:
    """-> thread-instructions (mix rows: cells) per clock per SM of probe `which` (see include/mss.h)."""
    v = C.c_double()
    _check(lib().mss_probe_pipe(int(which), int(iters), _stream(stream), C.byref(v)), "mss_probe_pipe")
    return v.value
