"""Synthetic genomes and reads standing in for the paper's datasets.

The paper maps Stampy-simulated Illumina reads (divergence 0.1-0.3, gaps up to 30 bp in the
read or the genome, section 2.5, Table 2) to E. coli K12
(4.6 Mbp) and human chr1 (GRCh37.p13). Neither the genomes, the SRA runs nor Stampy are
available offline, so the five BASELINE.json configs are restated here as seeded recipes with
the same shapes (genome size, read length, divergence, indel lengths).
is the prose version of this file.

Base codes: A=0, C=1, G=2, T=3, N=4 (uint8).  Complement of a code c<4 is 3-c; N stays N.

Wire format (include/mss.h): base i lives in bits [2*(i%16), +2) of uint32 word i//16;
N mask: bit (i%32) of word i//32, 1 = N; the 2-bit code under an N is 0.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np

A, C, G, T, N = 0, 1, 2, 3, 4
S0 = 14032136  # base seed (the arXiv number); genome seed S0+10c, reads seed S0+10c+1

_ALPHA = np.frombuffer(b"ACGTN", dtype=np.uint8)


def decode(codes: np.ndarray) -> str:
    return _ALPHA[np.asarray(codes, dtype=np.uint8)].tobytes().decode()


def encode(s: str) -> np.ndarray:
    lut = np.full(256, N, dtype=np.uint8)
    for i, ch in enumerate("ACGT"):
        lut[ord(ch)] = i
        lut[ord(ch.lower())] = i
    return lut[np.frombuffer(s.encode(), dtype=np.uint8)]


def revcomp(codes: np.ndarray) -> np.ndarray:
    """Reverse-complement along the last axis (N stays N)."""
    c = np.asarray(codes, dtype=np.uint8)[..., ::-1]
    return np.where(c < 4, 3 - c, c).astype(np.uint8)


def sha256_of(*arrays: np.ndarray) -> str:
    h = hashlib.sha256()
    for a in arrays:
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


# ----------------------------------------------------------------------------- wire format

_PACK_CHUNK = 1 << 26      # bases per packing chunk (multiple of 32): bounds the temporaries for Gbp-sized genomes


def pack_2bit(codes: np.ndarray, n_words: int | None = None):
    """codes (uint8, 0..4) -> (packed uint32[ceil(n/16)], nmask uint32[ceil(n/32)])."""
    codes = np.asarray(codes, dtype=np.uint8).ravel()
    n = codes.size
    nw = (n + 15) // 16 if n_words is None else n_words
    nmw = (nw * 16 + 31) // 32
    packed = np.zeros(nw, dtype=np.uint32)
    nmask = np.zeros(nmw, dtype=np.uint32)
    shifts = (2 * np.arange(16, dtype=np.uint32))[None, :]
    mshifts = np.arange(32, dtype=np.uint32)[None, :]
    for c0 in range(0, max(n, 1), _PACK_CHUNK):
        part = codes[c0:c0 + _PACK_CHUNK]
        k = part.size
        kw, km = (k + 15) // 16, (k + 31) // 32
        pad = np.zeros(kw * 16, dtype=np.uint8)
        pad[:k] = np.where(part < 4, part, 0)
        packed[c0 // 16:c0 // 16 + kw] = np.bitwise_or.reduce(pad.reshape(kw, 16).astype(np.uint32) << shifts, axis=1)
        isn = np.zeros(km * 32, dtype=np.uint8)
        isn[:k] = part >= 4
        nmask[c0 // 32:c0 // 32 + km] = np.bitwise_or.reduce(isn.reshape(km, 32).astype(np.uint32) << mshifts, axis=1)
    return packed, nmask


def unpack_2bit(packed: np.ndarray, nmask: np.ndarray | None, n: int) -> np.ndarray:
    packed = np.asarray(packed, dtype=np.uint32).ravel()
    idx = np.arange(n)
    codes = ((packed[idx // 16] >> (2 * (idx % 16)).astype(np.uint32)) & 3).astype(np.uint8)
    if nmask is not None:
        nm = np.asarray(nmask, dtype=np.uint32).ravel()
        isn = (nm[idx // 32] >> (idx % 32).astype(np.uint32)) & 1
        codes = np.where(isn == 1, N, codes).astype(np.uint8)
    return codes


def pack_reads(reads: np.ndarray, lens: np.ndarray, stride_words: int | None = None):
    """reads (n, max_len) uint8 codes, lens (n,) -> (packed (n, stride) uint32, nmask (n, ceil(stride/2)) uint32).

    Bits beyond lens[r] are zero in both arrays."""
    reads = np.asarray(reads, dtype=np.uint8)
    n, ml = reads.shape
    sw = (ml + 15) // 16 if stride_words is None else stride_words
    assert sw * 16 >= ml
    buf = np.zeros((n, sw * 16), dtype=np.uint8)
    valid = np.arange(ml)[None, :] < np.asarray(lens)[:, None]
    buf[:, :ml] = np.where(valid & (reads < 4), reads, 0)
    q = buf.reshape(n, sw, 16).astype(np.uint32)
    packed = np.bitwise_or.reduce(q << (2 * np.arange(16, dtype=np.uint32))[None, None, :], axis=2).astype(np.uint32)
    nmw = (sw + 1) // 2
    isn = np.zeros((n, nmw * 32), dtype=np.uint8)
    isn[:, :ml] = valid & (reads >= 4)
    b = isn.reshape(n, nmw, 32).astype(np.uint32)
    nmask = np.bitwise_or.reduce(b << np.arange(32, dtype=np.uint32)[None, None, :], axis=2).astype(np.uint32)
    return np.ascontiguousarray(packed), np.ascontiguousarray(nmask)


# ----------------------------------------------------------------------------- genomes

def _place_nonoverlapping(rng, total_len, lengths, occupied):
    """Draw a start for each length so that [start, start+len) avoids `occupied` (bool array); marks them."""
    starts = []
    for L in lengths:
        for _ in range(1000):
            s = int(rng.integers(0, total_len - L + 1))
            if not occupied[s:s + L].any():
                break
        else:
            raise RuntimeError("could not place segment")
        occupied[s:s + L] = True
        starts.append(s)
    return starts


def make_genome(n: int, seed: int, gc: float = 0.5, dup_frac: float = 0.0, n_frac: float = 0.0,
                dup_len=(1_000, 50_000), dup_div=(0.01, 0.05), n_len=(10_000, 1_000_000)):
    """Random genome of n bases with P(G)=P(C)=gc/2, P(A)=P(T)=(1-gc)/2.

    Optional (config 4): planted segmental duplicates until dup_frac*n bases are copies, each copy of
    length U[dup_len] mutated at a per-copy substitution rate U[dup_div]; then N runs of length U[n_len]
    until n_frac*n bases are N.  Returns (codes uint8[n], info dict)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    p = np.array([(1 - gc) / 2, gc / 2, gc / 2, (1 - gc) / 2])
    cdf = np.cumsum(p)
    if n <= _PACK_CHUNK * 16:
        g = np.searchsorted(cdf, rng.random(n, dtype=np.float32), side="right").astype(np.uint8)
        g = np.minimum(g, 3).astype(np.uint8)
    else:           # Gbp-sized genomes (config 6): the same draw rule chunk by chunk, to bound the temporaries
        g = np.empty(n, dtype=np.uint8)
        for c0 in range(0, n, _PACK_CHUNK):
            k = min(_PACK_CHUNK, n - c0)
            g[c0:c0 + k] = np.minimum(np.searchsorted(cdf, rng.random(k, dtype=np.float32), side="right"), 3)
    info = {"dups": [], "n_runs": []}
    occupied = np.zeros(n, dtype=bool)
    if dup_frac > 0:
        target = int(dup_frac * n)
        done = 0
        while done < target:
            L = int(rng.integers(dup_len[0], dup_len[1] + 1))
            L = min(L, target - done) if target - done >= dup_len[0] else L
            src = int(rng.integers(0, n - L + 1))
            (dst,) = _place_nonoverlapping(rng, n, [L], occupied)
            rate = float(rng.uniform(dup_div[0], dup_div[1]))
            seg = g[src:src + L].copy()
            mut = rng.random(L) < rate
            seg[mut] = (seg[mut] + rng.integers(1, 4, size=int(mut.sum())).astype(np.uint8)) % 4
            g[dst:dst + L] = seg
            info["dups"].append((src, dst, L, rate))
            done += L
    if n_frac > 0:
        target = int(n_frac * n)
        done = 0
        while done < target:
            L = int(rng.integers(n_len[0], n_len[1] + 1))
            L = min(L, max(target - done, 1))
            (s,) = _place_nonoverlapping(rng, n, [L], occupied)
            g[s:s + L] = N
            info["n_runs"].append((s, L))
            done += L
    return g, info


# ----------------------------------------------------------------------------- reads

def make_reads(genome: np.ndarray, n_reads: int, m: int, seed: int, *,
               sub_rate=(0.10, 0.30), indel_counts=(0, 1, 2), indel_prob=None, indel_max: int = 30,
               both_strands: bool = True, avoid_n: bool = False):
    """Simulate n_reads reads of length m (vectorised over reads).

    Recipe: strand ~ Bernoulli(0.5) if both_strands else forward; per-read
    substitution rate p ~ U[sub_rate] (a scalar sub_rate fixes it); number of indels uniform over
    indel_counts (or, if indel_prob is given, one indel with that probability); each indel is an
    insertion (random bases in the read) or a deletion (genome bases skipped) with probability 1/2,
    length U{1..min(indel_max, m//3)}, placed at a uniform read offset inside its segment: the whole
    read [1, m) for one indel, the halves [1, m//2) and [m//2, m) for two (so they never overlap).
    Genome span = m - inserted + deleted bases, start uniform over the genome (re-drawn until the span
    holds no N if avoid_n).  Genome-derived bases are substituted w.p. p by a uniform *other* base.
    Minus-strand reads are reverse-complemented.

    Returns dict(reads uint8 (n, m), lens int32 (n,), start int64, strand uint8, span int32, p float32)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    G = genome.size
    n = n_reads
    strand = (rng.random(n) < 0.5).astype(np.uint8) if both_strands else np.zeros(n, dtype=np.uint8)
    if np.isscalar(sub_rate):
        p = np.full(n, float(sub_rate), dtype=np.float32)
    else:
        p = rng.uniform(sub_rate[0], sub_rate[1], size=n).astype(np.float32)
    if indel_prob is not None:
        k = (rng.random(n) < indel_prob).astype(np.int64)
    else:
        k = np.asarray(indel_counts)[rng.integers(0, len(indel_counts), size=n)].astype(np.int64)
    lmax = max(1, min(indel_max, m // 3))
    L = rng.integers(1, lmax + 1, size=(n, 2))
    is_ins = rng.random((n, 2)) < 0.5
    u = rng.random((n, 2))
    h = m // 2
    lo = np.empty((n, 2), dtype=np.int64)
    hi = np.empty((n, 2), dtype=np.int64)
    lo[:, 0] = 1
    hi[:, 0] = np.where(k == 2, h, m)
    lo[:, 1] = h
    hi[:, 1] = m
    active = np.stack([k >= 1, k >= 2], axis=1)
    # insertion occupies read positions [pos, pos+L) and must leave one genome base after it in the segment
    room = np.where(is_ins, hi - lo - L, hi - lo)
    room = np.maximum(room, 1)
    pos = lo + np.floor(u * room).astype(np.int64)
    L = np.where(active, L, 0)
    insL = np.where(is_ins, L, 0)
    delL = np.where(is_ins, 0, L)
    span = (m - insL.sum(1) + delL.sum(1)).astype(np.int64)

    # start positions
    if avoid_n:
        csum = np.concatenate([[0], np.cumsum(genome >= 4, dtype=np.int64)])
    start = np.empty(n, dtype=np.int64)
    todo = np.arange(n)
    while todo.size:
        s = np.floor(rng.random(todo.size) * (G - span[todo] + 1)).astype(np.int64)
        start[todo] = s
        if not avoid_n:
            break
        bad = (csum[s + span[todo]] - csum[s]) > 0
        todo = todo[bad]

    j = np.arange(m, dtype=np.int64)[None, :]
    off = np.broadcast_to(j, (n, m)).copy()
    inserted = np.zeros((n, m), dtype=bool)
    for e in range(2):
        pe = pos[:, e:e + 1]
        off -= np.clip(j - pe, 0, insL[:, e:e + 1])
        off += np.where(j >= pe, delL[:, e:e + 1], 0)
        inserted |= (j >= pe) & (j < pe + insL[:, e:e + 1])
    src = start[:, None] + off
    reads = genome[np.minimum(src, G - 1)].astype(np.uint8)
    sub = (rng.random((n, m), dtype=np.float32) < p[:, None]) & ~inserted & (reads < 4)
    shift = rng.integers(1, 4, size=(n, m)).astype(np.uint8)
    reads = np.where(sub, (reads + shift) % 4, reads).astype(np.uint8)
    rnd = rng.integers(0, 4, size=(n, m)).astype(np.uint8)
    reads = np.where(inserted, rnd, reads).astype(np.uint8)
    minus = strand == 1
    if minus.any():
        reads[minus] = revcomp(reads[minus])
    return dict(reads=np.ascontiguousarray(reads), lens=np.full(n, m, dtype=np.int32), start=start,
                strand=strand, span=span.astype(np.int32), p=p, n_indel=k.astype(np.int32))


def make_quals(n_reads: int, m: int, seed: int) -> np.ndarray:
    """Synthetic phred base qualities, uint8 (n_reads, m), in read order (stands in for the real MiSeq qualities the
    paper's simulated reads carry).  Illumina-like shape: a per-read level ~ N(36, 3), a decline of
    0..14 towards the 3' end (linear in the position, slope drawn per read), per-base noise N(0, 3), values clipped
    to [2, 41]; with probability 0.15 the last U{1..m//4} bases are a Q2 tail (the "B-tail" of old Illumina runs)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    level = rng.normal(36.0, 3.0, size=(n_reads, 1))
    drop = rng.uniform(0.0, 14.0, size=(n_reads, 1))
    pos = np.arange(m, dtype=np.float64)[None, :] / max(m - 1, 1)
    q = level - drop * pos + rng.normal(0.0, 3.0, size=(n_reads, m))
    q = np.clip(np.rint(q), 2, 41).astype(np.uint8)
    tail = rng.random(n_reads) < 0.15
    tl = rng.integers(1, max(2, m // 4 + 1), size=n_reads)
    cut = (np.arange(m)[None, :] >= (m - tl)[:, None]) & tail[:, None]
    q[cut] = 2
    return np.ascontiguousarray(q)


# ----------------------------------------------------------------------------- the five configs

@dataclass(frozen=True)
class Config:
    c: int
    name: str
    genome_len: int
    frag_len: int
    overlap: int           # -1 = the paper's look-ahead (read length - 1)
    strands: int           # 1 fwd, 2 rev, 3 both (include/mss.h)
    gc: float = 0.5
    dup_frac: float = 0.0
    n_frac: float = 0.0
    groups: tuple = field(default_factory=tuple)   # (n_reads, m, sub_rate) per group
    indel_prob: float | None = None
    both_strands: bool = True
    avoid_n: bool = False
    genome_of: int | None = None   # reuse the genome of another config (configs 3, 5 use config 2's)

    @property
    def genome_seed(self):
        return S0 + 10 * (self.genome_of or self.c)

    @property
    def reads_seed(self):
        return S0 + 10 * self.c + 1

    @property
    def n_reads(self):
        return sum(g[0] for g in self.groups)

    @property
    def max_len(self):
        return max(g[1] for g in self.groups)

    def genome(self):
        return make_genome(self.genome_len, self.genome_seed, gc=self.gc, dup_frac=self.dup_frac, n_frac=self.n_frac)

    def reads(self, genome: np.ndarray, limit: int | None = None):
        """All groups concatenated (padded to max_len with N, lens holds the true length).

        `limit` keeps only the first `limit` reads of every group (same bytes as the full draw's prefix
        is NOT guaranteed; a limited draw is its own seeded input)."""
        outs = []
        ml = self.max_len
        for gi, (n, m, rate) in enumerate(self.groups):
            nn = n if limit is None else min(n, limit)
            r = make_reads(genome, nn, m, self.reads_seed + 100 * gi, sub_rate=rate, indel_prob=self.indel_prob,
                           both_strands=self.both_strands, avoid_n=self.avoid_n)
            if m < ml:
                padded = np.full((nn, ml), N, dtype=np.uint8)
                padded[:, :m] = r["reads"]
                r["reads"] = padded
            outs.append(r)
        return {k: np.concatenate([o[k] for o in outs]) for k in outs[0]}

    def cells(self, n_reads=None, lens=None):
        nfrag = -(-self.genome_len // self.frag_len)
        ns = 2 if self.strands == 3 else 1
        if lens is None:
            tot = sum(g[0] * g[1] for g in self.groups)
        else:
            tot = int(np.sum(lens))
        return tot * nfrag * self.frag_len * ns


CONFIGS = {
    1: Config(1, "tiny", 50_000, 1000, 0, 1, groups=((200, 100, 0.10),), indel_prob=0.5, both_strands=False),
    2: Config(2, "ecoli", 4_600_000, 4096, -1, 3, groups=((100_000, 100, (0.10, 0.30)),)),
    3: Config(3, "lensweep", 4_600_000, 4096, -1, 3, genome_of=2,
              groups=tuple((20_000, m, r) for m in (36, 51, 100, 150, 250) for r in (0.10, 0.20, 0.30))),
    4: Config(4, "chr1", 249_000_000, 16384, -1, 3, gc=0.41, dup_frac=0.02, n_frac=0.10,
              groups=((10_000, 150, 0.20),), avoid_n=True),
    5: Config(5, "throughput", 4_600_000, 4096, -1, 3, genome_of=2, groups=((1_000_000, 100, 0.30),)),
    # next-4: whole-genome-sized workload in the shape of the paper's Table 8 (PAPER.md:460-474, :182:
    # 100k x 76 bp reads against the 2.4 Gbp horse genome, fragment length 4800): the packed genome (0.9 GB) no longer fits L2
    6: Config(6, "wholegenome", 2_400_000_000, 4800, -1, 3, gc=0.41, groups=((100_000, 76, 0.20),)),
}


def config(c: int) -> Config:
    return CONFIGS[c]
