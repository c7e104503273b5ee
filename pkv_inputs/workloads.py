"""Workload generators: lengths, block tables, random tensors.  No attention math here.

Citations: PAPER.md:104-112 (§3.7, page-table generation)
(§3.8, trace families), PAPER.md:89 (calibration seed 20260622, held-out seeds
20260623-20260627), BASELINE.json ``configs`` (the concrete shapes).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

PAD_PAGE = 0x7FFFFFFF  # value of block-table entries a row does not own

TUNE_SEED = 20260622                       # PAPER.md:89 calibration seed
REPORT_SEEDS = (20260623, 20260624, 20260625, 20260626, 20260627)  # PAPER.md:89 held-out


@dataclass
class Workload:
    """One synthetic decode trace: shapes, step-0 lengths, block table."""

    name: str
    B: int
    Hq: int
    Hkv: int
    d: int
    page_size: int
    seq_lens: np.ndarray          # int32 [B], lengths at step 0
    steps: int                    # decode steps in the trace; N_i += 1 per step
    block_table: np.ndarray       # int32 [B, max_pages]; PAD_PAGE where unused
    num_pages: int                # size of the physical page universe
    hole_frac: float
    seed: int
    extra: dict = field(default_factory=dict)

    @property
    def max_pages(self) -> int:
        return int(self.block_table.shape[1])

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    def seq_lens_at(self, step: int) -> np.ndarray:
        """Lengths after ``step`` decode steps (each active row grows by one token)."""
        assert 0 <= step <= self.steps
        return (self.seq_lens + np.int32(step)).astype(np.int32)

    def pool_shape(self):
        """Default K/V pool layout [num_pages, page_size, Hkv, d] (BASELINE.json north_star)."""
        return (self.num_pages, self.page_size, self.Hkv, self.d)

    def kv_bytes_per_token(self) -> int:
        """K + V bytes of one token: FP16 caches, or one byte per element with extra["kv_elem_bytes"] = 1
        (FP8 caches, reading A28)."""
        return 2 * self.Hkv * self.d * int(self.extra.get("kv_elem_bytes", 2))


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def make_page_table(reserved_lens: Sequence[int], page_size: int, hole_frac: float,
                    rng: np.random.Generator, max_pages: Optional[int] = None):
    """PAPER.md:106-112.  Row i owns L_i = ceil(reserved_i / P) logical pages; the physical
    universe has ceil(L / (1 - rho)) ids; a seeded permutation of the universe gives each row a
    consecutive slice, so logical order is kept and physical ids are scattered.

    Returns (block_table int32 [B, max_pages], num_pages)."""
    reserved = np.asarray(reserved_lens, dtype=np.int64)
    L_i = (reserved + page_size - 1) // page_size
    L = int(L_i.sum())
    assert 0.0 <= hole_frac < 1.0
    universe = max(1, int(np.ceil(L / (1.0 - hole_frac) - 1e-9)))
    perm = rng.permutation(universe)
    width = int(L_i.max()) if len(L_i) else 0
    if max_pages is not None:
        assert max_pages >= width
        width = max_pages
    width = max(width, 1)
    table = np.full((len(L_i), width), PAD_PAGE, dtype=np.int32)
    off = 0
    for i, n in enumerate(L_i):
        n = int(n)
        table[i, :n] = perm[off:off + n].astype(np.int32)
        off += n
    return table, universe


def make_workload(name: str, seq_lens: Sequence[int], *, steps: int, hole_frac: float, seed: int,
                  rng: Optional[np.random.Generator] = None, Hq: int = 32, Hkv: int = 8,
                  d: int = 128, page_size: int = 16, extra: Optional[dict] = None) -> Workload:
    """Build a Workload from given step-0 lengths.  ``rng`` continues a stream that already drew
    the lengths (draw order: lengths, permutation); if None a fresh PCG64(seed) is used."""
    if rng is None:
        rng = _rng(seed)
    lens = np.asarray(seq_lens, dtype=np.int32)
    table, universe = make_page_table(lens.astype(np.int64) + steps, page_size, hole_frac, rng)
    return Workload(name=name, B=len(lens), Hq=Hq, Hkv=Hkv, d=d, page_size=page_size,
                    seq_lens=lens, steps=steps, block_table=table, num_pages=universe,
                    hole_frac=hole_frac, seed=seed, extra=dict(extra or {}))


# ---------------------------------------------------------------- length distributions

def bimodal_lengths(rng: np.random.Generator, B: int) -> np.ndarray:
    """BASELINE.json config 3: with p=0.5 uniform[256,1024], else uniform[16384,32768] (inclusive)."""
    pick_short = rng.random(B) < 0.5
    short = rng.integers(256, 1024, size=B, endpoint=True)
    long_ = rng.integers(16384, 32768, size=B, endpoint=True)
    return np.where(pick_short, short, long_).astype(np.int32)


def zipf_lengths(rng: np.random.Generator, B: int, s: float = 1.2, unit: int = 512,
                 cap: int = 65536) -> np.ndarray:
    """BASELINE.json config 4: N = min(65536, 512*k), k ~ Zipf(s=1.2)."""
    k = rng.zipf(s, size=B).astype(np.int64)
    return np.minimum(cap, unit * k).astype(np.int32)


def uniform_lengths(rng: np.random.Generator, B: int, lo: int = 1024, hi: int = 65536) -> np.ndarray:
    """BASELINE.json config 5: N ~ uniform[1024, 65536] (inclusive)."""
    return rng.integers(lo, hi, size=B, endpoint=True).astype(np.int32)


# ---------------------------------------------------------------- the five configs

def config1(seed: int = TUNE_SEED) -> Workload:
    """B=1, N=256, 16 pages = a slice of a permutation of a 64-page pool (rho=0.75); no splitting."""
    return make_workload("config1_b1_n256", [256], steps=0, hole_frac=0.75, seed=seed)


def config2(seed: int = TUNE_SEED, seq_len: int = 32768) -> Workload:
    """B=1 long context, N=32768: 2048 pages permuted in a 4096-page pool (rho=0.5)."""
    return make_workload("config2_b1_n%d" % seq_len, [seq_len], steps=0, hole_frac=0.5, seed=seed)


def config3(seed: int = TUNE_SEED, B: int = 8, steps: int = 50, Hkv: int = 8) -> Workload:
    """B=8 bimodal ragged trace, 50 decode steps (+1 token per step), rho=0.5.
    Lengths are drawn once at step 0 and then grow (reading A17)."""
    rng = _rng(seed)
    lens = bimodal_lengths(rng, B)
    name = "config3_b%d_bimodal" % B + ("" if Hkv == 8 else "_hkv%d" % Hkv)
    return make_workload(name, lens, steps=steps, hole_frac=0.5, seed=seed, rng=rng, Hkv=Hkv)


def config4(seed: int = TUNE_SEED, B: int = 8, steps: int = 50) -> Workload:
    """B=8 Zipf-like trace: N = min(65536, 512*k), k ~ Zipf(1.2); 50 steps; rho=0.5."""
    rng = _rng(seed)
    lens = zipf_lengths(rng, B)
    return make_workload("config4_b%d_zipf" % B, lens, steps=steps, hole_frac=0.5, seed=seed, rng=rng)


def config4_b4(seed: int = TUNE_SEED, steps: int = 50) -> Workload:
    """The B=4 bimodal boundary variant of config 4 (config 3's length distribution)."""
    rng = _rng(seed)
    lens = bimodal_lengths(rng, 4)
    return make_workload("config4_b4_bimodal", lens, steps=steps, hole_frac=0.5, seed=seed, rng=rng)


def config5(seed: int = TUNE_SEED, B: int = 128, steps: int = 20, Hkv: int = 8) -> Workload:
    """B=128 uniform large batch, N ~ U[1024, 65536], 20 steps, shuffled pool without holes
    (rho=0): about 17 GB of K+V at Hkv=8, 8.7 GB at Hkv=4."""
    rng = _rng(seed)
    lens = uniform_lengths(rng, B)
    return make_workload("config5_b%d_uniform_hkv%d" % (B, Hkv), lens, steps=steps, hole_frac=0.0,
                         seed=seed, rng=rng, Hkv=Hkv)


# ---------------------------------------------------------------- the paper's other trace families

PROMPT_CYCLE = (8192, 16384, 32768, 65536)     # PAPER.md:116 "cycles prompt lengths through 8K, 16K, 32K, and 64K"


def trace_lengths(family: str, rng: np.random.Generator, B: int, decoded_max: int = 256) -> np.ndarray:
    """Step-0 context lengths of the trace families of PAPER.md:116 (sec. 3.8).  A request's current
    length is its prompt length plus the tokens it has decoded so far; the paper prints
    no decode-length distribution, so the tokens decoded before step 0 are drawn from
    U[0, decoded_max) per row (decoded_max = 0: every row sits exactly at its prompt length, the
    case where rows of one prompt class share an exact length bucket).
      bucketed     prompts cycle through 8K, 16K, 32K, 64K
      homogeneous  a common 32K prompt, independent decode lengths
      bimodal      "one long request for every three shorter": rows 3, 7, ... long U[16384, 32768],
                   the others U[256, 1024] (config 3 uses BASELINE.json's p = 0.5 draw instead)
      uniform      U[1024, 65536]          zipf  min(65536, 512 k), k ~ Zipf(1.2)"""
    if family == "bucketed":
        prompt = np.array([PROMPT_CYCLE[i % 4] for i in range(B)], dtype=np.int64)
    elif family == "homogeneous":
        prompt = np.full(B, 32768, dtype=np.int64)
    elif family == "bimodal":
        short = rng.integers(256, 1024, size=B, endpoint=True)
        long_ = rng.integers(16384, 32768, size=B, endpoint=True)
        prompt = np.where(np.arange(B) % 4 == 3, long_, short).astype(np.int64)
    elif family == "uniform":
        return uniform_lengths(rng, B)
    elif family == "zipf":
        return zipf_lengths(rng, B)
    else:
        raise ValueError(family)
    decoded = rng.integers(0, decoded_max, size=B) if decoded_max > 0 else np.zeros(B, dtype=np.int64)
    return (prompt + decoded).astype(np.int32)


def trace(family: str, seed: int = TUNE_SEED, B: int = 8, steps: int = 50, decoded_max: int = 256,
          hole_frac: float = 0.0) -> Workload:
    """One of the paper's serving traces (main serving traces use rho = 0)."""
    rng = _rng(seed)
    lens = trace_lengths(family, rng, B, decoded_max)
    return make_workload("trace_%s_b%d" % (family, B), lens, steps=steps, hole_frac=hole_frac, seed=seed, rng=rng,
                         extra={"family": family, "decoded_max": decoded_max})


# ---------------------------------------------------------------- random tensors

def fill_normal_f16(shape, seed: int) -> np.ndarray:
    """N(0,1) rounded to FP16 (numpy; used where no GPU is present and for small cases)."""
    rng = _rng(seed)
    out = np.empty(shape, dtype=np.float16)
    flat = out.reshape(-1)
    chunk = 1 << 22
    for s in range(0, flat.size, chunk):
        e = min(flat.size, s + chunk)
        flat[s:e] = rng.standard_normal(e - s, dtype=np.float32).astype(np.float16)
    return out


def fill_pool_torch(shape, seed: int, device):
    """N(0,1) FP16 tensor generated on ``device`` in bounded chunks (large pools: config 5 is
    8.7 GB per tensor).  The oracle is given the same bits by copying the pages it needs to host."""
    import torch

    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    out = torch.empty(shape, dtype=torch.float16, device=device)
    flat = out.view(-1)
    chunk = 1 << 26
    for s in range(0, flat.numel(), chunk):
        e = min(flat.numel(), s + chunk)
        flat[s:e] = torch.randn(e - s, generator=gen, device=device, dtype=torch.float32).to(torch.float16)
    return out
