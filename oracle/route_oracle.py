"""Length-bucket route and calibrated cost model -- pure-Python oracle.
TEST INFRASTRUCTURE, NOT THE PRODUCT (shares no code with the C++/CUDA library; only tests/,
__graft_entry__.smoke() and bench.py's CPU legs may import it).

Follows
  * PAPER.md:71 (sec. 3.4) "a ragged step with B active requests can become many PersistentKV
    launches, one per route length"; PAPER.md:93 (sec. 3.6) "PersistentKV groups active requests
    by route length unless the single-bucket or workqueue mode is enabled"; PAPER.md:106 (sec. 3.7)
    "rounded up to page granularity, or to an optional bucket length in bucketed experiments";
    PAPER.md:204-206 (sec. 4.5) exact length buckets vs coarse masked buckets;
  * PAPER.md:81-89 (sec. 3.5), the cost model
        T_r = KVBytes / beta * max(1, C_min / C_r) + L_r * lambda + MergeBytes_r / beta
    with its promotion margins (1.05x for supported B8 steps, 1.50x at the B4 boundary) and its two
    eligibility gates (the calibrated G = 4 mapping only; no step below 16K tokens).

Readings of what the paper leaves open:
  A22 a row's route length is its true length rounded up to `bucket_tokens` (1 = exact length
      buckets); rows of equal route length form one bucket; buckets are visited in ascending route
      length, rows inside a bucket in ascending row index; rows with N_i = 0 form no bucket.
  A23 every bucket is one rectangular (B_b, Hkv, S) launch with the row-local bounds of
      PAPER.md:63-67 plus, when S > 1, its own merge launch: launches/step = sum over buckets
      (Table 4: 8 distinct lengths -> 16.00 launches, 8.00 merge launches).
  A24 "C_r is estimated decode CTA work per SM" = tasks / #SMs, the quantity Table 4 prints
      (73.1 = 2048 / 28, 45.7 = 1280 / 28).
  A25 the 16K gate tests the step's longest row ("short-context steps below 16K tokens").
  A26 margins: a candidate replaces the baseline route only if T_baseline / T_candidate clears the
      margin of its batch regime: 1.05 for B >= 8 and for B = 1 (the paper's two supported regimes),
      1.50 -- or the explicit ablation flag -- for 2 <= B <= 7 ("the B4 boundary").

  A27 B200 re-fit, makespan form of the occupancy term (not in the paper).  With equal tasks the
      paper's stream term is  KVBytes/beta * C_min/C_r = (KVBytes/tasks) / beta_cta  with
      beta_cta = beta / (C_min * #SMs): the time ONE CTA needs for its share at the rate a lone CTA
      streams.  For unequal shares (ragged rows under a fixed split count) the largest share
      decides:  stream = max(KVBytes/beta, max_share/beta_cta).  The library's persistent CTA takes
      units of HG KV heads (HG = the largest of 8, 4, 2, 1 dividing Hkv that leaves units for >= 85 % of
      the SMs, else 1 -- the smallest valid group when nothing fills the machine): one wave (units <= #SMs):
      max_share = the largest unit's bytes; several waves: KVBytes/#SMs + the largest unit's bytes
      when units are handed out dynamically (HG = 8), waves x the largest unit's bytes when they are
      dealt round-robin (HG < 8: several warps share a head).  A CTA that reads HG heads' slices of every page instead of whole pages
      streams at beta * eta(HG), eta = 1 / 0.96 / 0.94 / 0.87 for HG = 8 / 4 / 2 / 1 (measured).

Pins (tests/test_route_oracle.py): Table 4's bucket row (16.00 / 73.1 / 4.06 / 8.00), the cost of
both Table-4 routes worked out by hand from the printed constants (beta = 331.2 GB/s, C_min = 4,
lambda = 8.19 us), closed forms of each term, gates and margins on constructed cases.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, List, Optional, Sequence, Tuple

from . import workqueue_oracle as wq

ROUTE_BUCKET = 2


# ---------------------------------------------------------------- length buckets (A22, A23)

def route_length(N: int, bucket_tokens: int) -> int:
    """A22: true length rounded up to the bucket granularity (1 = exact)."""
    return wq.ceil_div(int(N), bucket_tokens) * bucket_tokens


def group_buckets(seq_lens: Sequence[int], bucket_tokens: int) -> List[Tuple[int, List[int]]]:
    """[(route_length, [row, ...]), ...] in ascending route length; rows ascending inside."""
    groups: Dict[int, List[int]] = {}
    for i, N in enumerate(seq_lens):
        if int(N) > 0:
            groups.setdefault(route_length(int(N), bucket_tokens), []).append(i)
    return sorted(groups.items())


@dataclass
class RouteCounters:
    """Table 4's columns for one decode step of one route."""
    launches: int            # decode + merge launches
    merge_launches: int
    tasks: int               # CTAs of all decode launches (rect buckets: incl. empty intervals)
    empty_tasks: int
    useful_kv_bytes: int
    merge_bytes: int
    buckets: int


def _queue_merge_bytes(q: wq.WorkQueue, G: int, d: int) -> int:
    """A14: partial states exist (one pass, (d+2) FP32 words per task and query head) whenever some
    row of the launch has more than one slot -- with the separate and with the fused merge."""
    max_n = max((b - a for a, b in zip(q.split_offsets, q.split_offsets[1:])), default=0)
    return wq.merge_bytes(q.num_tasks, G, d) if max_n > 1 else 0


def bucket_route(seq_lens: Sequence[int], Hkv: int, G: int, d: int, policy: wq.Policy,
                 bucket_tokens: int) -> Tuple[RouteCounters, List[Tuple[List[int], wq.WorkQueue]]]:
    """A23: one launch pair per bucket; every bucket's queue is the oracle's queue of the bucket's
    rows alone under `policy` (rectangular grid unless the policy says otherwise)."""
    per_bucket = []
    c = RouteCounters(0, 0, 0, 0, wq.useful_kv_bytes(seq_lens, Hkv, d), 0, 0)
    for _, rows in group_buckets(seq_lens, bucket_tokens):
        q = wq.build_workqueue([int(seq_lens[i]) for i in rows], Hkv, policy)
        per_bucket.append((rows, q))
        c.launches += q.decode_launches + q.merge_launches
        c.merge_launches += q.merge_launches
        c.tasks += q.num_tasks
        c.empty_tasks += q.empty_ctas
        c.merge_bytes += _queue_merge_bytes(q, G, d)
        c.buckets += 1
    return c, per_bucket


def single_route(seq_lens: Sequence[int], Hkv: int, G: int, d: int, policy: wq.Policy) -> RouteCounters:
    """The same counters for one launch pair over the whole batch (workqueue or rectangular)."""
    q = wq.build_workqueue([int(n) for n in seq_lens], Hkv, policy)
    return RouteCounters(q.decode_launches + q.merge_launches, q.merge_launches, q.num_tasks, q.empty_ctas,
                         wq.useful_kv_bytes(seq_lens, Hkv, d), _queue_merge_bytes(q, G, d), 1 if q.num_tasks else 0)


# ---------------------------------------------------------------- cost model

@dataclass(frozen=True)
class CostConstants:
    beta_gbps: float      # measured streaming read bandwidth
    lambda_us: float      # calibrated launch overhead
    c_min: float          # minimum occupancy target, CTAs per SM
    num_sms: int


RTX3060 = CostConstants(beta_gbps=331.2, lambda_us=8.19, c_min=4.0, num_sms=28)


@dataclass
class CostTerms:
    stream_us: float
    launch_us: float
    merge_us: float
    cta_work_per_sm: float

    @property
    def total_us(self) -> float:
        return self.stream_us + self.launch_us + self.merge_us


def route_cost(kv_bytes: int, merge_bytes: int, launches: int, tasks: int, k: CostConstants) -> CostTerms:
    """PAPER.md:83, term by term.  C_r = tasks / #SMs (A24).  Bytes / (GB/s * 1e3) = microseconds."""
    c_r = tasks / float(k.num_sms)
    occupancy = max(1.0, k.c_min / c_r) if c_r > 0 else 1.0
    stream = kv_bytes / (k.beta_gbps * 1e3) * occupancy
    launch = launches * k.lambda_us
    merge = merge_bytes / (k.beta_gbps * 1e3)
    return CostTerms(stream, launch, merge, c_r)


def cost_of(c: RouteCounters, k: CostConstants) -> CostTerms:
    return route_cost(c.useful_kv_bytes, c.merge_bytes, c.launches, c.tasks, k)


MARGIN_B8 = 1.05
MARGIN_B4 = 1.50
GATE_MIN_TOKENS = 16384   # PAPER.md:87 "below 16K tokens"
GATE_G = 4                # PAPER.md:87 "the calibrated G = 4 KV-head-group mapping"


def eligible(seq_lens: Sequence[int], G: int) -> bool:
    """The two hard gates of PAPER.md:87 (A25)."""
    return G == GATE_G and max((int(n) for n in seq_lens), default=0) >= GATE_MIN_TOKENS


def promotion_margin(B: int) -> float:
    """A26."""
    return MARGIN_B8 if (B >= 8 or B == 1) else MARGIN_B4


def select_route(candidates: Dict[str, float], baseline: Optional[str], seq_lens: Sequence[int], G: int,
                 allow_b4: bool = False) -> str:
    """Route with the smallest estimate (ties: first in insertion order).  With a baseline route
    (the paper's FlashInfer path) the gates and the no-regression margin decide whether the best
    candidate replaces it; at the B4 boundary the ablation flag stands in for the margin
    ("a stricter 1.50x estimate or an explicit ablation flag")."""
    names = [n for n in candidates if n != baseline]
    best = min(names, key=lambda n: candidates[n]) if names else baseline
    if baseline is None:
        return best
    B = sum(1 for n in seq_lens if int(n) > 0)
    if not names or not eligible(seq_lens, G):
        return baseline
    margin = promotion_margin(B)
    if margin == MARGIN_B4 and allow_b4:
        return best
    return best if candidates[baseline] / candidates[best] >= margin else baseline


# ---------------------------------------------------------------- A27: makespan form (B200 re-fit)

def heads_per_cta(Hkv: int, row_slots: int, num_sms: int) -> int:
    best = 1
    for hg in (8, 4, 2, 1):
        if hg > Hkv or Hkv % hg:
            continue
        best = hg
        if row_slots * (Hkv // hg) * 20 >= num_sms * 17:
            return hg
    return best


def max_share_bytes(seq_lens: Sequence[int], Hkv: int, d: int, q: wq.WorkQueue, tile_tokens: int, num_sms: int) -> int:
    """A27: bytes of the busiest CTA.  A unit = the HG tasks (row, kvh .., split) of one token range."""
    row_slots = q.split_offsets[-1]
    if row_slots == 0:
        return 0
    hg = heads_per_cta(Hkv, row_slots, num_sms)
    tokens = max(min(te * tile_tokens, int(seq_lens[i])) - tb * tile_tokens for (i, _, _, tb, te) in q.tasks)
    unit = max(tokens, 0) * 2 * hg * d * 2
    units = row_slots * (Hkv // hg)
    kv = wq.useful_kv_bytes(seq_lens, Hkv, d)
    if units <= num_sms:
        return unit
    if hg == 8:                      # dynamic hand-out (G <= 8: one warp per head at HG = 8)
        return kv // num_sms + unit
    return wq.ceil_div(units, num_sms) * unit      # round-robin: the busiest CTA may draw only largest units


HEAD_SLICE_EFFICIENCY = {8: 1.0, 4: 0.96, 2: 0.94, 1: 0.87}    # A27, measured on B200 (config 2, decode kernel alone)


def stream_makespan_us(kv_bytes: int, share_bytes: int, k: CostConstants, hg: int = 8) -> float:
    beta_cta = k.beta_gbps / (k.c_min * k.num_sms)
    return max(kv_bytes / (k.beta_gbps * HEAD_SLICE_EFFICIENCY[hg] * 1e3), share_bytes / (beta_cta * 1e3))
