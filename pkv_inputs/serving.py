"""Continuous-decode trace with arrival / finish dynamics -- inputs only, no attention arithmetic.

PAPER.md:93 (sec. 3.6): "Each request has an arrival time, prompt length, decode length, physical
page list, and dynamically growing current context length"; PAPER.md:116 for the prompt-length
families.  The paper prints no arrival process and no decode-length distribution; here (stated in
DESIGN.md sec. 4): arrivals are one request every `arrival_every` steps while a slot is free,
decode lengths are U[decode_lo, decode_hi], prompts come from `trace_lengths(family)`; a request
occupies one of `max_active` batch slots from its arrival until it has decoded its last token, then
the slot is empty (N = 0) until the next arrival takes it.  Pages: a request reserves
ceil((prompt + decode) / P) pages from a seeded free list (logical order kept,
physical ids scattered) and returns them when it finishes.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Iterator, List

import numpy as np

from .workloads import PAD_PAGE, trace_lengths


@dataclass
class ServingStep:
    step: int
    seq_lens: np.ndarray        # int32 [max_active]: current context length of every slot (0 = empty slot)
    block_table: np.ndarray     # int32 [max_active, max_pages] (a view that stays valid until the next step)
    started: List[int]          # slots taken by a request that arrived for this step
    finished: List[int]         # slots whose request decoded its last token in the previous step


class ServingTrace:
    def __init__(self, family: str, seed: int, requests: int = 32, max_active: int = 8, page_size: int = 16,
                 decode_lo: int = 8, decode_hi: int = 64, arrival_every: int = 2, prompt_div: int = 1):
        rng = np.random.Generator(np.random.PCG64(seed))
        self.P, self.B = page_size, max_active
        prompts = np.maximum(1, trace_lengths(family, rng, requests, decoded_max=0).astype(np.int64) // prompt_div)
        self.prompt = prompts
        self.decode = rng.integers(decode_lo, decode_hi, size=requests, endpoint=True).astype(np.int64)
        self.arrival_every = arrival_every
        need = (self.prompt + self.decode + page_size - 1) // page_size
        self.max_pages = int(need.max())
        # enough pages for the max_active largest requests at once, twice over (holes)
        self.num_pages = int(2 * np.sort(need)[-max_active:].sum())
        self.free = list(rng.permutation(self.num_pages).astype(np.int64))
        self.requests = requests

    def steps(self, max_steps: int = 10 ** 9) -> Iterator[ServingStep]:
        B, P = self.B, self.P
        table = np.full((B, self.max_pages), PAD_PAGE, dtype=np.int32)
        lens = np.zeros(B, dtype=np.int32)
        owner = [-1] * B                     # request in each slot
        left = np.zeros(B, dtype=np.int64)   # tokens the slot's request still has to decode
        pages: List[List[int]] = [[] for _ in range(B)]
        nxt, t, finished = 0, 0, []
        while t < max_steps and (nxt < self.requests or any(o >= 0 for o in owner)):
            started = []
            if t % self.arrival_every == 0 and nxt < self.requests:
                for s in range(B):
                    if owner[s] < 0:
                        n = int((self.prompt[nxt] + self.decode[nxt] + P - 1) // P)
                        if n > len(self.free):
                            break
                        pages[s] = [int(self.free.pop()) for _ in range(n)]
                        table[s, :] = PAD_PAGE
                        table[s, :n] = pages[s]
                        owner[s], lens[s], left[s] = nxt, int(self.prompt[nxt]), int(self.decode[nxt])
                        nxt += 1
                        started.append(s)
                        break
            # every active request decodes one token this step: its context includes that token
            for s in range(B):
                if owner[s] >= 0:
                    lens[s] += 1
                    left[s] -= 1
            yield ServingStep(t, lens.copy(), table, started, finished)
            finished = []
            for s in range(B):
                if owner[s] >= 0 and left[s] == 0:
                    self.free.extend(pages[s])
                    pages[s], owner[s], lens[s] = [], -1, 0
                    finished.append(s)
            t += 1
