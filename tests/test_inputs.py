"""CPU checks of the seeded input generators (no attention arithmetic in them): the serving trace with
arrival / finish dynamics and the trace families."""
import numpy as np

import pkv_inputs
from pkv_inputs import PAD_PAGE


def test_trace_families_shapes():
    for fam in ("bucketed", "homogeneous", "bimodal", "uniform", "zipf"):
        w = pkv_inputs.trace(fam, seed=7, B=8, steps=3)
        assert w.B == 8 and w.seq_lens.min() >= 1 and w.block_table.shape[0] == 8
        used = w.block_table[w.block_table != PAD_PAGE]
        assert len(np.unique(used)) == len(used) and used.max() < w.num_pages
    b = pkv_inputs.trace("bucketed", seed=7, B=8, steps=0, decoded_max=0).seq_lens
    assert list(b) == [8192, 16384, 32768, 65536] * 2
    bi = pkv_inputs.trace("bimodal", seed=7, B=8, steps=0, decoded_max=0).seq_lens
    assert all(bi[i] >= 16384 for i in (3, 7)) and all(bi[i] <= 1024 for i in (0, 1, 2, 4, 5, 6))
    assert np.array_equal(pkv_inputs.trace("zipf", seed=5).seq_lens, pkv_inputs.trace("zipf", seed=5).seq_lens)


def test_serving_trace_invariants():
    tr = pkv_inputs.ServingTrace("bimodal", seed=11, requests=20, max_active=4, decode_lo=3, decode_hi=9, prompt_div=16)
    prev, active_since, seen_started, total_tokens = None, {}, 0, 0
    for st in tr.steps():
        lens, table = st.seq_lens, st.block_table
        assert lens.shape == (4,) and table.shape == (4, tr.max_pages)
        for s in st.started:
            assert prev is None or prev[s] == 0 or s in st.finished            # only empty slots are taken
            seen_started += 1
        for s in range(4):
            if lens[s] > 0:
                need = -(-int(lens[s]) // 16)
                row = table[s, :need]
                assert np.all(row != PAD_PAGE) and row.max() < tr.num_pages
                if prev is not None and prev[s] > 0 and s not in st.started:
                    assert lens[s] == prev[s] + 1                               # one token per step
        rows = [table[s][table[s] != PAD_PAGE] for s in range(4) if lens[s] > 0]
        if rows:
            allp = np.concatenate(rows)
            assert len(np.unique(allp)) == len(allp)                            # no page shared by two active rows
        total_tokens += int((lens > 0).sum())
        prev = lens.copy()
        for s in st.finished:
            pass
    assert seen_started == 20 and total_tokens == int(tr.decode.sum())          # every request decodes all its tokens
    # same seed, same trace
    a = [s.seq_lens.tolist() for s in pkv_inputs.ServingTrace("uniform", seed=3, requests=6, max_active=2, prompt_div=64).steps()]
    b = [s.seq_lens.tolist() for s in pkv_inputs.ServingTrace("uniform", seed=3, requests=6, max_active=2, prompt_div=64).steps()]
    assert a == b and len(a) > 6
