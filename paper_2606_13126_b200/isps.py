"""Engine-less replay of the paper's request procedures on top of the host-side block pool (csrc/hasher.cu):

* ``compose`` - the user-side contract of PAPER.md:79-81, :123-128: pad to block boundaries, SSEP as the first token of every
  document, PDEP in front of the task suffix.
* ``isps_order`` - Interleaved Span-Prefill Scheduling: per mini-batch, one prefill-only request per
  distinct span (duplicates evicted), then the final prompts; FIFO order guarantees that the span prefills run first.
* ``replay`` - admit the ordered requests into a ``binding.Pool`` and count what would have to be prefilled.

Integer / token bookkeeping only: no attention arithmetic here.  The GPU work of a request is exactly the library calls with
the tables ``Pool.admit`` returns (tests/test_gpu_parity.py::test_pool_derived_tables_end_to_end).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np


def pad_to_block(tokens: np.ndarray, block_size: int, pad_id: int) -> np.ndarray:
    tokens = np.asarray(tokens, np.int32)
    n = -len(tokens) % block_size
    return np.concatenate([tokens, np.full(n, pad_id, np.int32)]) if n else tokens


def span_request(doc: np.ndarray, block_size: int, ssep: int, pad_id: int) -> np.ndarray:
    """[SSEP, doc...] padded to a block boundary: the unit that is prefilled once and cache-hits anywhere."""
    return pad_to_block(np.concatenate([[ssep], np.asarray(doc, np.int32)]), block_size, pad_id)


def compose(system: np.ndarray, docs: Sequence[np.ndarray], task: np.ndarray, block_size: int, ssep: int, pdep: int,
            pad_id: int, link_tokens: int = 0) -> np.ndarray:
    """Final prompt [system][SSEP,doc1]...[PDEP,task].  ``link_tokens`` > 0 is EPIC / LegoLink (:149): the
    first ``link_tokens`` tokens (a block multiple) of every document come BEFORE its SSEP, so they chain on the preceding
    context and are recomputed, while the rest cache-hits."""
    if link_tokens % block_size:
        raise ValueError("link_tokens must be a block multiple")
    parts = [pad_to_block(system, block_size, pad_id)]
    for d in docs:
        d = np.asarray(d, np.int32)
        if link_tokens:
            parts.append(d[:link_tokens])
            d = d[link_tokens:]
        parts.append(span_request(d, block_size, ssep, pad_id))
    parts.append(np.concatenate([[pdep], np.asarray(task, np.int32)]).astype(np.int32))
    return np.concatenate(parts).astype(np.int32)


def isps_order(mini_batches: Sequence[Sequence[Tuple[np.ndarray, Sequence[np.ndarray], np.ndarray]]], block_size: int,
               ssep: int, pdep: int, pad_id: int, link_tokens: int = 0) -> List[Tuple[str, np.ndarray]]:
    """``mini_batches[k]`` = logical requests (system, docs, task).  Returns the single ordered list ``out`` of PAPER.md:130-139:
    for every mini-batch the distinct span-prefill requests first, then its final prompts."""
    out: List[Tuple[str, np.ndarray]] = []
    seen = set()
    for batch in mini_batches:
        for system, docs, task in batch:
            for unit in [pad_to_block(system, block_size, pad_id)] + \
                        [span_request(np.asarray(d, np.int32)[link_tokens:], block_size, ssep, pad_id) for d in docs]:
                key = unit.tobytes()
                if key not in seen:                       # step 2: deduplicate
                    seen.add(key)
                    out.append(("span", unit))            # step 3: one prefill-only request per span
        for system, docs, task in batch:                  # step 4: final prompts, cache-hit composition
            out.append(("final", compose(system, docs, task, block_size, ssep, pdep, pad_id, link_tokens)))
    return out


def replay(pool, ordered: Sequence[Tuple[str, np.ndarray]], keep: int = 4) -> dict:
    """Admit the requests in order; a request's blocks are released ``keep`` requests later (a crude max_num_seqs)."""
    total = new = final_total = final_new = 0
    live = []
    for kind, toks in ordered:
        table, hit, slots, lo, n_new = pool.admit(toks)
        total += len(toks); new += n_new
        if kind == "final":
            final_total += len(toks); final_new += n_new
        live.append(table)
        if len(live) > keep:
            pool.release(live.pop(0))
    for t in live:
        pool.release(t)
    return dict(requests=len(ordered), tokens=total, prefilled_tokens=new, final_prompt_tokens=final_total,
                final_prompt_prefilled=final_new, **pool.stats())
