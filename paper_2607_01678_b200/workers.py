"""Host-side helpers of the workers mode (include/scape.h "Workers").

PAPER.md §IV-A (:178): "each worker only computes a portion of the top-k operations"; Fig. 7 (:218)
gathers the portions.  Which worker refreshes which layer is a host decision taken once; every
worker must take the SAME decision, so it is a pure function of the layer sizes and the world size.
No arithmetic of the method lives here.
"""
from typing import List, Sequence


def balance_layers(layer_sizes: Sequence[int], world: int) -> List[int]:
    """Owner of every layer: longest-processing-time greedy (largest layer first, always to the
    least loaded worker; ties to the lower worker / lower layer), so the top-k work per worker is
    within one layer of even.  Deterministic: every worker computes the same list."""
    if world < 1:
        raise ValueError("world must be >= 1")
    load = [0] * world
    owner = [0] * len(layer_sizes)
    for l in sorted(range(len(layer_sizes)), key=lambda i: (-int(layer_sizes[i]), i)):
        if layer_sizes[l] <= 0:
            raise ValueError("layer sizes must be positive")
        w = min(range(world), key=lambda r: (load[r], r))
        owner[l] = w
        load[w] += int(layer_sizes[l])
    return owner


def owned_word_ranges(offsets: Sequence[int], owner: Sequence[int], rank: int):
    """[first, end) ranges of 32-bit mask words in which worker `rank` may have bits (a word that
    holds a layer boundary belongs to both neighbours' ranges).  For callers that prefer an
    all-gather of word-aligned portions to the integer all-reduce of the whole mask."""
    out = []
    for l, o in enumerate(owner):
        if o != rank:
            continue
        a, b = int(offsets[l]) // 32, (int(offsets[l + 1]) + 31) // 32
        if out and out[-1][1] >= a:
            out[-1] = (out[-1][0], max(out[-1][1], b))
        else:
            out.append((a, b))
    return out


def exchange_plan(offsets: Sequence[int], owner: Sequence[int], numel: int):
    """What scape_step_exchange moves of the new mask (include/scape.h; the library computes the same
    plan itself: scape_exchange_plan): every maximal run of consecutive layers with one owner is a range
    of 32-bit mask words [first, end) that only this owner writes -> ([(first, end, owner)]); a word
    that holds a boundary between two runs is shared -> ([word numbers]).  A pure function of the
    layer offsets and owners: every worker derives the same plan."""
    n_words = (int(numel) + 31) // 32
    ranges, shared = [], []
    l, n = 0, len(owner)
    while l < n:
        e = l + 1
        while e < n and owner[e] == owner[l]:
            e += 1
        a, b = int(offsets[l]), int(offsets[e])
        w0, w1 = (a + 31) // 32, n_words if b == int(numel) else b // 32
        if w1 > w0:
            ranges.append((w0, w1, int(owner[l])))
        if a % 32 != 0 and (not shared or shared[-1] != a // 32):
            shared.append(a // 32)
        l = e
    return ranges, shared
