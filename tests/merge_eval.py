"""Link efficiency / purity of a sector-boundary merge (C7) against generator truth (pin M-E).

A track's truth key is the (particle, sector, arc) that holds >= 70 % of its hits (as in truth_eval.py).  The
EXPECTED links are, for every (particle, arc), the consecutive pieces (ordered by first row) that sit in adjacent
sectors of the same side and whose rows satisfy the merge's own row window; a produced link is GOOD when both ends
belong to the same (particle, arc).  Pure numpy; contains none of the merge arithmetic.
"""
from __future__ import annotations

from collections import defaultdict

import numpy as np

import truth_eval as TE


def track_truth_keys(tf, hit_offset, n_hits, hit_index, purity: float = 0.7) -> np.ndarray:
    seg = TE.segment_ids(tf)
    out = np.full(len(n_hits), -1, np.int64)
    for i in range(len(n_hits)):
        o = int(hit_offset[i])
        s = seg[hit_index[o:o + int(n_hits[i])]]
        s = s[s >= 0]
        if s.size == 0:
            continue
        v, c = np.unique(s, return_counts=True)
        j = int(np.argmax(c))
        if c[j] >= purity * int(n_hits[i]):
            out[i] = v[j]
    return out


def evaluate_links(keys, sector, first_row, last_row, nxt, max_row_gap: int = 12, max_row_overlap: int = 2) -> dict:
    n = len(keys)
    particle = np.where(keys >= 0, keys // (64 * 16), -1)
    arc = keys % 16
    links = [(a, int(nxt[a])) for a in range(n) if nxt[a] >= 0]
    good = sum(1 for a, b in links if keys[a] >= 0 and keys[b] >= 0 and particle[a] == particle[b] and arc[a] == arc[b])
    groups = defaultdict(list)
    for i in range(n):
        if keys[i] >= 0:
            groups[(int(particle[i]), int(arc[i]))].append(i)
    expected = got = 0
    for idx in groups.values():
        idx.sort(key=lambda i: (first_row[i], i))
        for a, b in zip(idx[:-1], idx[1:]):
            sa, sb = int(sector[a]), int(sector[b])
            adjacent = sa // 18 == sb // 18 and (sa % 18 - sb % 18) % 18 in (1, 17)
            rows_ok = last_row[a] + 1 - max_row_overlap <= first_row[b] <= last_row[a] + 1 + max_row_gap
            if adjacent and rows_ok and first_row[b] > first_row[a]:
                expected += 1
                got += int(nxt[a] == b)
    return dict(n_tracks=n, n_links=len(links), good=good, wrong=len(links) - good, expected=expected, got=got,
                efficiency=(got / expected if expected else float("nan")),
                wrong_rate=((len(links) - good) / len(links) if links else 0.0))
