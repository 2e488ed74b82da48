"""Efficiency / fake / clone rates of a set of tracks against generator truth (pin E1, BASELINE.json L5 (d)).

Definitions ([proposed]): a truth *segment* is one particle's clusters in one sector on one
monotone-in-x arc; it is *findable* with >= 60 clusters after dropout; it is *found* when some track has >= 70 % of
its hits from that segment.  A track is a *fake* when no segment holds 70 % of its hits, a *clone* when its
segment was already found by another track.  Pure numpy; takes hit lists by ORIGINAL cluster index.
"""
from __future__ import annotations

import numpy as np


def segment_ids(tf, n_rows: int = 152) -> np.ndarray:
    """int64 segment key per cluster: (particle, sector, arc); -1 for noise."""
    sector = (tf.row.astype(np.int64) // n_rows)
    seg = (tf.truth_track.astype(np.int64) * 64 + sector) * 16 + tf.truth_arc.astype(np.int64)
    seg[tf.truth_track < 0] = -1
    return seg


def evaluate(tf, hit_offset, n_hits, hit_index, pt_min: float = 0.2, findable_min: int = 60,
             purity: float = 0.7, n_rows: int = 152) -> dict:
    seg = segment_ids(tf, n_rows)
    valid = seg >= 0
    useg, inv, cnt = np.unique(seg[valid], return_inverse=True, return_counts=True)
    seg_compact = np.full(seg.shape[0], -1, np.int64)
    seg_compact[valid] = inv
    particle = useg // (64 * 16)
    pt = tf.tracks["pt"][particle]
    findable = (cnt >= findable_min) & (pt > pt_min)
    n_tracks = int(len(n_hits))
    found_by = np.zeros(len(useg), np.int32)
    n_fake = 0
    for i in range(n_tracks):
        o = int(hit_offset[i])
        s = seg_compact[hit_index[o:o + int(n_hits[i])]]
        s = s[s >= 0]
        if s.size == 0:
            n_fake += 1
            continue
        vals, c = np.unique(s, return_counts=True)
        j = int(np.argmax(c))
        if c[j] >= purity * int(n_hits[i]):
            found_by[vals[j]] += 1
        else:
            n_fake += 1
    n_findable = int(findable.sum())
    n_found = int(((found_by > 0) & findable).sum())
    n_clone = int(np.maximum(found_by - 1, 0).sum())
    return dict(n_tracks=n_tracks, n_findable=n_findable, n_found=n_found,
                efficiency=(n_found / n_findable if n_findable else float("nan")),
                fake_rate=(n_fake / n_tracks if n_tracks else 0.0),
                clone_rate=(n_clone / n_tracks if n_tracks else 0.0))
