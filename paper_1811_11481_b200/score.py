"""Truth scorer (harness only): efficiency / clone / fake rates after PAPER.md:129 (footnote 2).

A reconstructed track's label is the majority generator id of its clusters; it is *fake* if more
than 10 % of its clusters carry another label.  Without the sector merger (out of scope) every
sector crossing of a particle is its own segment, so the reference objects are (track, sector)
segments; *findable* segments have at least `min_hits` generator clusters in the sector.
"""
from __future__ import annotations

import numpy as np


def score(assignment: np.ndarray, truth: np.ndarray, sector_of_cluster: np.ndarray, n_tracks: int,
          min_hits: int = 70) -> dict:
    assignment = np.asarray(assignment)
    if n_tracks == 0:
        return dict(n_reco=0, n_findable=0, efficiency=0.0, clone_rate=0.0, fake_rate=0.0)
    sel = assignment >= 0
    a, t, s = assignment[sel].astype(np.int64), truth[sel].astype(np.int64), sector_of_cluster[sel].astype(np.int64)
    n_per_track = np.bincount(a, minlength=n_tracks)
    # majority label per reco track
    tmax = int(truth.max()) + 2
    key = a * tmax + (t + 1)
    uk, cnt = np.unique(key, return_counts=True)
    ka, kt = uk // tmax, uk % tmax - 1
    order = np.lexsort((-cnt, ka))
    first = np.ones(len(order), bool)
    first[1:] = ka[order][1:] != ka[order][:-1]
    maj_track, maj_label, maj_cnt = ka[order][first], kt[order][first], cnt[order][first]
    label = np.full(n_tracks, -1, np.int64)
    purity = np.zeros(n_tracks)
    label[maj_track] = maj_label
    purity[maj_track] = maj_cnt / np.maximum(1, n_per_track[maj_track])
    reco = n_per_track > 0
    fake = reco & ((purity < 0.9) | (label < 0))
    sec_of_track = np.full(n_tracks, -1, np.int64)
    sec_of_track[a] = s
    # findable (truth id, sector) segments
    sig = truth >= 0
    nsec = int(sector_of_cluster.max()) + 1
    seg = truth[sig].astype(np.int64) * nsec + sector_of_cluster[sig]
    useg, ucnt = np.unique(seg, return_counts=True)
    findable = useg[ucnt >= min_hits]
    good = reco & ~fake
    reco_seg = label[good] * nsec + sec_of_track[good]
    rs, rc = np.unique(reco_seg, return_counts=True)
    found = np.isin(findable, rs)
    clones = int((rc - 1).sum())
    return dict(n_reco=int(reco.sum()), n_findable=int(len(findable)),
                efficiency=float(found.mean()) if len(findable) else 0.0,
                clone_rate=clones / max(1, int(reco.sum())), fake_rate=float(fake.sum()) / max(1, int(reco.sum())))


def sector_of_cluster(sector_offsets: np.ndarray, n: int) -> np.ndarray:
    so = np.asarray(sector_offsets)
    return (np.searchsorted(so, np.arange(n), side="right") - 1).astype(np.int32)
