"""Track-finding efficiency, clone and fake rate against the generator truth (reported next to the throughput).

Definitions: PAPER.md:47 ("findable" = at least 70 cm inside the TPC, pT >= 200 MeV, |eta| <= 0.9); a final track
is matched to a truth track if >= 90 % of its hits carry that label.  Pure
bookkeeping on integer labels: none of the tracker's arithmetic lives here.
"""
from __future__ import annotations

import numpy as np


def report(ev, cluster_owner: np.ndarray, n_tracks: int, *, min_span_cm=70.0, min_pt=0.2, max_eta=0.9,
           match_frac=0.9) -> dict:
    """ev: datagen.Event (one or more windows); cluster_owner: final track index per cluster or -1."""
    n = ev.n_clusters
    R = ev.n_rows
    labels = ev.labels.astype(np.int64)
    slab = np.searchsorted(ev.row_offsets, np.arange(n), side="right") - 1
    inst, row = slab // R, slab % R
    x = ev.clusters[:, 0].astype(np.float64)
    sig = labels >= 0
    # truth segments: (label, instance)
    n_lab = int(labels.max()) + 1 if sig.any() else 0
    key = labels[sig] * ev.n_inst + inst[sig]
    uk, inv = np.unique(key, return_inverse=True)
    xmin = np.full(len(uk), np.inf)
    xmax = np.full(len(uk), -np.inf)
    np.minimum.at(xmin, inv, x[sig])
    np.maximum.at(xmax, inv, x[sig])
    seg_label = uk // ev.n_inst
    pt = np.asarray(ev.truth["pt"])[seg_label]
    eta = np.asarray(ev.truth["eta"])[seg_label]
    findable = ((xmax - xmin) >= min_span_cm) & (pt >= min_pt) & (np.abs(eta) <= max_eta)
    # tracks: majority label
    own = cluster_owner.astype(np.int64)
    att = own >= 0
    trk_n = np.bincount(own[att], minlength=n_tracks)
    # count (track, label) pairs among signal hits
    ts = att & sig
    pair = own[ts] * (n_lab + 1) + labels[ts]
    up, cnt = np.unique(pair, return_counts=True)
    ptrk, plab = up // (n_lab + 1), up % (n_lab + 1)
    best = np.zeros(n_tracks, np.int64)
    best_lab = np.full(n_tracks, -1, np.int64)
    order = np.argsort(cnt, kind="stable")
    best[ptrk[order]] = cnt[order]        # last write wins = largest count
    best_lab[ptrk[order]] = plab[order]
    matched = (trk_n > 0) & (best >= match_frac * trk_n)
    # instance of each track = instance of any of its clusters
    trk_inst = np.zeros(n_tracks, np.int64)
    trk_inst[own[att]] = inst[att]
    mkey = best_lab[matched] * ev.n_inst + trk_inst[matched]
    seg_index = {int(k): i for i, k in enumerate(uk)}
    hits_per_seg = np.zeros(len(uk), np.int64)
    for k in mkey:
        i = seg_index.get(int(k))
        if i is not None:
            hits_per_seg[i] += 1
    n_findable = int(findable.sum())
    found = int(((hits_per_seg > 0) & findable).sum())
    clones = int((hits_per_seg[hits_per_seg > 0] - 1).sum())
    n_matched = int(matched.sum())
    return dict(findable=n_findable, found=found, efficiency=found / max(n_findable, 1), tracks=int(n_tracks),
                matched=n_matched, fake_rate=(n_tracks - n_matched) / max(n_tracks, 1),
                clone_rate=clones / max(n_matched, 1),
                attached_signal_frac=float((att & sig).sum() / max(sig.sum(), 1)))
