"""Test-side physics bookkeeping against the generator's truth labels (no tracker arithmetic, no oracle code).

A *findable segment* is a (true track, sector) pair with >= `min_clusters` clusters ("findable =
>= 20 clusters in the sector").  A reconstructed track is matched to the true track that owns the majority of its
hits; it is a *fake* if that majority is below half of its hits or is noise (label -1).
"""
import numpy as np


def physics_summary(ev, out, min_clusters=20):
    """out: oracle- or CUDA-style result dict (cluster_track, trk_seed, trk_nhits, trk_first_hit, trk_hits)."""
    nrows = int(ev.params.n_rows)
    tt = np.asarray(ev.true_track).astype(np.int64)
    sec = np.asarray(ev.sector_row) // nrows
    K = int(out["trk_seed"].size)
    owner = np.repeat(np.arange(K), out["trk_nhits"])
    hits = out["trk_hits"]
    # majority truth label per reconstructed track
    lab = tt[hits]
    maj = np.full(K, -1, np.int64)
    purity = np.zeros(K)
    order = np.lexsort((lab, owner))
    lo, oo = lab[order], owner[order]
    start = np.nonzero(np.r_[True, (lo[1:] != lo[:-1]) | (oo[1:] != oo[:-1])])[0]
    cnt = np.diff(np.r_[start, lo.size])
    best = {}
    for s, c in zip(start, cnt):
        k = int(oo[s])
        if c > best.get(k, (0, 0))[0]:
            best[k] = (int(c), int(lo[s]))
    for k, (c, l) in best.items():
        maj[k] = l
        purity[k] = c / float(out["trk_nhits"][k])
    fake = (maj < 0) | (purity < 0.5)
    # findable segments
    sig = tt >= 0
    key = tt[sig] * 64 + sec[sig]
    uk, ucnt = np.unique(key, return_counts=True)
    findable = set(uk[ucnt >= min_clusters].tolist())
    trk_sector = np.asarray(ev.sector_row)[out["trk_seed"]] // nrows
    found_by = {}
    for k in range(K):
        if fake[k]:
            continue
        kk = int(maj[k]) * 64 + int(trk_sector[k])
        if kk in findable:
            found_by.setdefault(kk, []).append(k)
    # attached fraction: clusters of findable segments owned by a track whose majority is the same true track
    ct = np.asarray(out["cluster_track"])
    in_find = sig & np.isin(tt * 64 + sec, np.fromiter(findable, np.int64, len(findable)))
    idx = np.nonzero(in_find)[0]
    own = ct[idx]
    good = (own >= 0) & (maj[np.maximum(own, 0)] == tt[idx])
    return dict(tracks=K, findable=len(findable), found=len(found_by),
                efficiency=len(found_by) / max(len(findable), 1),
                duplicates=int(sum(len(v) - 1 for v in found_by.values())),
                fakes=int(np.count_nonzero(fake)),
                attached=float(np.count_nonzero(good)) / max(idx.size, 1),
                assigned=int(np.count_nonzero(ct >= 0)))
