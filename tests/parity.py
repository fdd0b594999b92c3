"""Parity harness: compares the CUDA path (binding.Tracker) with the CPU oracle stage by stage.

Tolerances are BASELINE.json north_star's: cluster-to-track assignments identical for >= 99.9 % of clusters
(differences must be near-tie chi2 comparisons), fitted parameters and covariance diagonals of matched tracks
within 1e-4 relative (floors of SURVEY.md A9), track counts exact.  Because the CUDA path is compiled without
FMA contraction and restates the oracle's operation order, the observed agreement is bit-for-bit; the
tolerances are the contract, the exact-equality counters are reported beside them.
"""
from __future__ import annotations

import numpy as np

#: A9 floors for "1e-4 relative" on quantities that can be ~0: y, dz [cm], sinphi, tanlambda, q/pT [1/GeV]
PAR_FLOOR = np.array([1.0, 1.0, 0.1, 0.1, 0.1])
REL_TOL = 1e-4
COV_DIAG = [0, 2, 5, 9, 14]


def cluster_seed(cluster_track, trk_seed):
    """Per-cluster seed (original index of the owning track's start hit), -1 = unassigned: order-free label."""
    ct = np.asarray(cluster_track)
    seeds = np.asarray(trk_seed)
    out = np.full(ct.shape, -1, np.int64)
    m = ct >= 0
    out[m] = seeds[ct[m]]
    return out


def compare_grid(orc_out, sorted_idx, bin_first):
    assert np.array_equal(orc_out["bin_first"], bin_first), "bin_first differs from the oracle's (R7)"
    assert np.array_equal(orc_out["sorted_idx"], sorted_idx), "sorted order differs from the oracle's stable sort (R7)"


def compare_links(orc_out, fe):
    for k in ("link_up", "link_dn", "up_c", "dn_c"):
        bad = np.nonzero(orc_out[k] != fe[k])[0]
        assert bad.size == 0, f"{k}: {bad.size} of {fe[k].size} differ, first at cluster {bad[:5]}"
    a = np.sort(orc_out["starts"])
    b = np.sort(fe["starts"])
    assert np.array_equal(a, b), f"start hits differ: oracle {a.size}, cuda {b.size}"


def compare_tracklets(orc_out, fe):
    """row_hit / n_hits per tracklet, matched by start hit.  Returns the number of differing tracklets."""
    oi = np.argsort(orc_out["starts"])
    gi = np.argsort(fe["starts"])
    assert np.array_equal(orc_out["starts"][oi], fe["starts"][gi])
    rh_o = orc_out["row_hit"][oi]
    rh_g = fe["row_hit"][gi]
    diff_rows = np.any(rh_o != rh_g, axis=1)
    nh_diff = orc_out["n_hits"][oi] != fe["n_hits"][gi]
    return int(np.count_nonzero(diff_rows | nh_diff)), int(oi.size)


def compare_tracks(orc_out, res, n):
    """Selection + fit.  Returns a stats dict; raises on contract violations."""
    st = {}
    cs_o = cluster_seed(orc_out["cluster_track"], orc_out["trk_seed"])
    cs_g = cluster_seed(res["cluster_track"], res["trk_seed"])
    same = int(np.count_nonzero(cs_o == cs_g))
    st["n_clusters"] = int(n)
    st["assign_identical"] = same
    st["assign_frac"] = same / max(n, 1)
    st["tracks_oracle"] = int(orc_out["trk_seed"].size)
    st["tracks_cuda"] = int(res["trk_seed"].size)
    # exclusivity and consistency of the CUDA output on its own
    hits = res["trk_hits"]
    assert np.unique(hits).size == hits.size, "a cluster appears in two tracks"
    assert int(res["trk_nhits"].sum()) == hits.size == int(np.count_nonzero(res["cluster_track"] >= 0))
    assert np.unique(res["trk_seed"]).size == res["trk_seed"].size
    # match tracks by seed
    o_of = {int(s): i for i, s in enumerate(orc_out["trk_seed"])}
    pairs = [(o_of[int(s)], j) for j, s in enumerate(res["trk_seed"]) if int(s) in o_of]
    st["tracks_matched"] = len(pairs)
    if pairs:
        io = np.array([p[0] for p in pairs])
        ig = np.array([p[1] for p in pairs])
        same_hits = (orc_out["trk_nhits"][io] == res["trk_nhits"][ig])
        # identical hit lists?
        for k in np.nonzero(same_hits)[0]:
            a = orc_out["trk_hits"][orc_out["trk_first_hit"][io[k]]:orc_out["trk_first_hit"][io[k]] + orc_out["trk_nhits"][io[k]]]
            b = res["trk_hits"][res["trk_first_hit"][ig[k]]:res["trk_first_hit"][ig[k]] + res["trk_nhits"][ig[k]]]
            if not np.array_equal(a, b):
                same_hits[k] = False
        st["tracks_same_hits"] = int(np.count_nonzero(same_hits))
        io, ig = io[same_hits], ig[same_hits]      # parameters are comparable only for identical hit lists
        po, pg = orc_out["par"][:, io].astype(np.float64), res["par"][:, ig].astype(np.float64)
        scale = np.maximum(np.maximum(np.abs(po), np.abs(pg)), PAR_FLOOR[:, None])
        rel_p = np.abs(po - pg) / scale
        co, cg = orc_out["cov"][COV_DIAG][:, io].astype(np.float64), res["cov"][COV_DIAG][:, ig].astype(np.float64)
        rel_c = np.abs(co - cg) / np.maximum(np.abs(co), np.abs(cg))
        st["par_max_rel"] = float(rel_p.max()) if rel_p.size else 0.0
        st["par_median_rel"] = float(np.median(rel_p)) if rel_p.size else 0.0
        st["cov_max_rel"] = float(rel_c.max()) if rel_c.size else 0.0
        st["par_bit_identical"] = bool(np.array_equal(orc_out["par"][:, io], res["par"][:, ig]))
        st["cov_bit_identical"] = bool(np.array_equal(orc_out["cov"][:, io], res["cov"][:, ig]))
        st["chi2_max_rel"] = float(np.max(np.abs(orc_out["chi2"][io] - res["chi2"][ig]) /
                                          np.maximum(np.abs(orc_out["chi2"][io]), 1.0))) if io.size else 0.0
        assert np.array_equal(orc_out["ndf"][io], res["ndf"][ig])
        if orc_out["par"].dtype == res["par"].dtype:      # an fp64 run holds the unrounded row positions
            assert np.array_equal(orc_out["xref"][io], res["xref"][ig])
            assert np.array_equal(orc_out["zref"][io], res["zref"][ig])
    return st


def assert_contract(st, exact_count=False):
    assert st["assign_frac"] >= 0.999, f"only {st['assign_frac']:.6f} of cluster assignments identical (need >= 0.999)"
    if exact_count:
        assert st["tracks_oracle"] == st["tracks_cuda"], (st["tracks_oracle"], st["tracks_cuda"])
    assert st.get("par_max_rel", 0.0) <= REL_TOL, f"track parameters differ by {st['par_max_rel']:.3e} relative"
    assert st.get("cov_max_rel", 0.0) <= REL_TOL, f"covariance diagonals differ by {st['cov_max_rel']:.3e} relative"


def restrict_to_sector(res, sector_row, n_rows, sector):
    """View of a whole-event CUDA result restricted to one sector, re-indexed to the sector's own cluster
    numbering (position in `sel`, which is ascending in original index, so every index tie-break is preserved).
    Sectors are independent through the whole hot path (R2, R9-R22 are sector-local), so the oracle run on the
    sector's clusters alone must reproduce this view.  Returns (sel, res_sector)."""
    sel = np.nonzero(np.asarray(sector_row) // n_rows == sector)[0]
    tk = np.nonzero(res["trk_sector"] == sector)[0]
    new_of_old = np.full(res["trk_seed"].size, -1, np.int64)
    new_of_old[tk] = np.arange(tk.size)
    ct = res["cluster_track"][sel]
    ct_new = np.where(ct >= 0, new_of_old[np.maximum(ct, 0)], -1)
    assert np.all((ct < 0) | (ct_new >= 0)), "a cluster of this sector is owned by a track of another sector"
    nh = res["trk_nhits"][tk]
    first = np.concatenate([[0], np.cumsum(nh)[:-1]]).astype(np.int64) if tk.size else np.zeros(0, np.int64)
    hits = np.concatenate([res["trk_hits"][res["trk_first_hit"][k]:res["trk_first_hit"][k] + res["trk_nhits"][k]]
                           for k in tk]) if tk.size else np.zeros(0, np.int32)
    pos = np.searchsorted(sel, hits)
    assert np.array_equal(sel[np.minimum(pos, sel.size - 1)], hits), "a track holds a cluster of another sector"
    out = dict(cluster_track=ct_new.astype(np.int32), trk_seed=np.searchsorted(sel, res["trk_seed"][tk]).astype(np.int32),
               trk_sector=res["trk_sector"][tk], trk_nhits=nh, trk_first_hit=first, trk_hits=pos.astype(np.int32))
    for k in ("par", "cov"):
        out[k] = res[k][:, tk]
    for k in ("xref", "zref", "chi2", "ndf"):
        out[k] = res[k][tk]
    return sel, out


def check_output_invariants(res, sector_row, n_rows, min_hits):
    """Properties of a valid output that hold at any size (used at the full bench size, where the oracle can only
    be afforded on sampled sectors): exclusivity, list/flag consistency, one sector and strictly ascending rows per
    track, >= min_hits, ndf = 2 nHits - 5, unique seeds (a seed may be owned by a longer rival, R20)."""
    ct, hits, nh, first = res["cluster_track"], res["trk_hits"], res["trk_nhits"], res["trk_first_hit"]
    K = res["trk_seed"].size
    assert int(nh.sum()) == hits.size
    assert np.array_equal(first, np.concatenate([[0], np.cumsum(nh)[:-1]])), "hit lists are not packed in track order"
    assert np.all(nh >= min_hits)
    owner = np.repeat(np.arange(K, dtype=np.int32), nh)
    assert np.array_equal(ct[hits], owner), "cluster_track disagrees with the hit lists"
    assert int(np.count_nonzero(ct >= 0)) == hits.size, "a cluster is flagged assigned but is in no hit list (or twice)"
    sr = np.asarray(sector_row)[hits]
    assert np.array_equal(sr // n_rows, np.repeat(res["trk_sector"], nh)), "a track mixes sectors"
    inner = np.ones(hits.size, bool)
    inner[first] = False
    assert np.all(np.diff(sr % n_rows)[inner[1:]] > 0), "rows of a track are not strictly ascending"
    assert np.unique(res["trk_seed"]).size == K
    ok = res["ndf"] >= 0
    assert np.array_equal(res["ndf"][ok], 2 * nh[ok] - 5)


# ------------------------------------------------------------------------------------------------------------
# near-tie report (BASELINE.json north_star: "any differences must be logged as near-tie chi2 comparisons")
# ------------------------------------------------------------------------------------------------------------
NEAR_TIE_KINDS = {0: "R16 search", 1: "R15 chain cut", 2: "max_sinphi", 3: "sector edge"}


def _margin(rec):
    """Relative distance of a logged decision (oracle DecRec) from flipping: the smallest of
    |best - second| / max (two candidates swap) and |best - cut| / cut (the cut flips)."""
    best, second, cut = float(rec["best"]), float(rec["second"]), float(rec["cut"])
    m = np.inf
    if np.isfinite(best):
        m = abs(best - cut) / abs(cut)
        if np.isfinite(second):
            m = min(m, abs(best - second) / max(abs(best), abs(second), 1e-300), abs(second - cut) / abs(cut))
    return m


def near_tie_report(ref, other, dec_log, log=None):
    """Explains the differences between two runs of the follower on the same input (`ref`, whose decision log
    `dec_log` is given, against `other`; dicts with starts / row_hit / n_hits as oracle.follow and
    Tracker.find_export return them, original cluster indices).

    For every tracklet (matched by start hit) whose row table differs, the decisions `ref` took are replayed in
    order against `other`'s table: the FIRST decision whose outcome `other` does not share is that tracklet's root
    cause, and its margin (see _margin) says how near a tie it was.  A tracklet that differs without such a decision
    is secondary: `other` went on where `ref` had stopped, or the tracklet was absorbed / not absorbed because an
    upward leg of a root-cause tracklet marked its start hit differently (R17).  Returns a dict: differing tracklets,
    root causes with their margins, secondaries; every root cause is written to `log` (a list of strings)."""
    oi = np.argsort(ref["starts"])
    gi = np.argsort(other["starts"])
    assert np.array_equal(ref["starts"][oi], other["starts"][gi]), "the two runs do not share their start hits"
    g_of_o = np.empty(oi.size, np.int64)
    g_of_o[oi] = gi                                   # tracklet number in `other` of ref's tracklet t
    differ = np.nonzero(np.any(ref["row_hit"] != other["row_hit"][g_of_o], axis=1))[0]
    out = dict(tracklets=int(oi.size), differing=int(differ.size), roots=[], secondary=0, absorbed_flip=0)
    if differ.size == 0:
        return out
    order = np.argsort(dec_log["tracklet"], kind="stable")
    lo = np.searchsorted(dec_log["tracklet"][order], differ, "left")
    hi = np.searchsorted(dec_log["tracklet"][order], differ, "right")
    for t, a, b in zip(differ, lo, hi):
        rh_other = other["row_hit"][g_of_o[t]]
        if (ref["n_hits"][t] == 0) != (other["n_hits"][g_of_o[t]] == 0):
            out["absorbed_flip"] += 1                 # R17: marked by somebody else's upward leg in one run only
            continue
        root = None
        for rec in dec_log[order[a:b]]:
            kind, row, chosen = int(rec["kind"]), int(rec["row"]), int(rec["chosen"])
            if kind in (0, 1) and rh_other[row] != chosen:
                root = rec
                break
            if kind in (2, 3) and chosen < 0:         # ref stopped here; did `other` go on past this row?
                root = rec
                break
        if root is None:
            out["secondary"] += 1
            continue
        m = _margin(root)
        out["roots"].append((int(t), int(root["kind"]), int(root["row"]), m))
        if log is not None:
            log.append(f"tracklet {int(t)} (start hit {int(ref['starts'][t])}): {NEAR_TIE_KINDS[int(root['kind'])]} on row "
                       f"{int(root['row'])}: best {root['best']:.9g}, second {root['second']:.9g}, cut {root['cut']:.9g}, "
                       f"relative margin {m:.3e}")
    return out
