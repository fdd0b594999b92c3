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
        st["cov_max_rel"] = float(rel_c.max()) if rel_c.size else 0.0
        st["par_bit_identical"] = bool(np.array_equal(orc_out["par"][:, io], res["par"][:, ig]))
        st["cov_bit_identical"] = bool(np.array_equal(orc_out["cov"][:, io], res["cov"][:, ig]))
        st["chi2_max_rel"] = float(np.max(np.abs(orc_out["chi2"][io] - res["chi2"][ig]) /
                                          np.maximum(np.abs(orc_out["chi2"][io]), 1.0))) if io.size else 0.0
        assert np.array_equal(orc_out["ndf"][io], res["ndf"][ig])
        assert np.array_equal(orc_out["xref"][io], res["xref"][ig])
        assert np.array_equal(orc_out["zref"][io], res["zref"][ig])
    return st


def assert_contract(st, exact_count=False):
    assert st["assign_frac"] >= 0.999, f"only {st['assign_frac']:.6f} of cluster assignments identical (need >= 0.999)"
    if exact_count:
        assert st["tracks_oracle"] == st["tracks_cuda"], (st["tracks_oracle"], st["tracks_cuda"])
    assert st.get("par_max_rel", 0.0) <= REL_TOL, f"track parameters differ by {st['par_max_rel']:.3e} relative"
    assert st.get("cov_max_rel", 0.0) <= REL_TOL, f"covariance diagonals differ by {st['cov_max_rel']:.3e} relative"
