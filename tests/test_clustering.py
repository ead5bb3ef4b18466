"""Candidate clustering (reading C10) — CPU only. The library's sweep + union-find against
(1) hand-worked cases that fix every clause of the definition (inclusive tolerances, chains, the tie rule, extents) and
(2) the oracle's O(n^2) written-out definition on random lists, plus the invariants any clustering must have."""
import numpy as np
import pytest

import oracle
import paper_1912_07704_b200 as aa


def _cands(rows):
    """rows: (sample, width, dm, snr, range, dm_index)"""
    c = np.zeros(len(rows), dtype=aa.CANDIDATE_DTYPE)
    for i, (s, w, dm, snr, r, di) in enumerate(rows):
        c[i] = (s, dm, snr, w, r, di)
    return c


def _as_sets(cl, cands):
    """clusters (library output) -> set of frozensets of member keys, recovered from extents is impossible, so compare via
    representatives and member counts; membership itself is compared through the oracle in the random test."""
    return sorted((int(k["best"]["sample"]), int(k["best"]["dm_index"]), int(k["members"])) for k in cl)


def test_hand_worked_cases():
    # two boxcars [100,104) and [106,110): 2 samples apart -> linked iff gap >= 2 (inclusive); DM differs by 0.5
    c = _cands([(100, 4, 10.0, 8.0, 0, 100), (106, 4, 10.5, 9.0, 0, 105)])
    assert len(aa.aa_cluster_candidates(c, 0.5, 1)) == 2
    one = aa.aa_cluster_candidates(c, 0.5, 2)
    assert len(one) == 1 and one[0]["members"] == 2 and float(one[0]["best"]["snr"]) == 9.0
    assert (int(one[0]["sample_min"]), int(one[0]["sample_end"])) == (100, 110)
    assert (float(one[0]["dm_min"]), float(one[0]["dm_max"])) == (10.0, 10.5)
    assert len(aa.aa_cluster_candidates(c, 0.49, 2)) == 2                       # DM tolerance is inclusive at 0.5 only
    # a chain: A-B linked, B-C linked, A-C not -> one cluster (connected components, not cliques)
    c = _cands([(0, 10, 1.0, 7.5, 0, 1), (12, 10, 2.0, 7.2, 0, 2), (24, 10, 3.0, 7.9, 0, 3)])
    k = aa.aa_cluster_candidates(c, 1.0, 2)
    assert len(k) == 1 and k[0]["members"] == 3 and int(k[0]["best"]["dm_index"]) == 3
    # a wide early boxcar reaches a later narrow one that starts inside it
    c = _cands([(0, 1000, 5.0, 8.0, 1, 7), (900, 1, 5.0, 8.5, 0, 50), (2000, 1, 5.0, 9.0, 0, 50)])
    k = aa.aa_cluster_candidates(c, 0.0, 0)
    assert _as_sets(k, c) == [(900, 50, 2), (2000, 50, 1)]
    # equal SNR: the representative is the first by (range, dm_index, sample); clusters are ordered the same way
    c = _cands([(50, 2, 4.0, 8.0, 1, 3), (51, 2, 4.0, 8.0, 0, 9), (500, 2, 4.0, 8.0, 0, 2)])
    k = aa.aa_cluster_candidates(c, 0.0, 0)
    assert [(int(x["best"]["range"]), int(x["best"]["dm_index"])) for x in k] == [(0, 2), (0, 9)]
    # empty list, bad tolerance
    assert len(aa.aa_cluster_candidates(c[:0], 1.0, 1)) == 0
    with pytest.raises(aa.AaError) as e:
        aa.aa_cluster_candidates(c, -1.0, 0)
    assert e.value.status == aa.AA_ERR_INVALID_ARG and "dm_tol" in e.value.message


def test_hand_worked_cases_pin_the_oracle():
    """The same hand-worked lists through oracle.cluster_candidates ALONE: member sets and representatives are stated here from
    the definition (reading C10), not taken from either implementation, so a mistake in the oracle's O(n^2) loop (a `<` for a
    `<=` in any of its three clauses, cliques instead of components, a wrong tie rule) fails without the library's help."""
    oc = lambda c, dm_tol, gap: tuple(map(list, oracle.cluster_candidates(c, dm_tol, gap)))
    # boxcars [100,104) and [106,110): 106 <= 100 + 4 + gap iff gap >= 2; |10.5 - 10.0| <= dm_tol iff dm_tol >= 0.5
    c = _cands([(100, 4, 10.0, 8.0, 0, 100), (106, 4, 10.5, 9.0, 0, 105)])
    assert oc(c, 0.5, 1) == ([[0], [1]], [0, 1])
    assert oc(c, 0.5, 2) == ([[0, 1]], [1])                     # inclusive at gap = 2 and at dm_tol = 0.5; best = snr 9.0
    assert oc(c, 0.49, 2) == ([[0], [1]], [0, 1])
    # the mirrored clause (the LATER boxcar is listed first): sample_a <= sample_b + width_b + gap at equality
    c = _cands([(106, 4, 10.5, 9.0, 0, 105), (100, 4, 10.0, 8.0, 0, 100)])
    assert oc(c, 0.5, 2) == ([[0, 1]], [0])
    assert oc(c, 0.5, 1) == ([[0], [1]], [0, 1])
    # a chain A-B, B-C linked, A-C not (24 > 0 + 10 + 2; |3 - 1| > 1): ONE cluster, connected components not cliques
    c = _cands([(0, 10, 1.0, 7.5, 0, 1), (12, 10, 2.0, 7.2, 0, 2), (24, 10, 3.0, 7.9, 0, 3)])
    assert oc(c, 1.0, 2) == ([[0, 1, 2]], [2])
    assert oc(c, 1.0, 1) == ([[0], [1], [2]], [0, 1, 2])        # 12 > 0 + 10 + 1: the chain falls apart
    # a wide early boxcar [0,1000) reaches the narrow one that starts inside it, not the one at 2000
    c = _cands([(0, 1000, 5.0, 8.0, 1, 7), (900, 1, 5.0, 8.5, 0, 50), (2000, 1, 5.0, 9.0, 0, 50)])
    assert oc(c, 0.0, 0) == ([[0, 1], [2]], [1, 2])
    # touching boxcars [0,1000) and [1000,1001) are linked at gap 0 (1000 <= 0 + 1000 + 0); one sample further is not
    c = _cands([(0, 1000, 5.0, 8.0, 0, 7), (1000, 1, 5.0, 8.5, 0, 7), (2002, 1, 5.0, 8.5, 0, 7)])
    assert oc(c, 0.0, 0) == ([[0, 1], [2]], [1, 2])
    assert oc(c, 0.0, 1000) == ([[0, 1], [2]], [1, 2])          # 2002 > 1000 + 1 + 1000
    assert oc(c, 0.0, 1001) == ([[0, 1, 2]], [1])               # equal snr 8.5: the earlier sample represents
    # equal SNR everywhere: the representative is the first by (range, dm_index, sample)
    c = _cands([(50, 2, 4.0, 8.0, 1, 3), (51, 2, 4.0, 8.0, 0, 9), (500, 2, 4.0, 8.0, 0, 2)])
    assert oc(c, 0.0, 0) == ([[0, 1], [2]], [1, 2])             # (0, 9, 51) sorts before (1, 3, 50)
    assert oc(c[:0], 1.0, 1) == ([], [])


@pytest.mark.parametrize("seed,n,dm_tol,gap", [(1, 300, 0.6, 3), (2, 500, 0.0, 0), (3, 400, 2.5, 40), (4, 1, 1.0, 1)])
def test_random_lists_equal_the_written_out_definition(seed, n, dm_tol, gap):
    rs = np.random.default_rng(seed)
    rows = [(int(rs.integers(0, 4000)), int(2 ** rs.integers(0, 7)), float(rs.integers(0, 40)) * 0.3, float(rs.integers(70, 90)) / 10.0,
             int(rs.integers(0, 3)), int(rs.integers(0, 50))) for _ in range(n)]
    c = _cands(rows)
    got = aa.aa_cluster_candidates(c, dm_tol, gap)
    clusters, reps = oracle.cluster_candidates(c, dm_tol, gap)
    assert len(got) == len(clusters) and int(got["members"].sum()) == n              # a partition of the list
    exp = {}
    for members, r in zip(clusters, reps):
        key = (int(c["range"][r]), int(c["dm_index"][r]), int(c["sample"][r]), float(c["snr"][r]))
        exp[key] = (len(members), min(int(c["sample"][m]) for m in members), max(int(c["sample"][m]) + int(c["width"][m]) for m in members),
                    min(float(c["dm"][m]) for m in members), max(float(c["dm"][m]) for m in members))
    keys = []
    for k in got:
        key = (int(k["best"]["range"]), int(k["best"]["dm_index"]), int(k["best"]["sample"]), float(k["best"]["snr"]))
        assert key in exp, key
        assert exp[key] == (int(k["members"]), int(k["sample_min"]), int(k["sample_end"]), float(k["dm_min"]), float(k["dm_max"]))
        keys.append(key[:3])
    assert keys == sorted(keys)                                                      # ordered by (range, dm_index, sample)
    # order of the input does not matter
    perm = rs.permutation(n)
    again = aa.aa_cluster_candidates(c[perm], dm_tol, gap)
    assert len(again) == len(got) and all(np.array_equal(again[f], got[f]) for f in ("members", "sample_min", "sample_end"))
    # widening a tolerance can only merge clusters
    assert len(aa.aa_cluster_candidates(c, dm_tol + 1.0, gap + 10)) <= len(got)
