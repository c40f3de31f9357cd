"""Pins of the NEXT-4 oracle (oracle/tangram_oracle_islands.cpp: GPU island construction): an
independent checker of the island definition (Eq. 1-3) and of the greedy stop condition, the evaluation clusters of
Tab. 3, hand-worked cases, limiting cases and relabelling."""
import itertools

import numpy as np
import pytest

import oracle
import tg_inputs as gen

EPS = (100, 50, 100)        # permille: 10 % compute, 5 % memory, 10 % intra-node bandwidth


def check_islands(prof, eps, of):
    """Eq. 1-3 of PAPER.md:181-189 for every island, straight from the definition."""
    gp, comp, mem, intra, inter = prof
    n = gp.size
    K = int(of.max()) + 1
    assert sorted(set(of.tolist())) == list(range(K))                                  # a partition, densely numbered
    first = [min(i for i in range(n) if of[i] == k) for k in range(K)]
    assert first == sorted(first)                                                      # numbered by the smallest node
    for k in range(K):
        I = [i for i in range(n) if of[i] == k]
        assert len({int(gp[i]) for i in I}) == 1                                       # same GPU count (R1)
        for a, b in itertools.combinations(I, 2):
            for arr, e in ((comp, eps[0]), (mem, eps[1]), (intra, eps[2])):            # Eq. 1 and Eq. 2
                hi, lo = max(int(arr[a]), int(arr[b])), min(int(arr[a]), int(arr[b]))
                assert hi * 1000 <= lo * (1000 + e)
        for a in I:                                                                    # Eq. 3
            for b in I:
                if a == b:
                    continue
                for c in range(n):
                    if of[c] != k:
                        assert int(inter[a, b]) >= int(inter[a, c])


def eq3_holds(inter, members):
    n = inter.shape[0]
    ins = set(members)
    inner = [int(inter[a, b]) for a in members for b in members if a != b]
    leaving = [int(inter[a, c]) for a in members for c in range(n) if c not in ins]
    return not inner or not leaving or min(inner) >= max(leaving)


def homogeneous(prof, eps, members):
    gp, comp, mem, intra, _ = prof
    if len({int(gp[i]) for i in members}) != 1:
        return False
    return all(max(int(arr[i]) for i in members) * 1000 <= min(int(arr[i]) for i in members) * (1000 + e)
               for arr, e in ((comp, eps[0]), (mem, eps[1]), (intra, eps[2])))


@pytest.mark.parametrize("name,expect", [("C1", 2), ("C2", 2), ("C3", 4)])
def test_evaluation_clusters_of_table_3(name, expect):
    """C1 has two GPU types, C2 two, C3 four; PAPER.md:376-378 counts up to 4 islands on C3."""
    prof = gen.cluster_profile(name)
    of, ig, ic, bw = oracle.islands(*prof, *EPS)
    check_islands(prof, EPS, of)
    assert ig.size == expect
    assert int(ig.sum()) == int(prof[0].sum())
    if name == "C1":
        assert ig.tolist() == [16, 16] and ic.tolist() == [16000, 16000] and bw.tolist() == [[100, 25], [25, 100]]
    if name == "C3":
        assert ig.tolist() == [4, 4, 8, 4] and ic.tolist() == [16000, 16000, 32000, 80000]
        assert bw[0].tolist() == [32, 25, 25, 25]                                      # single-node island: its intra-node link


def test_hand_worked_three_nodes():
    """Three identical nodes.  Links 0<->1 at 100, everything touching node 2 at 10.
    Alone in the cluster: {0,1} merge first (linkage 100); then {0,1}+{2}: slowest inner link 10, nothing leaves -> valid:
    one island (Eq. 3 only compares with links LEAVING the island).
    With a fourth node of another type reachable at 25: {0,1} has inner 100 >= leaving max(10, 25); {0,1,2} would have inner
    10 < leaving 25 -> not an island.  Result {0,1}, {2}, {3}."""
    gp, comp, mem, intra = (np.array([4, 4, 4], np.int32), np.array([100] * 3, np.int32), np.array([16000] * 3, np.int32),
                            np.array([32] * 3, np.int32))
    inter = np.array([[0, 100, 10], [100, 0, 10], [10, 10, 0]], np.int32)
    of, ig, ic, bw = oracle.islands(gp, comp, mem, intra, inter, *EPS)
    assert of.tolist() == [0, 0, 0] and ig.tolist() == [12] and bw.tolist() == [[10]]
    gp4, comp4, mem4, intra4 = (np.append(gp, 8).astype(np.int32), np.append(comp, 300).astype(np.int32),
                                np.append(mem, 80000).astype(np.int32), np.append(intra, 600).astype(np.int32))
    inter4 = np.full((4, 4), 25, np.int32)
    inter4[:3, :3] = inter
    np.fill_diagonal(inter4, 0)
    of, ig, ic, bw = oracle.islands(gp4, comp4, mem4, intra4, inter4, *EPS)
    assert of.tolist() == [0, 0, 1, 2] and ig.tolist() == [8, 4, 8]
    assert bw.tolist() == [[100, 10, 25], [10, 32, 25], [25, 25, 600]]


def test_hand_worked_asymmetric_link():
    """Two identical nodes, a third of another type.  0->1 at 50 but 1->0 at 20; node 1 reaches the outsider at 30.
    Eq. 3 for {0,1} needs inter[1][0] = 20 >= inter[1][2] = 30: false -> three islands.  Raising 1->0 to 30 makes it one."""
    gp, comp, mem, intra = (np.array([4, 4, 2], np.int32), np.array([100, 100, 500], np.int32),
                            np.array([16000, 16000, 94000], np.int32), np.array([32, 32, 900], np.int32))
    inter = np.array([[0, 50, 10], [20, 0, 30], [10, 10, 0]], np.int32)
    assert oracle.islands(gp, comp, mem, intra, inter, *EPS)[0].tolist() == [0, 1, 2]
    inter[1, 0] = 30
    assert oracle.islands(gp, comp, mem, intra, inter, *EPS)[0].tolist() == [0, 0, 1]


def test_random_clusters_satisfy_the_definition_and_the_stop_condition():
    for seed in range(300):
        prof = gen.random_cluster(seed)
        of, ig, ic, bw = oracle.islands(*prof, *EPS)
        check_islands(prof, EPS, of)
        gp, comp, mem, intra, inter = prof
        K = ig.size
        members = [[i for i in range(gp.size) if of[i] == k] for k in range(K)]
        for k in range(K):
            assert ig[k] == sum(int(gp[i]) for i in members[k]) and ic[k] == min(int(mem[i]) for i in members[k])
        for j in range(K):
            for k in range(K):
                if j != k:
                    assert bw[j, k] == min(int(inter[a, b]) for a in members[j] for b in members[k])
        # greedy stop condition: two islands whose union is homogeneous and closed under Eq. 3 were in one step-2 group
        # only if the run-cutting separated them; islands that ARE mergeable must come from different groups, i.e. their
        # union must violate the run construction -- so at least no mergeable pair may exist among islands that share
        # exact compute, memory and intra-node values (those are never separated by a cut)
        for j, k in itertools.combinations(range(K), 2):
            same = all(len({int(arr[i]) for i in members[j] + members[k]}) == 1 for arr in (gp, comp, mem, intra))
            if same:
                assert not eq3_holds(inter, members[j] + members[k])


def test_limits_and_relabelling():
    # uniform links and wide tolerances: one island per GPU count
    gp = np.array([4, 4, 8, 8, 4], np.int32)
    comp = np.array([100, 140, 300, 310, 90], np.int32)
    mem = np.array([16000, 20000, 80000, 80000, 16000], np.int32)
    intra = np.array([32, 40, 600, 600, 32], np.int32)
    inter = np.full((5, 5), 50, np.int32)
    np.fill_diagonal(inter, 0)
    of, ig, _, _ = oracle.islands(gp, comp, mem, intra, inter, 1000, 1000, 1000)
    assert of.tolist() == [0, 0, 1, 1, 0] and ig.tolist() == [12, 16]
    # zero tolerances: only exactly equal nodes may share an island
    of0 = oracle.islands(gp, comp, mem, intra, inter, 0, 0, 0)[0]
    assert of0.tolist() == [0, 1, 2, 3, 4]
    # relabelling the nodes permutes the islands (same partition)
    for seed in range(40):
        prof = gen.random_cluster(900 + seed)
        n = prof[0].size
        perm = np.argsort(gen.urand(seed, 7, np.arange(n), 0, 1 << 20), kind="stable")
        p2 = tuple(a[perm] for a in prof[:4]) + (prof[4][np.ix_(perm, perm)],)
        of1 = oracle.islands(*prof, *EPS)[0]
        of2 = oracle.islands(*p2, *EPS)[0]
        part1 = {frozenset(int(i) for i in np.nonzero(of1 == k)[0]) for k in range(of1.max() + 1)}
        part2 = {frozenset(int(perm[i]) for i in np.nonzero(of2 == k)[0]) for k in range(of2.max() + 1)}
        ties = len(set(prof[4][~np.eye(n, dtype=bool)].tolist())) < n * (n - 1)
        assert part1 == part2 or ties          # (with tied links the greedy order may depend on the labels)
