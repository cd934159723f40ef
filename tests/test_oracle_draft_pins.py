"""Pins of the draft-side level expansion of the oracle (NEXT-4): a hand example with exactly representable scores,
brute force, and the invariant that the tree built level by level has the path scores Eq. 5 gives (O1, pinned
separately), so the expansion's running scores are the gate's path scores bit for bit."""
import numpy as np
import pytest

from oracle import echo_oracle as orc


def test_hand_example():
    # k = 2.  level 0: virtual root 0.0, children logq (-0.5, -0.25) -> order by score: child 1 (-0.25), child 0 (-0.5)
    l0 = orc.draft_expand(0, 2, np.zeros((1, 1), np.float32), np.asarray([[[-0.5, -0.25]]], np.float32),
                          np.asarray([[[7, 9]]], np.int32))
    assert l0["sel_parent"].tolist() == [[-1, -1]] and l0["token"].tolist() == [[9, 7]]
    assert l0["score"].tolist() == [[-0.25, -0.5]]
    # level 1: parents (-0.25, -0.5); children of slot 0: (-1.0, -0.125), of slot 1: (-0.125, -2.0)
    # scores: (0,0) -1.25, (0,1) -0.375, (1,0) -0.625, (1,1) -2.5 -> keep (0,1) then (1,0)
    l1 = orc.draft_expand(1, 2, l0["score"], np.asarray([[[-1.0, -0.125], [-0.125, -2.0]]], np.float32),
                          np.asarray([[[1, 2], [3, 4]]], np.int32))
    assert l1["sel_parent"].tolist() == [[0, 1]] and l1["token"].tolist() == [[2, 3]]
    assert l1["score"].tolist() == [[-0.375, -0.625]] and l1["logq"].tolist() == [[-0.125, -0.125]]
    # ties: equal scores keep (parent slot, child rank) order
    t = orc.draft_expand(1, 2, np.asarray([[-0.5, -0.5]], np.float32), np.full((1, 2, 2), -0.5, np.float32),
                         np.asarray([[[1, 2], [3, 4]]], np.int32))
    assert t["sel_parent"].tolist() == [[0, 0]] and t["token"].tolist() == [[1, 2]]


@pytest.mark.parametrize("seed,k", [(0, 8), (1, 10), (2, 16), (3, 3)])
def test_levels_build_a_tree_whose_path_scores_match(seed, k):
    rng = np.random.default_rng(seed)
    R, L = 5, 4
    parent, logq_all, score_all = [[] for _ in range(R)], [[] for _ in range(R)], [[] for _ in range(R)]
    ps = np.zeros((R, 1), np.float32)
    for lvl in range(L):
        kp = 1 if lvl == 0 else k
        cl = np.log(rng.dirichlet(np.full(k, 0.3), size=(R, kp)) + 1e-9).astype(np.float32)
        ct = rng.integers(0, 1000, (R, kp, k)).astype(np.int32)
        out = orc.draft_expand(lvl, k, ps, cl, ct)
        for i in range(R):
            s = out["score"][i]
            assert all(s[j] >= s[j + 1] for j in range(k - 1))                       # kept in score order
            allc = sorted((np.float32(np.float32(ps[i, p]) + cl[i, p, c]) for p in range(kp) for c in range(k)), reverse=True)
            assert [float(x) for x in s] == [float(x) for x in allc[:k]]              # the k best, brute force
            for j in range(k):
                parent[i].append(-1 if lvl == 0 else (lvl - 1) * k + int(out["sel_parent"][i, j]))
                logq_all[i].append(out["logq"][i, j]); score_all[i].append(out["score"][i, j])
        ps = out["score"]
    offs = np.arange(R + 1, dtype=np.int32) * (L * k)
    S, depth = orc.path_scores(offs, np.concatenate([np.asarray(p, np.int32) for p in parent]),
                               np.concatenate([np.asarray(q, np.float32) for q in logq_all]))
    assert np.array_equal(S, np.concatenate([np.asarray(s, np.float32) for s in score_all]))
    assert depth.reshape(R, L, k).transpose(1, 0, 2).reshape(L, -1).tolist() == [[l] * (R * k) for l in range(L)]
