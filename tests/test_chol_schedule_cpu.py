"""Host logic of rows c, d1: the static schedule of the tiled Cholesky task graph
(csrc/chol_schedule.cu) is executed here by a plain simulator of the kernel's flag protocol -- every CTA runs
its list in order, a task completes only when the flags of all its operands are set -- and must (i) never
deadlock, (ii) produce every tile of L and of the block-diagonal inverse exactly once, (iii) apply the k-updates
of every tile in ascending order without a gap (the property that makes the result independent of the CTA count),
(iv) keep the chain tasks on the first list in column order.  No GPU, no arithmetic."""
import numpy as np
import pytest

import paper_1608_04329_b200 as hsp


def simulate(nt, sb, K):
    rows, makespan = hsp.chol_schedule(nt, sb, K)
    lists = [[tuple(int(v) for v in r[1:]) for r in rows if r[0] == k] for k in range(K)]
    assert sum(len(l) for l in lists) == len(rows)
    doneL, doneB, doneP = set(), set(), set()
    applied = {}                       # (kind, i, j) -> number of k-updates applied so far (ascending, no gap)
    parked = {}                        # slot -> (kind, i, j)
    pos = [0] * K
    total, done = len(rows), 0
    while done < total:
        progress = False
        for k in range(K):
            while pos[k] < len(lists[k]):
                typ, i, j, kb, ke, si, so = lists[k][pos[k]]
                if typ == 0:
                    need = [("L", i, q) for q in range(kb, ke)] + ([("L", j, q) for q in range(kb, ke)] if i != j else [])
                    if so < 0 and i != j:
                        need.append(("L", j, j))
                elif typ == 1:          # inverse tile W(j,i), i < j
                    need = [("L", j, q) for q in range(kb, ke)] + [("L", i, i) if q == i else ("B", i, q) for q in range(kb, ke)] + [("L", j, j)]
                elif typ == 2:
                    assert k == 0
                    need = []
                elif typ == 3:
                    assert k == 0
                    need = [("L", j, j)]
                else:
                    assert k == 0 and typ == 4
                    need = [("L", i, j)]
                ok = all((t[1], t[2]) in (doneL if t[0] == "L" else doneB) for t in need)
                if si >= 0 and si not in doneP:
                    ok = False
                if not ok:
                    break
                # bookkeeping of the k-updates
                if typ in (0, 1):
                    key = ("L" if typ == 0 else "B", i, j)
                    first = 0 if typ == 0 else i
                    if si >= 0:
                        assert parked.pop(si) == key
                    assert applied.get(key, first) == kb, (key, applied.get(key), kb)
                    applied[key] = ke
                    if so >= 0:
                        assert so not in parked and so not in doneP
                        parked[so] = key; doneP.add(so)
                    else:
                        assert ke == (j if typ == 0 else j), (key, ke)
                        (doneL if typ == 0 else doneB).add((i, j))
                elif typ == 2:
                    key = ("L", j, j)
                    # A_jj arrives through SYRK(j-1) (or is the Q tile for j = 0)
                    assert applied.get(key, 0) == j
                    assert (j, j) not in doneL
                    doneL.add((j, j))
                elif typ == 3:          # TRSM(j): tile (j+1, j) from its parked accumulator (all k < j applied)
                    key = ("L", i, j)
                    assert i == j + 1
                    if si >= 0:
                        assert parked.pop(si) == key
                    assert applied.get(key, 0) == j
                    doneL.add((i, j))
                else:                   # SYRK(j): A(j+1,j+1) -= L(j+1,j) L(j+1,j)^T on top of the parked k < j
                    key = ("L", i, i)
                    assert i == j + 1
                    if si >= 0:
                        assert parked.pop(si) == key
                    assert applied.get(key, 0) == j
                    applied[key] = j + 1
                pos[k] += 1; done += 1; progress = True
        assert progress, f"deadlock at nt={nt} sb={sb} K={K}: {done}/{total} tasks"
    assert not parked
    assert doneL == {(i, j) for i in range(nt) for j in range(i + 1)}
    assert doneB == {(i, j) for j in range(nt) for i in range(j) if i // sb == j // sb}
    chain = [t for t in lists[0] if t[0] >= 2]
    if chain:
        assert lists[0] == chain and all(not any(t[0] >= 2 for t in l) for l in lists[1:])
        assert [t[2] for t in chain if t[0] == 2] == list(range(nt))
    return makespan


@pytest.mark.parametrize("nt", [1, 2, 3, 5, 8, 16, 21, 32])
def test_schedule_is_deadlock_free_complete_and_ordered(nt):
    sb = nt if nt <= 20 else 8
    spans = []
    for K in (1, 2, 3, 4, 8, 16, 20, 48, 148):
        if K > nt * nt:
            continue
        spans.append((K, simulate(nt, sb, K)))
    # the cost-model makespan does not get worse with more CTAs (beyond the chain bound it stays flat)
    for (k0, m0), (k1, m1) in zip(spans[1:], spans[2:]):
        assert m1 <= m0 * 1.05, spans


def test_schedule_c4_shape_and_small_superblocks():
    simulate(63, 8, 104)
    simulate(63, 8, 148)
    simulate(9, 2, 5)
    simulate(12, 1, 7)           # no inverse tiles off the diagonal at all


def test_schedule_very_large_problem_round_robin():
    """nt > 96 (p > 6144): the greedy search is skipped, tasks are dealt round-robin in id order, no chain CTA."""
    rows, _ = hsp.chol_schedule(100, 8, 37)
    assert not (rows[:, 1] >= 2).any()
    simulate(100, 8, 37)


def test_schedule_rejects_bad_arguments():
    assert hsp.lib().hsp_dbg_chol_schedule(0, 1, 1, None, 0, None) == -1
    assert hsp.lib().hsp_dbg_chol_schedule(2, 1, 5, None, 0, None) == -1
