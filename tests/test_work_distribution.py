"""Host-side checks (no GPU) of the tensor-core regimes' work distribution (csrc/gemm_i8_tcgen05.cuh
"Work distribution"), through vipir_testing_work_items: every (unit, chunk) item is visited exactly once;
within a unit chunks are visited in increasing order group by group; a group waits only for groups with
a lower id, and only after it has worked through every item another group may be waiting for -- the
argument for deadlock freedom; and the split removes the wave-quantisation loss."""
import itertools

import pytest

from paper_2606_11536_b200 import build, vipir


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


CASES = [(74, 256, 2), (148, 1024, 4), (74, 34, 2), (148, 3, 4), (7, 1, 5), (5, 23, 1), (148, 149, 2), (3, 10, 7),
         (74, 73, 3), (74, 75, 3), (1, 9, 4), (16, 16, 16), (148, 255, 8)]


@pytest.mark.parametrize("G,n_units,nc", CASES)
@pytest.mark.parametrize("split", [0, 1])
def test_every_item_once_and_in_order(G, n_units, nc, split):
    seen = {}
    per_group = []
    for g in range(G):
        items = vipir.testing_work_items(g, G, n_units, nc, split)
        per_group.append(items)
        for pos, (u, c, w) in enumerate(items):
            assert (u, c) not in seen, (u, c)
            assert u < n_units and c < nc
            seen[(u, c)] = (g, pos, w)
    assert len(seen) == n_units * nc
    for u in range(n_units):
        owners = [seen[(u, c)][0] for c in range(nc)]
        assert owners == sorted(owners), (u, owners)                 # later chunks on the same or a higher group
        for c in range(nc):
            g, pos, w = seen[(u, c)]
            first_of_group = c == 0 or seen[(u, c - 1)][0] != g
            assert w == (c > 0 and first_of_group), (u, c)           # waits exactly where another group's chunks precede
            if c > 0 and not first_of_group:
                assert seen[(u, c - 1)][1] == pos - 1                # same group: consecutive, in program order
    if not split:
        assert not any(w for _, _, w in itertools.chain.from_iterable(per_group))


@pytest.mark.parametrize("G,n_units,nc", CASES)
def test_waits_point_down_and_producers_come_first(G, n_units, nc):
    """Deadlock freedom: group g waits only on chunks owned by groups < g, and inside every group all items
    that are not waits-on-others ... precisely: an item some other group waits on (the last chunk a group
    holds of a unit continued elsewhere) is never preceded, in its own group, by a waiting item."""
    owner = {}
    order = {}
    for g in range(G):
        for pos, (u, c, w) in enumerate(vipir.testing_work_items(g, G, n_units, nc, 1)):
            owner[(u, c)] = g
            order[(u, c)] = (pos, w)
    for (u, c), g in owner.items():
        pos, w = order[(u, c)]
        if w:
            assert owner[(u, c - 1)] < g
    # simulate: a group advances through its list; a waiting item needs chunk c-1 of its unit done
    lists = [vipir.testing_work_items(g, G, n_units, nc, 1) for g in range(G)]
    ptr = [0] * G
    done = set()
    progress = True
    while progress:
        progress = False
        for g in range(G):                      # any fair schedule works; also try only-one-group-at-a-time below
            while ptr[g] < len(lists[g]):
                u, c, w = lists[g][ptr[g]]
                if w and (u, c - 1) not in done:
                    break
                done.add((u, c))
                ptr[g] += 1
                progress = True
    assert len(done) == n_units * nc            # nobody is stuck
    # worst case for residency: only groups 0..k are running for any k (tickets are handed out in start order)
    for k in range(G):
        ptr = [0] * (k + 1)
        done = set()
        for g in range(k + 1):                  # lower tickets never depend on higher ones: each finishes in turn
            for u, c, w in lists[g]:
                assert not w or (u, c - 1) in done, (k, g, u, c)
                done.add((u, c))


def test_split_balances_the_last_round():
    # BASELINE.json configs[4]: 256 units of 2 chunks on 74 CTA pairs: 7 chunk-items per group instead of 8
    G, n_units, nc = 74, 256, 2
    assert max(len(vipir.testing_work_items(g, G, n_units, nc, 1)) for g in range(G)) == 7
    assert max(len(vipir.testing_work_items(g, G, n_units, nc, 0)) for g in range(G)) == 8
    # full rounds are round-robin over units (sibling N tiles run side by side)
    assert [u for u, c, w in vipir.testing_work_items(5, G, n_units, nc, 1)][:6] == [5, 5, 79, 79, 153, 153]
