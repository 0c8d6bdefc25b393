"""Pins of the oracle's topology-aware replica placement (reading R38; "place the k replicas on
nodes under k distinct switches or racks, ensuring that a single infrastructure event affects at most one copy of any
given shard"): brute force over every failure-domain map of small rings, the paper's own motivating case (owner and
replica under one switch), the special case that reduces to the plain ring (R25), and recovery of a whole failed
domain on the byte-level ring oracle.  CPU only."""
import itertools

import numpy as np
import pytest

from oracle import oracle as O
from oracle import ring as R
from paper_2607_01646_b200 import workloads as W

from test_oracle_shard import HP, tbits


def brute_force_holders(domains, r, k):
    """Lexicographically smallest tuple of ring distances whose ranks sit in pairwise distinct domains, all
    different from the owner's — by enumeration."""
    D = len(domains)
    best = None
    for dist in itertools.combinations(range(1, D), k):
        doms = [domains[r]] + [domains[(r + j) % D] for j in dist]
        if len(set(doms)) == k + 1:
            best = dist
            break                                   # combinations() yields tuples in lexicographic order
    return None if best is None else [(r + j) % D for j in best]


@pytest.mark.parametrize("D", [2, 3, 4, 5, 6])
def test_nearest_admissible_ranks_by_brute_force_over_every_domain_map(D):
    for domains in itertools.product(range(min(D, 4)), repeat=D):
        n_dom = len(set(domains))
        for k in range(1, min(D, 4)):
            for r in range(D):
                want = brute_force_holders(domains, r, k)
                if n_dom < k + 1:
                    assert want is None
                    with pytest.raises(O.OracleError):
                        R.holders_topology_aware(domains, r, k)
                else:
                    assert want is not None and R.holders_topology_aware(domains, r, k) == want, (domains, r, k)
            if n_dom >= k + 1:
                place = R.placement(D, k, domains)
                # "a single infrastructure event affects at most one copy of any given shard"
                assert R.max_copies_in_one_domain(domains, place) == 1
                for d in set(domains):
                    assert R.recoverable_with(place, [q for q in range(D) if domains[q] == d])


def test_the_papers_motivating_case_owner_and_replica_under_one_switch():
    # two ranks per switch, k = 1: on the plain ring rank 2i's replica sits on rank 2i+1 — the same switch
    D, k = 8, 1
    domains = [q // 2 for q in range(D)]
    plain = R.placement(D, k)
    assert R.max_copies_in_one_domain(domains, plain) == 2
    assert not R.recoverable_with(plain, [0, 1])                    # switch 0 fails: rank 0's shard is gone
    aware = R.placement(D, k, domains)
    assert aware[0] == [2] and aware[1] == [2] and aware[7] == [0]
    assert R.max_copies_in_one_domain(domains, aware) == 1
    for d in range(D // 2):
        assert R.recoverable_with(aware, [2 * d, 2 * d + 1])
    # k = 2 survives any TWO switches failing at once only if the copies sit under three distinct switches
    aware2 = R.placement(D, 2, domains)
    assert R.max_copies_in_one_domain(domains, aware2) == 1
    for a, b in itertools.combinations(range(D // 2), 2):
        assert R.recoverable_with(aware2, [2 * a, 2 * a + 1, 2 * b, 2 * b + 1])
    assert not R.recoverable_with(R.placement(D, 2), [0, 1, 2, 3])   # plain ring, k = 2: rank 0, 1, 2 all under switches 0, 1


@pytest.mark.parametrize("D,k", [(3, 1), (5, 2), (6, 4)])
def test_one_rank_per_domain_is_the_plain_ring(D, k):
    domains = [10 + q for q in range(D)]
    assert R.placement(D, k, domains) == R.placement(D, k)
    assert R.recoverable_with(R.placement(D, k), [0]) == R.recoverable(D, k, [0])
    for failed in itertools.chain.from_iterable(itertools.combinations(range(D), n) for n in range(D + 1)):
        assert R.recoverable_with(R.placement(D, k), failed) == R.recoverable(D, k, failed)


def test_a_whole_failed_domain_is_recovered_byte_for_byte_and_resumes():
    D, k = 6, 2
    domains = [0, 0, 1, 1, 2, 2]
    wl = W.tiny_workload([3000, 77], dp_size=D)
    ring = R.OracleRing(wl.layout(), D, k, chunk_bytes=4096, domains=domains)
    ref = R.OracleRing(wl.layout(), D, k, chunk_bytes=4096, domains=domains)
    assert ring.place == [[2, 4], [2, 4], [4, 0], [4, 0], [0, 2], [0, 2]]
    assert sorted(h for (h, _) in ring.recv) == [0] * 4 + [2] * 4 + [4] * 4    # ranks 1, 3, 5 hold nothing
    segs = [(tid, off, ln) for tid, _, off, ln in ring.shards[0].segments]
    gs = {t: [tbits(W.gen_grads(wl, segs, ring.shards[0].n_padded, t, 20 + r)) for r in range(D)] for t in range(1, 7)}
    for rg in (ring, ref):
        for r, o in enumerate(rg.shards):
            o.set_state(W.init_params(o.n, o.n_padded, 50 + r).numpy())
    for t in range(1, 5):
        for rg in (ring, ref):
            for r, o in enumerate(rg.shards):
                o.step(gs[t][r], **HP, step=t)
                o.snapshot()
                rg.replicate(r)
    for r in range(D):                                   # received bytes == the owner's local slot (R26)
        for h in ring.place[r]:
            assert np.array_equal(ring.recv[(h, r)][0], ring.shards[r].replica[0])
    ring.fail([2, 3])                                    # switch 1 goes down with both of its ranks
    assert ring.recover(2) == 4 and ring.recover(3) == 4
    for t in (5, 6):
        for rg in (ring, ref):
            for r, o in enumerate(rg.shards):
                o.step(gs[t][r], **HP, step=t)
    for a, b in zip(ring.shards, ref.shards):
        assert a.p.tobytes() == b.p.tobytes() and a.m.tobytes() == b.m.tobytes() and a.v.tobytes() == b.v.tobytes()
    # owner + both holders in ONE failure event: lost
    ring.fail([0, 2, 4])
    with pytest.raises(O.OracleError):
        ring.recover(0)
