"""Host-side model of the attention kernel's K/V ring protocol (paper_2607_07724_b200/csrc/attn.cu).

The sparse attention kernel streams K and V tiles through shared-memory rings guarded by mbarriers
that are waited on BY PARITY.  A parity wait for "occupant r of this slot has landed" succeeds when
the number of completed phases c satisfies c = r + 1 (mod 2) -- so it is only sound if c can never be
r - 1 when the wait is posted, i.e. if the slot's previous occupant was consumed by the SAME thread.
The first two-thread build (QK and PV issued by different threads, one shared ring) violated that and
produced wrong bits / lost arrivals on the GPU.  This file is a small randomised discrete-event model
of producer / QK thread / PV thread / softmax with parity-waited barriers.  It must (a) find the bug
in the shared-ring design and (b) find nothing -- no stale tile, no deadlock -- in the designs the
kernel uses: one ring per consumer (two issuing threads) and one ring, one consumer.
No GPU, no oracle: host logic only.
"""
import random

import pytest


class Bar:
    """mbarrier with an arrival count of one: `c` = completed phases; waits are by parity."""

    def __init__(self):
        self.c = 0

    def passes(self, r):          # wait for the completion of phase r, expressed as parity r & 1
        return (self.c & 1) != (r & 1)


def simulate(n, ns_k, ns_v, shared, two_threads, seed, max_steps=200000):
    """Returns None if all n iterations complete with every MMA reading the tile it expects, else a
    string describing the first violation ("stale ..." or "deadlock")."""
    rng = random.Random(seed)
    ahead = 2 if two_threads else 1
    # ring position (= load order) of K(i), V(j); one shared sequence or two separate ones
    order = [("K", i) for i in range(min(ahead, n))]
    for j in range(n):
        if j + ahead < n:
            order.append(("K", j + ahead))
        order.append(("V", j))
    if shared:
        ns = ns_k + ns_v
        seq = {tile: p for p, tile in enumerate(order)}
        slot = {tile: p % ns for tile, p in seq.items()}
        occ = {tile: p // ns for tile, p in seq.items()}
        nslots = ns
    else:
        slot, occ = {}, {}
        for t, i in order:
            if t == "K":
                slot[(t, i)], occ[(t, i)] = i % ns_k, i // ns_k
            else:
                slot[(t, i)], occ[(t, i)] = ns_k + i % ns_v, i // ns_v
        nslots = ns_k + ns_v
    full = [Bar() for _ in range(nslots)]
    empty = [Bar() for _ in range(nslots)]
    content = [None] * nslots            # tile currently in the slot's bytes
    inflight = []                        # (slot, tile, remaining delay)
    s_full, s_free = [Bar(), Bar()], [Bar(), Bar()]
    p_full, o_done = Bar(), Bar()
    st = dict(load=0, qk=0, pv=0, sm=0, sm_read=False, qk_stage=0, pv_stage=0)

    def step_producer():
        if st["load"] >= len(order):
            return False
        tile = order[st["load"]]
        s, r = slot[tile], occ[tile]
        if r > 0 and not empty[s].passes(r - 1):
            return False
        inflight.append([s, tile, rng.randint(1, 80)])   # TMA latency: up to several iterations
        st["load"] += 1
        return True

    def issue(tile):
        """The MMA reads the slot now: it must hold `tile`; the commit then frees the slot."""
        sl = slot[tile]
        if content[sl] != tile:
            return f"stale: MMA for {tile} read slot {sl} holding {content[sl]}"
        empty[sl].c += 1                 # tcgen05.commit -> kv_empty (instantaneous in the model)
        return True

    # Waits are posted one after the other and are STICKY, as in the kernel: a wait that has passed is
    # not evaluated again when the thread later blocks on its next barrier.
    def step_qk():
        i = st["qk"]
        if i >= n:
            return False
        if not two_threads and i >= 2 and st["pv"] < i - 1:
            return False                 # single thread: QK(i) comes after PV(i-2) in program order
        if st["qk_stage"] == 0:
            if not full[slot[("K", i)]].passes(occ[("K", i)]):
                return False
            st["qk_stage"] = 1
        if i >= 2 and not s_free[i & 1].passes((i - 2) >> 1):
            return False
        r = issue(("K", i))
        if r is not True:
            return r
        s_full[i & 1].c += 1
        st["qk"] += 1
        st["qk_stage"] = 0
        return True

    def step_pv():
        j = st["pv"]
        if j >= n:
            return False
        if not two_threads and st["qk"] < min(j + 2, n):
            return False                 # single thread: QK(j+1) is issued before PV(j)
        if st["pv_stage"] == 0:
            if not full[slot[("V", j)]].passes(occ[("V", j)]):
                return False
            st["pv_stage"] = 1
        if not p_full.passes(j):
            return False
        r = issue(("V", j))
        if r is not True:
            return r
        o_done.c += 1
        st["pv"] += 1
        st["pv_stage"] = 0
        return True

    def step_softmax():
        j = st["sm"]
        if j >= n:
            return False
        if not st["sm_read"]:
            if not s_full[j & 1].passes(j >> 1):
                return False
            s_free[j & 1].c += 1
            st["sm_read"] = True
            return True
        if j > 0 and not o_done.passes(j - 1):
            return False
        p_full.c += 1
        st["sm"] += 1
        st["sm_read"] = False
        return True

    actors = [step_producer, step_qk, step_pv, step_softmax]
    for _ in range(max_steps):
        progressed = False
        for item in inflight[:]:         # TMA landings
            item[2] -= 1
            if item[2] <= 0:
                content[item[0]] = item[1]
                full[item[0]].c += 1
                inflight.remove(item)
                progressed = True
        rng.shuffle(actors)
        for a in actors:
            if rng.random() < 0.7:
                r = a()
                if isinstance(r, str):
                    return r
                progressed = progressed or bool(r)
        if st["pv"] >= n and st["sm"] >= n:
            return None
        if not progressed and not inflight:
            # one deterministic sweep before declaring a deadlock (the random skips may have idled)
            if not any(a() for a in (step_producer, step_qk, step_pv, step_softmax)):
                return f"deadlock at load={st['load']} qk={st['qk']} pv={st['pv']} sm={st['sm']}"
    return "no termination"


def test_shared_ring_with_two_consumers_is_caught():
    """The design of the racy build: the model must expose it (stale tile or deadlock)."""
    bad = [simulate(n, 3, 2, shared=True, two_threads=True, seed=s) for n in (8, 32) for s in range(40)]
    assert any(b is not None for b in bad)


@pytest.mark.parametrize("ns_k,ns_v", [(3, 2), (2, 2), (4, 4), (2, 3), (1, 1)])
def test_one_ring_per_consumer_is_sound(ns_k, ns_v):
    for n in list(range(1, 12)) + [32, 64, 65]:
        for seed in range(12):
            assert simulate(n, ns_k, ns_v, shared=False, two_threads=True, seed=seed) is None, (n, seed)


@pytest.mark.parametrize("ns", [2, 4, 5, 8])
def test_single_consumer_shared_ring_is_sound(ns):
    for n in list(range(1, 12)) + [32, 65]:
        for seed in range(12):
            assert simulate(n, ns, 0, shared=True, two_threads=False, seed=seed) is None, (n, seed)
