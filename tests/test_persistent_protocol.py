"""Host-side model of the persistent attention kernel's protocol (attn64p_kernel, csrc/attn.cu).

In the persistent kernel every role -- scheduler / list builder, TMA producer, QK thread, PV thread, softmax
warps -- runs through the CTA's work items on its own, and all hand-offs are mbarriers waited on BY PARITY with
phases derived from running counters (iterations, non-empty items, ring positions).  Such a wait is sound only
if, whenever it is polled for phase r, the barrier has completed r or r + 1 phases -- never r + 2 (the waiter
would hang) and never r - 1 (it would pass early).  This file is a randomised discrete-event model of that
protocol: asynchronous TMA landings and MMA completions (in order per issuing thread), items of random length
including empty ones, random interleavings.  It checks
  * no deadlock, and the r / r + 1 rule at every poll of every barrier,
  * every buffer hand-off: S read before it is overwritten, P consumed before it is overwritten, O read by the
    epilogue before the next item's first PV, the Q buffer written only after the QKs that read it, the right Q
    tile / K / V tile under every MMA, list buffers rewritten only after every consumer left the item,
and, as a control, that the variant in which EMPTY items also post q_full (the first draft of the design) is
caught.  No GPU, no oracle: host logic only.
"""
import random

import pytest


class Hazard(Exception):
    pass


class Bar:
    def __init__(self, name, count=1):
        self.name, self.count, self.c, self.pending = name, count, 0, 0

    def arrive(self):
        self.pending += 1
        if self.pending == self.count:
            self.pending = 0
            self.c += 1


def wait(bar, r):
    """parity wait for the completion of phase r (0-based), polled until it passes"""
    while True:
        if bar.c not in (r, r + 1):
            raise Hazard(f"{bar.name}: polled for phase {r} with {bar.c} phases complete")
        if bar.c == r + 1:
            return
        yield False


class Model:
    def __init__(self, lengths, nsk, nsv, seed, pieces=2, empty_items_post_q=False):
        self.rng = random.Random(seed)
        self.lengths, self.nsk, self.nsv, self.pieces = lengths, nsk, nsv, pieces
        self.bad_empty = empty_items_post_q
        B = Bar
        self.q_full, self.o_free = B("q_full"), B("o_free")
        self.p_full = [B("p_full0"), B("p_full1")]
        self.s_full = [B("s_full0"), B("s_full1")]
        self.s_free = [B("s_free0"), B("s_free1")]
        self.o_done = [B("o_done0"), B("o_done1")]
        self.list_full = [B("list_full0"), B("list_full1")]
        self.list_free = [B("list_free0", 4), B("list_free1", 4)]   # softmax, producer, QK, PV
        self.kv_full = [B(f"kv_full{i}") for i in range(nsk + nsv)]
        self.kv_empty = [B(f"kv_empty{i}") for i in range(nsk + nsv)]
        self.list = [None, None]          # (item index or -1, length)
        self.ring = [None] * (nsk + nsv)  # tile in the slot's bytes
        self.s_content, self.s_read = [None, None], [None, None]
        self.p_content = [None, None]
        self.q_content = [None, None]     # non-empty item index whose Q tile is in the buffer
        self.qk_done_item = -1            # last non-empty item all of whose QKs completed
        self.pv_done = -1                 # last completed PV (running iteration)
        self.epilogue_read = -1           # last non-empty item whose O the epilogue has read
        self.left = dict(sm=-1, prod=-1, qk=-1, pv=-1)   # last item each consumer has left
        self.events = []                  # [time, fn]
        self.now = 0
        self.last_done = dict(qk=0, pv=0)

    def after(self, delay, fn):
        self.events.append([self.now + delay, fn])

    def mma(self, who, fn):
        """completion of an MMA batch: in order per issuing thread"""
        t = max(self.last_done[who], self.now + self.rng.randint(1, 30))
        self.last_done[who] = t
        self.events.append([t, fn])

    # ---- roles -------------------------------------------------------------------------------------
    def scheduler(self):
        for n in range(len(self.lengths) + 1):
            buf = n & 1
            if n >= 2:
                yield from wait(self.list_free[buf], (n - 2) >> 1)
                if min(self.left.values()) < n - 2:
                    raise Hazard(f"list[{buf}] rewritten for item {n} while a consumer is still in item {n - 2}")
            yield True                    # fetch + compaction take a while
            self.list[buf] = (-1, 0) if n == len(self.lengths) else (n, self.lengths[n])
            self.list_full[buf].arrive()
            if n == len(self.lengths):
                return

    def producer(self):
        gk = gv = 0
        for n in range(len(self.lengths) + 1):
            buf = n & 1
            yield from wait(self.list_full[buf], n >> 1)
            item, n_it = self.list[buf]
            if item < 0:
                return

            def load(kind, idx, slot, use):
                yield from wait(self.kv_empty[slot], use - 1) if use > 0 else iter(())
                tile = (kind, item, idx)

                def land(slot=slot, tile=tile):
                    self.ring[slot] = tile
                    self.kv_full[slot].arrive()
                self.after(self.rng.randint(1, 60), land)
                yield True
            for i in range(min(2, n_it)):
                yield from load("K", i, gk % self.nsk, gk // self.nsk)
                gk += 1
            for j in range(n_it):
                if j + 2 < n_it:
                    yield from load("K", j + 2, gk % self.nsk, gk // self.nsk)
                    gk += 1
                yield from load("V", j, self.nsk + gv % self.nsv, gv // self.nsv)
                gv += 1
            self.left["prod"] = n
            self.list_free[buf].arrive()

    def qk(self):
        gi = gk = ne = 0
        for n in range(len(self.lengths) + 1):
            buf = n & 1
            yield from wait(self.list_full[buf], n >> 1)
            item, n_it = self.list[buf]
            if item < 0:
                return
            self.left["qk"] = n
            self.list_free[buf].arrive()
            if n_it == 0 and not self.bad_empty:
                continue
            yield from wait(self.q_full, ne)
            qb = ne & 1
            me = ne
            ne += 1
            for i in range(n_it):
                slot = gk % self.nsk
                yield from wait(self.kv_full[slot], gk // self.nsk)
                if gi >= 2:
                    yield from wait(self.s_free[gi & 1], (gi - 2) >> 1)
                    if self.s_read[gi & 1] != gi - 2:
                        raise Hazard(f"QK({gi}) overwrites S before softmax({gi - 2}) read it")
                if self.ring[slot] != ("K", item, i):
                    raise Hazard(f"QK({gi}) read slot {slot} holding {self.ring[slot]}")
                if self.q_content[qb] != me:
                    raise Hazard(f"QK of item #{me} read Q buffer {qb} holding #{self.q_content[qb]}")

                def done(gi=gi, slot=slot, last=(i == n_it - 1), me=me):
                    self.s_content[gi & 1] = gi
                    self.kv_empty[slot].arrive()
                    self.s_full[gi & 1].arrive()
                    if last:
                        self.qk_done_item = me
                self.mma("qk", done)
                gi += 1
                gk += 1
                yield True

    def pv(self):
        gj = gv = ne = 0
        for n in range(len(self.lengths) + 1):
            buf = n & 1
            yield from wait(self.list_full[buf], n >> 1)
            item, n_it = self.list[buf]
            if item < 0:
                return
            self.left["pv"] = n
            self.list_free[buf].arrive()
            if n_it == 0:
                continue
            if ne > 0:
                yield from wait(self.o_free, ne - 1)
                if self.epilogue_read != ne - 1:
                    raise Hazard(f"first PV of item #{ne} overwrites O before epilogue #{ne - 1} read it")
            ne += 1
            for jj in range(n_it):
                slot = self.nsk + gv % self.nsv
                yield from wait(self.kv_full[slot], gv // self.nsv)
                yield from wait(self.p_full[gj & 1], gj >> 1)
                if self.ring[slot] != ("V", item, jj):
                    raise Hazard(f"PV({gj}) read slot {slot} holding {self.ring[slot]}")
                if self.p_content[gj & 1] != gj:
                    raise Hazard(f"PV({gj}) read P buffer holding {self.p_content[gj & 1]}")

                def done(gj=gj, slot=slot):
                    self.pv_done = gj
                    self.kv_empty[slot].arrive()
                    self.o_done[gj & 1].arrive()
                self.mma("pv", done)
                gj += 1
                gv += 1
                yield True

    def softmax(self):
        gj = ne = 0
        q_ready = False

        def put_q(k):
            if self.qk_done_item < k - 2:
                raise Hazard(f"Q buffer {k & 1} rewritten for item #{k} before the QKs of #{k - 2} completed")
            self.q_content[k & 1] = k
            self.q_full.arrive()
        for n in range(len(self.lengths) + 1):
            buf = n & 1
            yield from wait(self.list_full[buf], n >> 1)
            item, n_it = self.list[buf]
            if item < 0:
                return
            if n_it == 0:
                if self.bad_empty:        # the first draft: empty items take part in the q_full sequence
                    self.q_content[ne & 1] = ne
                    self.q_full.arrive()
                    ne += 1
                self.left["sm"] = n
                self.list_free[buf].arrive()
                yield True
                continue
            if not q_ready:
                yield True                # global-memory latency of the tile
                put_q(ne)
            q_ready = False
            ne += 1
            pieces = False
            for j in range(n_it):
                if j == n_it - self.pieces and n_it >= self.pieces:
                    nb = (n + 1) & 1
                    lf = self.list_full[nb]
                    if lf.c == ((n + 1) >> 1) + 1 and self.list[nb][0] >= 0 and self.list[nb][1] > 0:
                        pieces = True
                        if self.qk_done_item < ne - 2:
                            raise Hazard(f"first Q piece for item #{ne} before the QKs of #{ne - 2} completed")
                if gj >= 2:
                    yield from wait(self.s_full[gj & 1], gj >> 1)
                    yield from wait(self.o_done[gj & 1], (gj - 2) >> 1)
                else:
                    yield from wait(self.s_full[gj & 1], gj >> 1)
                if self.s_content[gj & 1] != gj:
                    raise Hazard(f"softmax({gj}) read S holding {self.s_content[gj & 1]}")
                self.s_read[gj & 1] = gj
                self.s_free[gj & 1].arrive()
                yield True
                if gj >= 2 and self.pv_done < gj - 2:
                    raise Hazard(f"P({gj}) overwrites P({gj - 2}) before its PV completed")
                self.p_content[gj & 1] = gj
                self.p_full[gj & 1].arrive()
                gj += 1
                yield True
            # item boundary
            if pieces:
                self.q_content[ne & 1] = ne
                self.q_full.arrive()
                q_ready = True
            else:
                nb = (n + 1) & 1
                yield from wait(self.list_full[nb], (n + 1) >> 1)
                if self.list[nb][0] >= 0 and self.list[nb][1] > 0:
                    yield True
                    put_q(ne)
                    q_ready = True
            yield from wait(self.o_done[(gj - 1) & 1], (gj - 1) >> 1)
            if self.pv_done < gj - 1:
                raise Hazard("epilogue before the last PV completed")
            self.epilogue_read = ne - 1
            self.o_free.arrive()
            self.left["sm"] = n
            self.list_free[buf].arrive()
            yield True

    # ---- driver ------------------------------------------------------------------------------------
    def run(self, max_steps=400000):
        actors = {k: getattr(self, k)() for k in ("scheduler", "producer", "qk", "pv", "softmax")}
        idle = 0
        for _ in range(max_steps):
            self.now += 1
            progressed = False
            for ev in sorted([e for e in self.events if e[0] <= self.now], key=lambda e: e[0]):
                self.events.remove(ev)
                ev[1]()
                progressed = True
            names = list(actors)
            self.rng.shuffle(names)
            for k in names:
                if self.rng.random() < 0.6:
                    try:
                        progressed = bool(next(actors[k])) or progressed
                    except StopIteration:
                        del actors[k]
                        progressed = True
            if not actors:
                return None
            idle = 0 if (progressed or self.events) else idle + 1
            if idle > 200:
                return "deadlock with " + ", ".join(sorted(actors))
        return "no termination"


def simulate(lengths, nsk, nsv, seed, **kw):
    try:
        return Model(lengths, nsk, nsv, seed, **kw).run()
    except Hazard as e:
        return str(e)


def _lengths(rng, n_items, p_empty):
    out = []
    for _ in range(n_items):
        out.append(0 if rng.random() < p_empty else rng.choice([1, 1, 2, 3, 4, 5, 8, 13]))
    return out


@pytest.mark.parametrize("nsk,nsv", [(4, 3), (2, 2), (1, 1), (3, 2)])
def test_persistent_protocol_is_sound(nsk, nsv):
    rng = random.Random(17 * nsk + nsv)
    for case in range(60):
        lengths = _lengths(rng, rng.randint(1, 12), rng.choice([0.0, 0.2, 0.6]))
        for pieces in (2, 4):
            r = simulate(lengths, nsk, nsv, seed=case, pieces=pieces)
            assert r is None, (lengths, pieces, case, r)


def test_runs_of_empty_items_and_single_blocks():
    for lengths in ([0, 0, 0], [0, 3, 0, 0, 2, 0], [1] * 9, [0, 1, 0, 1, 0, 1], [5, 0, 0, 0, 0, 7], [2, 2, 0, 2]):
        for seed in range(25):
            assert simulate(lengths, 4, 3, seed=seed) is None, (lengths, seed)


def test_empty_items_in_the_q_full_sequence_are_caught():
    """Control: if empty items also post q_full, the softmax can run two phases ahead of the QK thread."""
    rng = random.Random(5)
    found = 0
    for case in range(80):
        lengths = _lengths(rng, 10, 0.6)
        if simulate(lengths, 4, 3, seed=case, empty_items_post_q=True) is not None:
            found += 1
    assert found > 0
