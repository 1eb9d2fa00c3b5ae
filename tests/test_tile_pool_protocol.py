"""Model check of the tile-buffer pool of the pass kernels (csrc/sso_ring.cuh, TileRing): G groups of a CTA share NB >= G
shared-memory buffers; tiles 0 .. nloc-1 are loaded in order, each into whichever buffer was just emptied, and consumed
in the same order (tickets); every buffer carries the number of its tile and the parity of its fill, written when the
fill is issued and kept until the tile is consumed.  The model interleaves the groups at random and checks what the kernel relies on:
every tile is consumed exactly once, nobody waits for ever, and a waiter never matches the parity of an older fill
of its buffer (the failure of a fixed ticket -> buffer map, which the second model reproduces)."""
import random

import pytest

def run_pool(NB, G, nloc, seed, fixed_map=False):
    rng = random.Random(seed)
    issued = [0] * NB      # fills issued into each buffer
    landed = [0] * NB      # fills completed (a load lands some time after it is issued)
    inflight = []          # (buffer) loads issued and not yet landed
    tag = [None] * NB      # (tile, parity) of the fill each buffer holds
    tile_of_fill = {}

    def issue(tile, b):
        par = issued[b] & 1
        tile_of_fill[(b, issued[b])] = tile
        issued[b] += 1
        tag[b] = (tile, par)
        inflight.append(b)

    for b in range(NB):
        if b < nloc:
            issue(b, b)
    nxt, ticket = NB, 0
    state = []
    for g in range(G):
        state.append(["wait", ticket])
        ticket += 1
    consumed = []
    for _ in range(400000):
        if all(s[0] == "done" for s in state):
            return "ok", consumed
        if inflight and rng.random() < 0.3:  # a load lands
            b = inflight.pop(rng.randrange(len(inflight)))
            landed[b] += 1
            continue
        g = rng.choice([g for g in range(G) if state[g][0] != "done"])
        st = state[g]
        if st[0] == "wait":
            s = st[1]
            if s >= nloc:
                st[0] = "done"
                continue
            if fixed_map:
                b, f = s % NB, s // NB
                par = f & 1
            else:
                hit = [bb for bb in range(NB) if tag[bb] is not None and tag[bb][0] == s]
                if not hit:
                    continue  # the fill of this tile has not been issued yet: spin
                b = hit[0]
                par = tag[b][1]
                f = issued[b] - 1
            # mbarrier.try_wait.parity(par): true iff the last COMPLETED phase of the barrier has parity par
            if landed[b] >= 1 and ((landed[b] - 1) & 1) == par:
                if fixed_map and landed[b] - 1 != f:
                    return "alias", consumed  # matched a phase that is two fills old
                if not fixed_map:
                    assert landed[b] - 1 == f
                    assert tile_of_fill[(b, f)] == s
                consumed.append(s)
                state[g] = ["work", s, b]
        else:  # finished a tile: draw the next ticket, refill the emptied buffer
            _, s, b = st
            state[g] = ["wait", ticket]
            ticket += 1
            t = nxt
            nxt += 1
            if t < nloc:
                if fixed_map:
                    issued[b] += 1
                    inflight.append(b)
                else:
                    issue(t, b)
    return "stuck", consumed


@pytest.mark.parametrize("NB", [1, 2, 3, 4, 5, 8, 12])
def test_pool_consumes_every_tile_once_and_never_hangs(NB):
    for G in range(1, NB + 1):
        for nloc in (0, 1, 2, NB - 1, NB, NB + 1, 3 * NB + 2, 57):
            if nloc < 0:
                continue
            for seed in range(12):
                verdict, consumed = run_pool(NB, G, nloc, seed)
                assert verdict == "ok", (NB, G, nloc, seed, verdict)
                assert sorted(consumed) == list(range(nloc)), (NB, G, nloc, seed)


def test_fixed_ticket_to_buffer_map_aliases_or_hangs():
    """The design that was NOT adopted: ticket s -> buffer s mod NB, fill s div NB.  A group can lap a slow one and wait
    on a buffer whose previous fill has not landed; its parity then matches a phase that is two fills old."""
    bad = 0
    for seed in range(200):
        verdict, _ = run_pool(3, 3, 40, seed, fixed_map=True)
        bad += verdict != "ok"
    assert bad > 0
