"""Host model of the TMA-ring protocol of k_tc_encode_rvq's level phase (tc_encode_rvq.cu): P producer warps take the
128-codeword chunks in turn (producer p: chunks p, p + P, ...), each chunk is `nkb` codebook tiles in consecutive ring
slots, the MMA issuer consumes the tiles in order, and every slot has a `full` and an `empty` mbarrier that carry ONE
phase bit.  A producer that runs two uses of a slot ahead of the consumer passes its parity wait on the still-initial
barrier and overwrites an unconsumed tile -- the launch failure of round 2's first three-producer version (ring of 7
slots, nkb = 4).  The kernel therefore bounds the producers in use by `ring_slots // nkb`; this test checks that rule,
and that the bound is not vacuous, on random interleavings of the actors."""
import random

import pytest


def simulate(producers, nkb, ring, nchunks, seed):
    rnd = random.Random(seed)
    ntiles = nchunks * nkb
    full_phase = [0] * ring          # completed phases of the slot's `full` barrier
    empty_phase = [0] * ring         # ... of its `empty` barrier
    slot_tile = [None] * ring
    prod = [dict(chunk=p, j=0) for p in range(producers)]
    consumed = 0
    for _ in range(200000):
        if consumed == ntiles:
            return "ok"
        actor = rnd.randrange(producers + 1)
        if actor == producers:                                   # the MMA issuer
            st, ph = consumed % ring, (consumed // ring) & 1
            if (full_phase[st] & 1) != ph:                       # try_wait.parity(ph) succeeds
                if slot_tile[st] != consumed:
                    return f"the issuer reads tile {slot_tile[st]} instead of {consumed}"
                empty_phase[st] += 1                             # tcgen05.commit -> empty barrier
                consumed += 1
        else:
            pr = prod[actor]
            if pr["chunk"] >= nchunks:
                continue
            it = pr["chunk"] * nkb + pr["j"]
            st, ph = it % ring, (it // ring) & 1
            if (empty_phase[st] & 1) != (ph ^ 1):                # try_wait.parity(ph ^ 1) succeeds
                if slot_tile[st] is not None and slot_tile[st] >= consumed:
                    return f"tile {it} overwrites the unconsumed tile {slot_tile[st]}"
                slot_tile[st] = it
                full_phase[st] += 1                              # expect_tx + the bytes landing
                pr["j"] += 1
                if pr["j"] == nkb:
                    pr["j"] = 0
                    pr["chunk"] += producers
    return "deadlock"


@pytest.mark.parametrize("nkb,ring", [(1, 5), (2, 8), (4, 7), (4, 8), (4, 12), (2, 3), (1, 2)])
def test_producers_bounded_by_ring_over_tiles_per_chunk_are_safe(nkb, ring):
    p2 = max(1, min(3, ring // nkb))                             # tc_encode_rvq.cu: p.p2
    for seed in range(200):
        assert simulate(p2, nkb, ring, 24, seed) == "ok", (p2, nkb, ring, seed)


def test_three_producers_on_a_seven_slot_ring_overwrite():
    outcomes = {simulate(3, 4, 7, 24, seed) for seed in range(200)}
    assert any("overwrites" in o or "reads tile" in o for o in outcomes)
