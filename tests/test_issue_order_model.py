"""Host-side model of the attention kernel's operand-ring protocol (paper_2605_30519_b200/csrc/attn_tcgen05.cu: batch_pos_qk /
batch_pos_pv, the MMA issuer's batch order and the barrier parities it derives from a batch's position).  The kernel keeps ring
positions REGULAR -- QK_t at 2t-2 (t >= 2), PV_t at 2t+3 -- also at the end of the sequence where QK batches have run out, and
computes a slot's mbarrier parity from the position alone.  That is only right if (a) the issue order visits positions in
increasing order, (b) every earlier position of the same slot was really used (else the barrier has completed fewer phases than
the formula assumes) and (c) a slot is refilled only after its previous tenant was consumed.  Checked here for every tile count."""
import pytest

NSTAGE = 5


def pos_qk(t):
    return t if t < 2 else 2 * t - 2


def pos_pv(t):
    return 2 * t + 3


def issue_order(T):
    """QK_0, QK_1, then per tile t: QK_{t+2} (if it exists), PV_t -- the unrolled issuer's order."""
    seq = [("qk", t) for t in range(min(T, 2))]
    for t in range(T):
        if t + 2 < T:
            seq.append(("qk", t + 2))
        seq.append(("pv", t))
    return seq


@pytest.mark.parametrize("T", range(1, 64))
def test_ring_positions_and_parities(T):
    seq = issue_order(T)
    assert sorted(seq) == sorted([("qk", t) for t in range(T)] + [("pv", t) for t in range(T)])
    positions = [pos_qk(t) if k == "qk" else pos_pv(t) for k, t in seq]
    assert positions == sorted(positions) and len(set(positions)) == len(positions)  # (a) strictly increasing
    used = set(positions)
    for p in positions:
        # (b) the parity the kernel waits for is (p // NSTAGE) & 1: the slot must have been filled p // NSTAGE times before
        earlier = [q for q in range(p % NSTAGE, p, NSTAGE)]
        assert all(q in used for q in earlier), (T, p, earlier)
    # (c) producer / consumer interleaving: a position is produced (TMA) only after position p - NSTAGE was consumed, and the
    # consumer needs p produced: simulate both walking their own ordered lists and make sure neither starves
    k_items = [pos_qk(t) for t in range(T)]
    v_items = [pos_pv(t) for t in range(T)]
    produced, consumed = set(), set()
    ki = vi = ci = 0
    progress = True
    while progress:
        progress = False
        for items, idx_name in ((k_items, "k"), (v_items, "v")):
            i = ki if idx_name == "k" else vi
            while i < len(items) and (items[i] < NSTAGE or (items[i] - NSTAGE) in consumed):
                produced.add(items[i])
                i += 1
                progress = True
            if idx_name == "k":
                ki = i
            else:
                vi = i
        while ci < len(positions) and positions[ci] in produced:
            consumed.add(positions[ci])
            ci += 1
            progress = True
    assert ci == len(positions) and ki == T and vi == T, (T, ci, ki, vi)


def test_softmax_barrier_phase_formulas():
    """s_full[p] / p_full[p] / pv_done[p] complete once per tile of parity p: tile t is completion number t >> 1, so its waiters
    use parity (t >> 1) & 1; the issuer's round-relative form ((I >> 1) & 1) ^ (round & 1) must agree for rounds of 10 tiles."""
    for t in range(0, 200):
        r, i = divmod(t, 10)
        assert ((i >> 1) & 1) ^ (r & 1) == (t >> 1) & 1
        if t >= 2:  # s_free[p] completion for tile t - 2, seen by QK_t (round-relative J = i + 2 .. 11 in the kernel, same identity)
            assert (((t >> 1) - 1) & 1) == ((((i >> 1) - 1) & 1) ^ (r & 1)) % 2
