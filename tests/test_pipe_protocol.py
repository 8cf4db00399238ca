"""Scheduling simulation of the slot hand-over protocol of csrc/stage_pipe.cu (no GPU; host logic).

The pipelined stage kernel hands shared-memory slots between producer groups and consumer warps through mbarriers whose
waits test a phase PARITY (`mbarrier.try_wait.parity`): a waiter that is two phases away from the barrier passes (or
blocks) wrongly.  This file models the protocol at the level of "who waits for / arrives on which barrier phase", runs
it under random warp scheduling, and checks for every parameter set the library instantiates (Cfg<DIM,N> in
stage_pipe.cu: NG producer groups, NS slots, NB items per quad, CW consumer warps) that nothing deadlocks and no
consumer ever works on a slot that does not hold its quad.  It also keeps the counter-example that motivated the rule
"every consumer warp takes part in the hand-over of every quad": with warps skipping the quads they have no item in,
3-D N = 1 (NB = 1) reads stale slots and hangs.
"""
import random

import pytest


class Bar:
    def __init__(self, count):
        self.count, self.pending, self.phase = count, count, 0

    def arrive(self):
        self.pending -= 1
        if self.pending == 0:
            self.phase += 1
            self.pending = self.count

    def test(self, parity):          # try_wait.parity: has the phase with this parity completed?
        return (self.phase & 1) != parity


def simulate(NG, NS, NB, CW, WPG, NQ, seed, every_quad, late_release=0):
    rng = random.Random(seed)
    full = [Bar(WPG) for _ in range(NS)]
    empty = [Bar(CW if every_quad else NB) for _ in range(NS)]
    gbar = [[0, 0] for _ in range(NG)]
    content = [-1] * NS
    stale = []

    def producer(g):
        def wait_empty(q):
            slot, use = q % NS, q // NS
            if use > 0:
                while not empty[slot].test((use - 1) & 1):
                    yield
        if g < NQ:
            yield from wait_empty(g)                       # prologue: issue the group's first quad
        ql = g
        while ql < NQ:
            if ql + NG < NQ:
                yield from wait_empty(ql + NG)             # issue the next quad one iteration ahead
            gen = gbar[g][1]
            gbar[g][0] += 1
            if gbar[g][0] == WPG:
                gbar[g][0] = 0
                gbar[g][1] += 1
            while gbar[g][1] == gen:                       # bar.sync of the group
                yield
            yield                                          # flux arithmetic
            b = full[ql % NS]
            ph = b.phase
            b.arrive()
            if b.phase != ph:
                content[ql % NS] = ql
            ql += NG

    def consumer(cw):
        if every_quad:
            for q in range(NQ):
                slot, use = q % NS, q // NS
                while not full[slot].test(use & 1):
                    yield
                if ((cw - q * NB) % CW + CW) % CW < NB:    # this warp owns an item of the quad
                    if content[slot] != q:
                        stale.append((cw, q, content[slot]))
                    yield
                    for _ in range(late_release):          # LAYER: the directional contractions still read the
                        if content[slot] != q:             # slot's flux tiles; it is released only after them
                            stale.append((cw, q, content[slot]))
                        yield
                empty[slot].arrive()
        else:
            it = cw
            while it < NQ * NB:
                q = it // NB
                slot, use = q % NS, q // NS
                while not full[slot].test(use & 1):
                    yield
                if content[slot] != q:
                    stale.append((cw, q, content[slot]))
                yield
                empty[slot].arrive()
                it += CW

    procs = [producer(g) for g in range(NG) for _ in range(WPG)] + [consumer(c) for c in range(CW)]
    alive = list(range(len(procs)))
    for _ in range(400000):
        if not alive:
            return True, stale
        i = rng.choice(alive)
        try:
            next(procs[i])
        except StopIteration:
            alive.remove(i)
    return False, stale


def _binding():
    """The constants come from the built library; without it (a host that never ran the build) these tests skip
    instead of failing at import."""
    try:
        from paper_2607_00199_b200 import binding
    except (ImportError, OSError) as e:
        pytest.skip("libalegb.so is not available: %s" % e)
    return binding


def _cfg(dim, N, layer=False):
    """(NG, NS, NB, CW, warps per group) of the kernel compiled for (dim, N), read from the library itself
    (alegb_pipe_config / alegb_pipe_config_layer report Cfg<DIM,N,LAYER> of csrc/stage_pipe.cu), so that the simulation
    cannot drift from the kernel."""
    binding = _binding()
    c = (binding.alegb_pipe_config_layer if layer else binding.alegb_pipe_config)(dim, N)
    return c["producer_groups"], c["slots"], c["items_per_quad"], c["consumer_warps"], c["warps_per_group"]


def test_library_reports_a_consistent_configuration():
    binding = _binding()
    for dim, N in [(2, 1), (2, 4), (3, 1), (3, 3), (3, 4)]:
        plain = binding.alegb_pipe_config(dim, N)
        try:
            layer = binding.alegb_pipe_config_layer(dim, N)
        except binding.AlegbError as e:                          # 3-D N = 4: no ring of such slots fits shared memory
            assert e.status == binding.UNSUPPORTED and (dim, N) == (3, 4)
            continue
        Np = (N + 1) * (N + 2) // 2 if dim == 2 else (N + 1) * (N + 2) * (N + 3) // 6
        assert layer["items_per_quad"] == (Np + 7) // 8 <= layer["consumer_warps"]
        assert layer["producer_groups"] * layer["warps_per_group"] == layer["producer_warps"]
        assert layer["slots"] >= max(layer["producer_groups"], 2)
        assert layer["smem_bytes"] <= 227 * 1024
        assert layer["slots"] <= plain["slots"]                  # dim more flux tiles per slot
        if dim == 3:
            assert layer["producer_groups"] == 1                 # the four producer warps share one quad
    for dim, N in [(2, 1), (2, 4), (3, 1), (3, 3), (3, 4)]:
        c = binding.alegb_pipe_config(dim, N)
        Np = (N + 1) * (N + 2) // 2 if dim == 2 else (N + 1) * (N + 2) * (N + 3) // 6
        assert c["items_per_quad"] == (Np + 7) // 8 <= c["consumer_warps"]
        assert c["producer_groups"] * c["warps_per_group"] == c["producer_warps"]
        assert c["slots"] >= c["producer_groups"]            # a group's wait on `empty` is at most one phase off
        assert c["smem_bytes"] <= 227 * 1024
    with pytest.raises(binding.AlegbError) as e:
        binding.alegb_pipe_config(3, 5)
    assert e.value.status == binding.UNSUPPORTED


@pytest.mark.parametrize("dim,N", [(2, 1), (2, 2), (2, 3), (2, 4), (2, 5), (3, 1), (3, 2), (3, 3), (3, 4)])
def test_shipped_configurations_neither_deadlock_nor_read_stale_slots(dim, N):
    for seed in range(6):
        done, stale = simulate(*_cfg(dim, N), NQ=40, seed=seed, every_quad=True)
        assert done and not stale


@pytest.mark.parametrize("dim,N", [(2, 1), (2, 2), (2, 3), (2, 4), (2, 5), (3, 1), (3, 2), (3, 3), (3, 4)])
def test_layer_configurations_neither_deadlock_nor_read_stale_slots(dim, N):
    """The LAYER instantiation (the default stage kernel of a 3-D mesh with an absorbing layer): other producer
    grouping and ring depth, and a consumer warp holds a slot through the directional contractions before it arrives
    on `empty`."""
    binding = _binding()
    try:
        cfg = _cfg(dim, N, layer=True)
    except binding.AlegbError as e:
        assert e.status == binding.UNSUPPORTED
        pytest.skip("no LAYER instantiation for dim=%d N=%d (the separate layer kernel covers it)" % (dim, N))
    for seed in range(6):
        done, stale = simulate(*cfg, NQ=40, seed=seed, every_quad=True, late_release=1 + dim)
        assert done and not stale


def test_skipping_quads_breaks_low_orders():
    """The protocol before the fix (a consumer warp waits only on the quads it owns an item of)."""
    bad = 0
    for seed in range(4):
        done, stale = simulate(1, 4, 1, 8, 4, NQ=40, seed=seed, every_quad=False)    # 3-D N = 1 as it was shipped
        bad += (not done) or bool(stale)
        done, stale = simulate(2, 4, 3, 8, 2, NQ=40, seed=seed, every_quad=False)    # the hang seen on config 5
        bad += (not done) or bool(stale)
    assert bad == 8
    for seed in range(4):                                   # and the same parameters under the rule
        assert simulate(1, 4, 1, 8, 4, 40, seed, True) == (True, [])
        assert simulate(2, 4, 3, 8, 2, 40, seed, True) == (True, [])
