"""The grid-wide scalar all-reduce of a parameter move (row A4) on its own: pimc_exchange_selftest runs the
exchange variants that were measured for DESIGN.md "exchange" on a cooperative launch of one CTA per SM and reports SM
clock ticks per round.  This test checks what must hold for ANY variant -- every CTA ends up with the same bits (all CTAs
must take the same accept decision) and the total is the exact sum to rounding -- and prints the timing table that
profiles/r02_exchange_probe.md quotes (`python -m pytest tests/test_gpu_exchange.py -m gpu -s`)."""
import pytest

pytestmark = pytest.mark.gpu

MODES = [(0, "flat all-gather, every thread polls one line at once (round 1)"),
         (109, "flat all-gather, first poll held 450 cycles (round 2, the sweep kernel's)"),
         (1, "two-hop butterfly by one warp"),
         (2, "block sum, one warp gathers all"),
         (4, "communication warp gathers all"),
         (5, "fixed-point integer accumulation in L2 (order-independent)"),
         (6, "software-pipelined, two speculative evaluations per round (2 x work)"),
         (10, "push into private inboxes")]


def test_every_exchange_variant_gives_all_ctas_the_same_exact_total():
    import paper_1103_4887_b200 as P
    rows = []
    for work in (0, 75):
        base = P.exchange_selftest(-1, 0, 256, 3000, work)["cycles_per_round"]
        hop = P.exchange_selftest(3, 0, 256, 3000, work)["cycles_per_round"] - base
        rows.append(f"work = {work:3d} iterations = {base:6.0f} cycles per round; one L2 hop (ring) = {hop:5.0f}")
        for mode, name in MODES:
            r = P.exchange_selftest(mode, 0, 256, 3000, work)
            assert r["n_distinct"] == 1, (mode, r)                      # one decision grid-wide
            assert r["max_abs_err"] < 1e-9, (mode, r)                   # and it is the sum (partials are O(0.5), 148 x 256 of them)
            extra = r["cycles_per_round"] - base * (2 if mode == 6 else 1)
            rows.append(f"    mode {mode:3d}  {extra:7.0f} cycles on top of the work   {name}")
    print("\n" + "\n".join(rows))


def test_exchange_on_fewer_ctas_and_smaller_blocks():
    import paper_1103_4887_b200 as P
    for n, T in ((1, 64), (2, 256), (13, 128), (37, 256), (74, 32)):
        for mode in (0, 1, 4, 5, 100):
            r = P.exchange_selftest(mode, n, T, 300, 3)
            assert r["n_distinct"] == 1 and r["max_abs_err"] < 1e-9, (n, T, mode, r)


def test_components_of_a_block_sum():
    # what DESIGN.md quotes: xor tree ~207 cycles, barrier + serial 8-sum ~307, block_sum_db (tree sum now) in between
    import paper_1103_4887_b200 as P
    base = P.exchange_selftest(-1, 0, 256, 3000, 0)["cycles_per_round"]
    out = {name: (P.exchange_selftest(mode, 0, 256, 3000, 0)["cycles_per_round"] - base) / 4
           for mode, name in ((7, "block_sum_db"), (8, "warp xor tree"), (9, "barrier + serial sum of 8"))}
    print("\ncycles each:", {k: round(v) for k, v in out.items()})
    assert 50 < out["warp xor tree"] < 1000 and out["block_sum_db"] > out["warp xor tree"]


def test_latency_probes_l2_hit_map_and_one_way_packet():
    # the two measurements DESIGN.md 6.1a rests its "the hop is the L2 path itself" on, re-runnable (pimc_latency_selftest).  The figures
    # are SM clock ticks of a fixed TIME (an idle GPU that has not clocked up yet counts ~ 0.67x as many), so only ratios are asserted
    import paper_1103_4887_b200 as Pm
    Pm.fp64_peak(200)                                                # clock the SMs up
    m = Pm.latency_selftest(0, 128)
    print("L2 hit map:", m)
    assert 100 < m["near"] < m["far"] < 1000 and m["far"] < 1.5 * m["near"], m     # an L2 hit: a few hundred ticks; the far die costs little more
    assert m["group_a"] + m["group_b"] >= 100
    one_way = {how: Pm.latency_selftest(how, 1) for how in (1, 2, 3, 4, 5)}
    print("one-way ticks to the neighbouring SM (1 st.relaxed, 2 atom.exch, 3 red.max, 4 st.volatile, 5 st.release):", one_way)
    for how in (1, 2, 3, 4):
        assert 1.5 * m["far"] < one_way[how] < 10 * m["far"], (one_way, m)          # a packet needs several L2-hit times whatever publishes it
        assert 0.8 < one_way[how] / one_way[1] < 1.25, one_way                         # (same lines, same pair: the store flavour does not matter)
    assert one_way[5] > 1.2 * one_way[1]                                               # a release store is the slow way
    # where the line lives: fast only when writer, reader and the line's home share a die; across the dies every line is slow
    w = Pm.latency_selftest(6, 16)
    print("line-address sweep:", w)
    assert w["same_min"] < 0.8 * w["same_max"] and 0.2 <= w["frac_fast"] <= 0.8, w      # two classes of lines for a same-die pair
    assert w["cross_min"] > 1.25 * w["same_min"] and w["cross_max"] < 1.3 * w["cross_min"], w   # one (slow) class across the dies
