"""The roofline's work constants are COUNTED, not estimated (SURVEY.md §8(d) "Fix W_site and W_eval once (from the oracle's
operation count)"): oracle/count_work.py restates the oracle's arithmetic on a counting number type, checks the restatement bit
for bit against the compiled oracle, and writes oracle/work_constants.json; bench.py's literals must equal that file."""
import json
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_counted_work_matches_the_committed_constants_and_bench():
    from oracle import count_work
    site, ev = count_work._validate_and_count()          # asserts bit-identity with the compiled oracle along the way
    committed = json.load(open(os.path.join(ROOT, "oracle", "work_constants.json")))
    assert committed["slots_per_site_update"] == site.slots and committed["slots_per_param_eval"] == ev.slots
    assert committed["calls_per_site_update"] == site.calls and committed["calls_per_param_eval"] == ev.calls
    # what the count must contain: 4 RHS x 3 gates = 12 tanh per increment; two Box-Muller pairs and three logarithms per update
    assert site.calls["tanh"] == 12 and ev.calls["tanh"] == 12
    assert site.calls["log"] == 3 and site.calls["sqrt"] == 2 and site.calls["sincos"] == 2
    assert site.ops >= site.slots and ev.ops >= ev.slots and site.slots > ev.slots
    src = open(os.path.join(ROOT, "bench.py")).read()
    w_site = float(re.search(r"^W_SITE_ORACLE\s*=\s*([0-9.]+)", src, re.M).group(1))
    w_eval = float(re.search(r"^W_EVAL_ORACLE\s*=\s*([0-9.]+)", src, re.M).group(1))
    assert w_site == site.slots and w_eval == ev.slots


def test_counting_number_type_counts_fma_pairs_once():
    from oracle.count_work import C, Tally
    t = Tally()
    a, b, c = C(2.0, t), C(3.0, t), C(5.0, t)
    r = a * b + c                       # one FMA
    assert r.v == 11.0 and t.slots == 1 and t.ops == 2
    r = (a * b) * c + (a + b)           # mul, mul (fused with the add), add
    assert t.slots == 1 + 3 and t.ops == 2 + 4
    p = a * b
    _ = p + c; _ = p + c                # a product can be fused only once
    assert t.slots == 4 + 1 + 0 + 1
