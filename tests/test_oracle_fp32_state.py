"""Pins for the fp32-state branches of the oracle (state_dtype = 32): the checker of the fp32 variant of config 3
(BASELINE.json configs[3] "run in both fp64 and fp32"; PAPER.md:246 runs in single precision).

Nothing here calls the oracle on both sides: expectations are built from the Philox words with exact rational arithmetic
(fractions.Fraction) and explicit roundings to float32, or from the fp64 formulas within float32 rounding bounds.
"""
from fractions import Fraction

import numpy as np

import oracle
from oracle import OracleChain
from workloads import MODEL_HH, make_workload

STREAM_PROPOSAL, STREAM_ACCEPT, STREAM_PARAM = 0, 1, 2
SEED = 77


def f32(v):
    """Round a Fraction / float to the nearest float32 (one rounding: the inputs used here are exact in float64)."""
    return np.float32(float(v))


def is_f32(a):
    a = np.asarray(a, dtype=np.float64)
    return np.all(a.astype(np.float32).astype(np.float64) == a)


def chain(kind, M=40):
    w = make_workload(2, M=M)
    o = OracleChain.from_workload(w, state_dtype=32)
    o.set_proposal(w.w_state, w.w_param, kind)
    return w, o


def test_fp32_state_is_rounded_on_entry():
    w, o = chain(1)
    x, p = o.get_path()
    assert is_f32(x) and is_f32(p)
    assert np.array_equal(x, np.asarray(w.x0[0], np.float32).astype(np.float64))
    assert np.array_equal(p, np.asarray(w.p0[0], np.float32).astype(np.float64))
    assert not is_f32(w.p0[0])          # the input is NOT float-representable to begin with: the rounding is real


def test_fp32_uniform_proposals_are_the_exact_rational_rounded_twice():
    # x' = RN32(x + RN32(w32 (2u - 1))), u = ((word >> 9) + 1/2) 2^-23 exactly (SURVEY.md R3, fp32 mode)
    w, o = chain(1)
    x0, _ = o.get_path()
    t0 = o.sweep_index
    o.sweep(1, SEED, do_params=False)
    tr = o.trace()
    # sites of the EVEN half-sweep see the initial path (their proposal is x0 + step); check those
    for n in range(0, w.M + 1, 2):
        words = oracle.draw_words(SEED, t0, 0, n, STREAM_PROPOSAL, 0)
        for a in range(4):
            u = (Fraction(int(words[a]) >> 9) + Fraction(1, 2)) / 2**23
            assert Fraction(float(oracle.u01f_from_word(int(words[a])))) == u          # exact, strictly inside (0, 1)
            step = f32(Fraction(float(np.float32(w.w_state[a]))) * (2 * u - 1))
            expect = np.float32(np.float64(np.float32(x0[n, a])) + np.float64(step))
            assert tr["xprop"][n, a] == np.float64(expect), (n, a)
    assert is_f32(tr["xprop"])


def test_fp32_gaussian_proposals_follow_the_fp64_box_muller_within_float_rounding():
    w, o = chain(0)
    x0, _ = o.get_path()
    t0 = o.sweep_index
    o.sweep(1, SEED, do_params=False)
    tr = o.trace()
    assert is_f32(tr["xprop"])
    eps = 2.0**-23
    worst = 0.0
    for n in range(0, w.M + 1, 2):
        words = oracle.draw_words(SEED, t0, 0, n, STREAM_PROPOSAL, 0)
        for pair in range(2):
            u1 = float(oracle.u01f_from_word(int(words[2 * pair]))); u2 = float(oracle.u01f_from_word(int(words[2 * pair + 1])))
            r = np.sqrt(-2.0 * np.log(u1))
            z = (r * np.cos(2 * np.pi * u2), r * np.sin(2 * np.pi * u2))       # words (0,1) -> components (0,1); (2,3) -> (2,3)
            for j in range(2):
                a = 2 * pair + j
                ws = float(np.float32(w.w_state[a]))
                expect = x0[n, a] + ws * z[j]
                # float rounding of the sum, of the product, of z, and of the angle 2 pi u2 (|d angle| <= 4 eps => |dz| <= 4 eps r)
                tol = 1.01 * eps * abs(expect) + ws * (3 * eps * abs(z[j]) + 5 * eps * r) + 1e-30
                err = abs(tr["xprop"][n, a] - expect)
                worst = max(worst, err / tol)
                assert err <= tol, (n, a, err, tol)
    assert worst > 1e-3          # the comparison is at float resolution, not vacuous
    # power: the sin / cos pairing matters at this tolerance
    words = oracle.draw_words(SEED, t0, 0, 0, STREAM_PROPOSAL, 0)
    u1 = float(oracle.u01f_from_word(int(words[0]))); u2 = float(oracle.u01f_from_word(int(words[1])))
    r = np.sqrt(-2 * np.log(u1))
    swapped = x0[0, 0] + float(np.float32(w.w_state[0])) * r * np.sin(2 * np.pi * u2)
    assert abs(tr["xprop"][0, 0] - swapped) > 1e-4 * float(w.w_state[0])


def test_fp32_accept_uniform_is_the_float_log_of_word_0():
    w, o = chain(1)
    t0 = o.sweep_index
    o.sweep(1, SEED, do_params=False)
    tr = o.trace()
    assert is_f32(tr["logu"])
    for n in range(w.M + 1):
        words = oracle.draw_words(SEED, t0, 0, n, STREAM_ACCEPT, 0)
        u = (Fraction(int(words[0]) >> 9) + Fraction(1, 2)) / 2**23
        ref = np.log(np.float64(float(u)))
        assert abs(tr["logu"][n] - ref) <= 2.0**-23 * abs(ref) + 1e-45, n      # within one float ulp of the exact logarithm
    # ... and not the fp64 accept uniform of words (0, 1): those differ by far more than a float ulp somewhere
    w64 = [np.log(oracle.u01_from_two_words(*[int(v) for v in oracle.draw_words(SEED, t0, 0, n, STREAM_ACCEPT, 0)[:2]])) for n in range(w.M + 1)]
    assert np.max(np.abs(np.asarray(w64) - tr["logu"])) > 1e-4


def test_fp32_parameter_proposals_are_formed_in_float():
    # p' = RN32(p32 + RN32(step)), step = w_p z0 from the fp64 Box-Muller of words (0, 1) of the parameter stream; log u stays fp64
    w, o = chain(0)
    _, p0 = o.get_path()
    t0 = o.sweep_index
    o.sweep(1, SEED)
    tr = o.trace()
    assert is_f32(tr["pprop"])
    p = p0.copy()
    for l in range(7):
        words = [int(v) for v in oracle.draw_words(SEED, t0, 0, l, STREAM_PARAM, 0)]
        z = oracle.box_muller(oracle.u01_from_word(words[0]), oracle.u01_from_word(words[1]))
        step = w.w_param[l] * z[0]
        expect = np.float64(np.float32(np.float32(p[l]) + np.float32(step)))
        assert tr["pprop"][l] == expect, l
        assert tr["logup"][l] == np.log(oracle.u01_from_two_words(words[2], words[3]))
        if tr["accp"][l]:
            p[l] = expect
    _, p1 = o.get_path()
    assert np.array_equal(p1, p) and is_f32(p1)


def test_fp32_chain_stays_float_representable_and_differs_from_fp64():
    w, o = chain(0, M=64)
    o64 = OracleChain.from_workload(w, state_dtype=64)
    o.sweep(20, SEED); o64.sweep(20, SEED)
    x, p = o.get_path()
    assert is_f32(x) and is_f32(p)
    x64, _ = o64.get_path()
    assert not is_f32(x64)
    # same Philox words, different uniforms (23-bit vs 32-bit): the two chains are close but not equal
    assert 0 < np.max(np.abs(x - x64)[:, 0]) < 5.0
    assert MODEL_HH == 1
