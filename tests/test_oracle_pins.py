"""Pins of the CPU oracle against things other than itself (CPU only, -m "not gpu").

P1  brute-force bitwise MAP on cycle-free codes, n <= 20 (sum-product is exact on trees)   -> whole CN/VN recursion,
    syndrome sign, exclusion sets, LLR sign convention, and (lifted trees) the shift rule inside the decoder
P2  brute-force block-ML on tiny codes with cycles                                          -> convergence sanity
P3  closed forms of a single check (degree 2, degree 3; printed value -0.3894400606)          -> CN formula, Phi
P4  Phi values from independent formulas, Phi(Phi(x)) = x                                     -> Phi
P5  syndrome <-> codeword equivalence, bit exact                                              -> syndrome sign vs the
    paper's own zero-syndrome Algorithm 1
P6  syndrome invariant against an independent dense mat-vec                                   -> pass flag, Step 4
P7  noiseless limit                                                                           -> clamp / overflow
P8  degree-1 variable invariant                                                       -> posterior sum
P9  lifting rule against np.roll of the identity                                      -> H construction
P10 frame independence                                                                        -> batching
S4  decision tie rule (bit 0 iff L_v >= 0) at posteriors that are EXACTLY zero          -> Step 4, both places
+   dense tanh-product BP (another formula, another data structure) on small cyclic codes     -> flooding schedule
"""
import math

import numpy as np
import pytest

from paper_1702_07740_b200 import workloads as W
from tests.helpers import (bitwise_map_llr, block_ml_word, dense_h, random_tree_code, tanh_rule_bp_dense,
                           tie_cases)

BIG = 1e300  # msg_max "disabled"


# ----------------------------------------------------------------------------------------------------------- P4
def test_phi_spot_values_and_involution(oracle_lib):
    # independent formulas: -ln tanh(x/2) directly (fine for moderate x) and 2 atanh(e^-x) (large x)
    for x in (0.05, 0.3, 1.0, 2.5, 6.0):
        assert oracle_lib.phi(x) == pytest.approx(-math.log(math.tanh(x / 2.0)), rel=1e-13)
    for x in (6.0, 12.0, 20.0, 30.0, 80.0):
        assert oracle_lib.phi(x) == pytest.approx(2.0 * math.atanh(math.exp(-x)), rel=1e-13)
    for x in (1e-6, 1e-3):  # small x: -ln(x/2) + x^2/12 - ...
        assert oracle_lib.phi(x) == pytest.approx(-math.log(x / 2.0) + x * x / 12.0, rel=1e-12)
    # SURVEY.md P4 digits
    assert oracle_lib.phi(1.0) == pytest.approx(0.7719368329, abs=1e-10)
    assert oracle_lib.phi(1e-3) == pytest.approx(7.600902543, abs=1e-9)
    assert oracle_lib.phi(20.0) == pytest.approx(4.122307245e-9, rel=1e-9)
    for x in np.geomspace(1e-6, 30.0, 60):
        assert oracle_lib.phi(oracle_lib.phi(x)) == pytest.approx(x, rel=1e-10)
    assert oracle_lib.phi(0.0) == math.inf
    assert oracle_lib.phi(1000.0) == 0.0


# ----------------------------------------------------------------------------------------------------------- P9
@pytest.mark.parametrize("Z", [1, 2, 4, 5])
def test_lifting_rule_matches_printed_rule(oracle_lib, Z):
    rng = np.random.default_rng(100 + Z)
    base = rng.integers(-1, Z, size=(3, 5)).astype(np.int32)
    base[0, 0] = Z - 1  # make sure the largest shift is present
    rows, cols = oracle_lib.build_h_coo(base, Z)
    H = np.zeros((3 * Z, 5 * Z), dtype=np.uint8)
    H[rows, cols] = 1
    assert rows.size == int((base >= 0).sum()) * Z
    np.testing.assert_array_equal(H, dense_h(base, Z))
    if Z == 1:
        np.testing.assert_array_equal(H, (base >= 0).astype(np.uint8))
    # the workload generator's syndrome uses the same rule
    x = rng.integers(0, 2, size=(4, 5 * Z), dtype=np.uint8)
    np.testing.assert_array_equal(W.syndrome_of(base, Z, x), (x.astype(np.int64) @ H.T.astype(np.int64)) % 2)


# ----------------------------------------------------------------------------------------------------------- P3
def _single_check(oracle_lib, Q, s):
    d = len(Q)
    base = np.zeros((1, d), dtype=np.int32)
    r = oracle_lib.decode(base, 1, np.array([Q], dtype=np.float32), np.array([[s]], dtype=np.uint8), 1, 0,
                          msg_max=BIG, want_messages=True)
    return r.msg_cv[0], r.posterior[0]


def test_single_check_closed_forms(oracle_lib):
    # degree 2: the message to one variable is the other one's LLR (Phi o Phi = id), sign flipped by s
    a, b = np.float32(0.7), np.float32(-1.3)
    m, post = _single_check(oracle_lib, [a, b], 0)
    assert m[0] == pytest.approx(float(b), rel=1e-12) and m[1] == pytest.approx(float(a), rel=1e-12)
    m1, _ = _single_check(oracle_lib, [a, b], 1)
    np.testing.assert_allclose(m1, -m, rtol=0, atol=0)
    assert post[0] == pytest.approx(float(a) + float(b), rel=1e-12)
    # degree 3: m = 2 atanh(tanh(a/2) tanh(b/2)) = ln((1 + e^{a+b}) / (e^a + e^b))
    c = np.float32(2.1)
    m, _ = _single_check(oracle_lib, [c, a, b], 0)
    fa, fb, fc = float(a), float(b), float(c)
    want0 = math.log((1 + math.exp(fa + fb)) / (math.exp(fa) + math.exp(fb)))
    assert m[0] == pytest.approx(want0, rel=1e-12)
    assert m[0] == pytest.approx(2 * math.atanh(math.tanh(fa / 2) * math.tanh(fb / 2)), rel=1e-12)
    assert m[1] == pytest.approx(2 * math.atanh(math.tanh(fc / 2) * math.tanh(fb / 2)), rel=1e-12)
    assert m[2] == pytest.approx(2 * math.atanh(math.tanh(fc / 2) * math.tanh(fa / 2)), rel=1e-12)
    # SURVEY.md P3 digits (a = 0.7, b = -1.3 exactly; fp32 inputs are within 3e-8 of those)
    assert want0 == pytest.approx(-0.3894400606, abs=2e-7)


def test_clamp_and_degenerate_inputs(oracle_lib):
    # degree-1 check: empty exclusion set -> S = 0 -> |m| = msg_max, sign (-1)^s  (S11)
    for s, sign in ((0, 1.0), (1, -1.0)):
        base = np.zeros((1, 1), dtype=np.int32)
        r = oracle_lib.decode(base, 1, np.array([[0.25]], np.float32), np.array([[s]], np.uint8), 1, 0,
                              want_messages=True)
        assert r.msg_cv[0, 0] == sign * 30.0
        assert r.posterior[0, 0] == 0.25 + sign * 30.0
    # an exactly-zero input erases the check for everyone else; +-0.0 count as positive (S3)
    m, _ = _single_check(oracle_lib, [0.0, 1.5, -2.0], 0)
    assert m[1] == 0.0 and m[2] == 0.0 and m[0] < 0
    m, _ = _single_check(oracle_lib, [-0.0, 1.5, 2.0], 0)
    assert m[1] == 0.0 and not np.signbit(m[1]) and m[0] > 0
    # huge inputs: Phi underflows to 0, message is clamped, no NaN
    base = np.zeros((1, 3), dtype=np.int32)
    r = oracle_lib.decode(base, 1, np.array([[1e4, -1e4, 3e3]], np.float32), np.zeros((1, 1), np.uint8), 3, 0,
                          want_messages=True)
    assert np.isfinite(r.posterior).all() and np.isfinite(r.msg_cv).all()
    np.testing.assert_array_equal(np.abs(r.msg_cv[0]), [30.0, 30.0, 30.0])
    np.testing.assert_array_equal(np.sign(r.msg_cv[0]), [-1.0, 1.0, -1.0])


# ------------------------------------------------------------------------------------------- S4 (P:361 tie rule)
@pytest.mark.parametrize("k", range(8))
def test_decision_tie_rule(oracle_lib, k):
    """P:361 as printed (reading S4): L_v >= 0 -> bit 0, also at L_v = +0.0 and -0.0.  A decoder that tests L_v > 0
    instead gives bit 1 on every variable below."""
    base, Z, llr, syn, max_iter, ties = tie_cases()[k]
    for prec in (64, 32):
        r = oracle_lib.decode(base, Z, llr[None], syn[None], max_iter, 0, precision=prec)
        assert (r.posterior[0, ties] == 0.0).all()
        assert (r.hard[0, ties] == 0).all()
    if base.shape[1] == 1:
        # the all-zero decision satisfies s = 0 but not s = 1; the flag follows the decisions (a ">" decoder would
        # report the opposite in both cases)
        assert r.passed[0] == (1 if syn[0] == 0 else 0)
    # just below the tie the bit is 1
    if max_iter > 0 and base.shape[1] == 1 and syn[0] == 0:
        r = oracle_lib.decode(base, Z, (llr - np.float32(1e-3))[None], syn[None], max_iter, 0)
        assert (r.posterior[0] < 0).all() and (r.hard[0] == 1).all()


# ----------------------------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_exact_map_on_trees(oracle_lib, seed):
    rng = np.random.default_rng(seed)
    base = random_tree_code(rng, n_target=15, max_check_deg=5)
    m, n = base.shape
    H = dense_h(base, 1)
    assert (H.sum(axis=1) >= 2).all()
    Q = rng.normal(0.0, 2.0, size=n).astype(np.float32)
    s = rng.integers(0, 2, size=m, dtype=np.uint8)
    want = bitwise_map_llr(H, s, Q)
    r = oracle_lib.decode(base, 1, Q[None], s[None], 2 * n, 0, msg_max=BIG)
    np.testing.assert_allclose(r.posterior[0], want, rtol=1e-12, atol=1e-12)
    np.testing.assert_array_equal(r.hard[0], (want < 0).astype(np.uint8))
    # bitwise-MAP decisions need not form a word with H x = s; the flag must simply tell the truth
    assert r.passed[0] == int((((H.astype(np.int64) @ r.hard[0]) % 2) == s).all()) and r.iters[0] == 2 * n
    # one iteration fewer than needed must NOT be exact everywhere (the test is sensitive to the iteration count)
    r1 = oracle_lib.decode(base, 1, Q[None], s[None], 1, 0, msg_max=BIG)
    assert np.abs(r1.posterior[0] - want).max() > 1e-6


@pytest.mark.parametrize("seed,Z", [(10, 2), (11, 3), (12, 3)])
def test_exact_map_on_lifted_trees(oracle_lib, seed, Z):
    """A tree base graph lifted by Z with arbitrary shifts is Z disjoint trees: still exact, and now every shift
    value matters (a wrong shift direction pairs the wrong LLRs)."""
    rng = np.random.default_rng(seed)
    base = random_tree_code(rng, n_target=6, max_check_deg=4)
    nz = base >= 0
    base[nz] = rng.integers(0, Z, size=int(nz.sum()))
    if Z > 1:
        base[np.nonzero(nz)[0][0], np.nonzero(nz)[1][0]] = Z - 1
    H = dense_h(base, Z)
    m, n = H.shape
    assert n <= 20
    Q = rng.normal(0.0, 2.0, size=n).astype(np.float32)
    s = rng.integers(0, 2, size=m, dtype=np.uint8)
    want = bitwise_map_llr(H, s, Q)
    r = oracle_lib.decode(base, Z, Q[None], s[None], 2 * n, 0, msg_max=BIG)
    np.testing.assert_allclose(r.posterior[0], want, rtol=1e-12, atol=1e-12)


# ----------------------------------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("seed", [20, 21, 22])
def test_block_ml_on_tiny_cyclic_code(oracle_lib, seed):
    rng = np.random.default_rng(seed)
    Z = 4
    base = np.full((3, 5), -1, dtype=np.int32)
    pattern = np.array([[1, 1, 0, 1, 0], [0, 1, 1, 0, 1], [1, 0, 1, 1, 1]], dtype=bool)
    base[pattern] = rng.integers(0, Z, size=int(pattern.sum()))
    H = dense_h(base, Z)
    n = H.shape[1]
    agree = 0
    for trial in range(6):
        x = rng.integers(0, 2, size=n, dtype=np.uint8)
        s = (H.astype(np.int64) @ x) % 2
        sigma = 0.45  # high SNR
        y = (1.0 - 2.0 * x) + sigma * rng.standard_normal(n)
        Q = (2 * y / sigma ** 2).astype(np.float32)
        r = oracle_lib.decode(base, Z, Q[None], s[None].astype(np.uint8), 50, 1)
        ml_word, ml_ell = block_ml_word(H, s, Q)
        if r.passed[0]:
            np.testing.assert_array_equal((H.astype(np.int64) @ r.hard[0]) % 2, s)
            ell_bp = float(((1 - r.hard[0].astype(np.float64)) * Q).sum())
            assert ml_ell >= ell_bp - 1e-9
            agree += int((r.hard[0] == ml_word).all())
    assert agree >= 4


# ------------------------------------------------------------------------------- flooding schedule, other formula
@pytest.mark.parametrize("Z,n_iter", [(1, 1), (3, 2), (4, 5), (5, 12)])
def test_matches_dense_tanh_rule_bp(oracle_lib, Z, n_iter):
    rng = np.random.default_rng(30 + Z)
    base = np.full((4, 7), -1, dtype=np.int32)
    pattern = rng.random((4, 7)) < 0.55
    pattern[:, 0] = True
    pattern[0, :] = True
    base[pattern] = rng.integers(0, Z, size=int(pattern.sum()))
    H = dense_h(base, Z)
    m, n = H.shape
    Q = rng.normal(0.3, 1.5, size=n).astype(np.float32)
    s = rng.integers(0, 2, size=m, dtype=np.uint8)
    want = tanh_rule_bp_dense(H, Q.astype(np.float64), s, n_iter, msg_max=30.0)
    r = oracle_lib.decode(base, Z, Q[None], s[None], n_iter, 0)
    np.testing.assert_allclose(r.posterior[0], want, rtol=1e-9, atol=1e-9)


# ----------------------------------------------------------------------------------------------------------- P5
def test_syndrome_codeword_equivalence_bit_exact(oracle_lib):
    cfg, base, Z, fr = W.make_config(1, n_frames=4)
    sign = (1.0 - 2.0 * fr.x.astype(np.float32))
    for prec in (64, 32):
        a = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, 20, 0, precision=prec)
        b = oracle_lib.decode(base, Z, fr.llr * sign, np.zeros_like(fr.syndrome), 20, 0, precision=prec)
        np.testing.assert_array_equal(a.posterior, b.posterior * sign.astype(np.float64))
        np.testing.assert_array_equal(a.hard ^ fr.x, b.hard)
        np.testing.assert_array_equal(a.passed, b.passed)
    # early stop on: same stopping iteration
    a = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, 50, 1)
    b = oracle_lib.decode(base, Z, fr.llr * sign, np.zeros_like(fr.syndrome), 50, 1)
    np.testing.assert_array_equal(a.iters, b.iters)
    np.testing.assert_array_equal(a.hard ^ fr.x, b.hard)


# ------------------------------------------------------------------------------------------------------ P6, P10
def test_syndrome_invariant_and_frame_independence(oracle_lib):
    cfg, base, Z, fr = W.make_config(1)
    H = dense_h(base, Z).astype(np.int64)
    for early in (0, 1):
        r = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, early)
        ok = ((r.hard.astype(np.int64) @ H.T) % 2 == fr.syndrome).all(axis=1)
        np.testing.assert_array_equal(r.passed.astype(bool), ok)
        assert 0 < ok.sum() < len(ok) or ok.all()      # config 1 has both converged and stuck frames
        if early:
            assert (r.iters[ok] >= 1).all() and (r.iters[~ok] == cfg.max_iter).all()
            # stopping early means: the same frame with max_iter = iters-1 had not passed yet
            f = int(np.argmax(ok))
            r_prev = oracle_lib.decode(base, Z, fr.llr[f:f + 1], fr.syndrome[f:f + 1], int(r.iters[f]) - 1, 1)
            assert r_prev.passed[0] == 0
        else:
            assert (r.iters == cfg.max_iter).all()
    # P10: a frame alone, in a batch, or permuted gives bit-identical outputs
    r_all = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, 30, 1)
    perm = np.random.default_rng(5).permutation(len(fr.llr))
    r_perm = oracle_lib.decode(base, Z, fr.llr[perm], fr.syndrome[perm], 30, 1, threads=3)
    np.testing.assert_array_equal(r_all.posterior[perm], r_perm.posterior)
    np.testing.assert_array_equal(r_all.iters[perm], r_perm.iters)
    r_one = oracle_lib.decode(base, Z, fr.llr[3:4], fr.syndrome[3:4], 30, 1)
    np.testing.assert_array_equal(r_all.posterior[3], r_one.posterior[0])
    np.testing.assert_array_equal(r_all.hard[3], r_one.hard[0])


# ----------------------------------------------------------------------------------------------------------- P7
@pytest.mark.parametrize("A", [25.0, 1e4])
def test_noiseless_limit(oracle_lib, A):
    cfg, base, Z, fr = W.make_config(1, n_frames=3)
    llr = (A * (1.0 - 2.0 * fr.x.astype(np.float32))).astype(np.float32)
    r = oracle_lib.decode(base, Z, llr, fr.syndrome, 10, 1)
    np.testing.assert_array_equal(r.hard, fr.x)
    np.testing.assert_array_equal(r.iters, 1)
    np.testing.assert_array_equal(r.passed, 1)
    assert np.isfinite(r.posterior).all()
    # every posterior keeps the channel sign and is reinforced by |M(v)| clamped messages at most
    assert (np.sign(r.posterior) == np.sign(llr)).all()
    # max_iter = 0: decisions from the channel alone, iters = 0, pass by direct check
    r0 = oracle_lib.decode(base, Z, llr, fr.syndrome, 0, 1)
    np.testing.assert_array_equal(r0.hard, fr.x)
    np.testing.assert_array_equal(r0.iters, 0)
    np.testing.assert_array_equal(r0.passed, 1)
    np.testing.assert_array_equal(r0.posterior, llr.astype(np.float64))


# ----------------------------------------------------------------------------------------------------------- P8
def test_degree1_variable_posterior(oracle_lib):
    cfg, base, Z, fr = W.make_config(1, n_frames=2)
    r = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, 7, 0, want_messages=True)
    rows, cols = oracle_lib.build_h_coo(base, Z)
    deg = np.bincount(cols, minlength=base.shape[1] * Z)
    d1 = np.nonzero(deg == 1)[0]
    assert d1.size == (base.shape[1] - cfg.code.n_core) * Z
    edge_of = np.full(base.shape[1] * Z, -1)
    edge_of[cols] = np.arange(cols.size)        # for degree-1 variables this is their only edge
    for f in range(2):
        want = fr.llr[f, d1].astype(np.float64) + r.msg_cv[f, edge_of[d1]]
        np.testing.assert_array_equal(r.posterior[f, d1], want)


def test_check_from_iter_semantics(oracle_lib):
    """Early-termination scheduling: with the test enabled from iteration T0 on, a frame that first
    satisfies H xhat = s at t1 stops at max(t1, first passing t >= T0); the decisions of a stopped frame satisfy the
    syndrome; T0 = 1 is the plain decode; T0 > max_iter never stops but still reports pass from the last decisions."""
    cfg, base, Z, fr = W.make_config(1)
    plain = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1)
    same = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, check_from=1)
    np.testing.assert_array_equal(plain.iters, same.iters)
    np.testing.assert_array_equal(plain.hard, same.hard)
    for T0 in (5, 12, 30):
        r = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, check_from=T0)
        stopped = r.iters < cfg.max_iter
        assert (r.iters[stopped] >= T0).all()
        assert (r.iters >= plain.iters).all()
        # the state at iteration t does not depend on when the test runs: same as a fixed-count decode
        for f in np.nonzero(stopped)[0][:3]:
            fixed = oracle_lib.decode(base, Z, fr.llr[f], fr.syndrome[f], int(r.iters[f]), 0)
            np.testing.assert_array_equal(fixed.hard[0], r.hard[f])
            np.testing.assert_array_equal(fixed.posterior[0], r.posterior[f])
        np.testing.assert_array_equal(W.syndrome_of(base, Z, r.hard[r.passed.astype(bool)]),
                                      fr.syndrome[r.passed.astype(bool)])
    never = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, check_from=cfg.max_iter + 1)
    off = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 0)
    np.testing.assert_array_equal(never.iters, off.iters)
    np.testing.assert_array_equal(never.passed, off.passed)
    np.testing.assert_array_equal(never.hard, off.hard)
