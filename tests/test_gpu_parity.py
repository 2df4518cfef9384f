"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Run on the B200 box with `pytest -m gpu`.

Bar (BASELINE.json north_star): fixed iteration count, early stop off:
    |L_gpu - L_oracle| <= 1e-3 * max(1, |L_oracle|)   for every variable,
    hard bits identical wherever |L_oracle| > 1e-2;
early stop on: per-frame pass flags and iteration counts agree with the oracle (statistical consistency is judged
on the same inputs, so the comparison is per frame).

fp32 noise floor: flooding BP on a frame that does not converge is a chaotic
map; 1-ulp differences grow ~1.2x per iteration for ANY fp32 evaluation, including the oracle's own float
instantiation, which measures that floor on the same inputs.  A frame is UNPINNED only where the floor itself exceeds
HALF the tolerance (tests/parity_cases.py); there the GPU deviation must stay within UNPINNED_FACTOR x the floor and the
frame is printed.  Everywhere else the stated tolerance is asserted as it stands.  profiles/r02_parity_report.md
(written on the B200 by tests/parity_report.py) records err, floor and hard-bit mismatches per config / frame /
iteration count.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1702_07740_b200 import workloads as W  # noqa: E402
from tests.helpers import bitwise_map_llr, dense_h, random_tree_code, tie_cases  # noqa: E402
from tests import parity_cases as PC  # noqa: E402
from tests.parity_cases import HARD_MIN, TOL, rel_err  # noqa: E402


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_1702_07740_b200 import binding
    return binding


def gpu_decode(B, base, Z, llr, syn, max_iter, early_stop, want_posterior=True, check_from_iter=1):
    return PC.gpu_decode(B, base, Z, llr, syn, max_iter, early_stop, want_posterior, check_from_iter)


def assert_parity(oracle_lib, B, base, Z, llr, syn, n_iter, label):
    """Fixed iteration count, early stop off (tests/parity_cases.py has the rule).  Returns (max rel err per frame,
    fp32 floor per frame where it was needed, else nan)."""
    case = PC.run_fixed(oracle_lib, B, base, Z, llr, syn, n_iter, label)
    for f in case.frames:
        if f.unpinned:
            print(f"{label}: frame {f.frame} iter {n_iter}: UNPINNED (fp32 floor {f.floor:.2e} > tol/2), gpu err "
                  f"{f.err:.2e}, hard-bit mismatches where |L| > 1e-2: {f.hard_mismatch} of {f.decided}")
    assert case.ok, f"{label} iter {n_iter}: {case.failures()}"
    return (np.array([f.err for f in case.frames]),
            np.array([np.nan if f.floor is None else f.floor for f in case.frames]))


# ------------------------------------------------------------------------------------------------ config 1 (full)
@pytest.mark.parametrize("n_iter", [1, 2, 5, 10, 20, 35, 50])
def test_config1_fixed_iterations(oracle_lib, B, n_iter):
    cfg, base, Z, fr = W.make_config(1)
    err, floor = assert_parity(oracle_lib, B, base, Z, fr.llr, fr.syndrome, n_iter, "cfg1")
    print(f"cfg1 iter {n_iter}: max err {err.max():.2e}, median {np.median(err):.2e}, floor max {np.nanmax(floor) if np.isfinite(floor).any() else float('nan'):.2e}")


def test_config1_early_stop_matches_oracle(oracle_lib, B):
    cfg, base, Z, fr = W.make_config(1)
    ref = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1)
    hard, iters, passed, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1)
    np.testing.assert_array_equal(passed, ref.passed)
    np.testing.assert_array_equal(iters, ref.iters)
    ok = ref.passed.astype(bool)
    assert ok.any() and not ok.all()
    np.testing.assert_array_equal(hard[ok], ref.hard[ok])
    assert rel_err(post[ok], ref.posterior[ok]).max() <= TOL
    np.testing.assert_array_equal(W.syndrome_of(base, Z, hard[ok]), fr.syndrome[ok])


@pytest.mark.parametrize("check_from", [2, 7, 13, 50, 60])
def test_config1_check_from_iter_matches_oracle(oracle_lib, B, check_from):
    """Early-termination scheduling: the test runs at iterations >= check_from only."""
    cfg, base, Z, fr = W.make_config(1)
    ref = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, check_from=check_from)
    hard, iters, passed, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1,
                                           check_from_iter=check_from)
    np.testing.assert_array_equal(passed, ref.passed)
    np.testing.assert_array_equal(iters, ref.iters)
    stopped = ref.iters < cfg.max_iter
    assert (iters[stopped] >= check_from).all()
    ok = ref.passed.astype(bool)
    np.testing.assert_array_equal(hard[ok], ref.hard[ok])
    assert rel_err(post[ok], ref.posterior[ok]).max() <= TOL


# ----------------------------------------------------------------------- reduced-Z versions of configs 2, 3, 5
@pytest.mark.parametrize("cfg_index,Z,n_iter", [(2, 333, 30), (3, 1000, 30), (5, 517, 40), (3, 257, 8), (2, 64, 12)])
def test_reduced_configs_fixed_iterations(oracle_lib, B, cfg_index, Z, n_iter):
    cfg, base, Z, fr = W.make_config(cfg_index, Z=Z, n_frames=4)
    err, floor = assert_parity(oracle_lib, B, base, Z, fr.llr, fr.syndrome, n_iter, f"cfg{cfg_index}/Z{Z}")
    print(f"cfg{cfg_index} Z={Z} iter {n_iter}: max err {err.max():.2e}")


@pytest.mark.parametrize("cfg_index,snr_point,Z", [(5, 5, 2000), (5, 3, 2000), (3, 0, 500)])
def test_reduced_configs_early_stop(oracle_lib, B, cfg_index, snr_point, Z):
    cfg, base, Z, fr = W.make_config(cfg_index, snr_point=snr_point, Z=Z, n_frames=6)
    max_iter = min(cfg.max_iter, 120)
    ref = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, max_iter, 1)
    hard, iters, passed, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, max_iter, 1)
    print(f"cfg{cfg_index} snr{snr_point} Z={Z}: oracle pass {ref.passed} iters {ref.iters}; gpu {passed} {iters}")
    np.testing.assert_array_equal(passed, ref.passed)
    np.testing.assert_array_equal(iters, ref.iters)
    ok = ref.passed.astype(bool)
    np.testing.assert_array_equal(hard[ok], ref.hard[ok])
    np.testing.assert_array_equal(W.syndrome_of(base, Z, hard[ok]), fr.syndrome[ok])


# --------------------------------------------------------------------------------- full-size configs (n = 1e6)
@pytest.mark.parametrize("cfg_index,n_iter", [(2, 50), (3, 50)])
def test_full_size_single_frame(oracle_lib, B, cfg_index, n_iter):
    """Configs 2 and 3 at full size, parity mode: 50 fixed iterations, early stop off."""
    cfg, base, Z, fr = W.make_config(cfg_index)
    assert fr.llr.shape == (1, 1000000)
    err, floor = assert_parity(oracle_lib, B, base, Z, fr.llr, fr.syndrome, n_iter, f"cfg{cfg_index}")
    print(f"cfg{cfg_index} full size iter {n_iter}: max err {err.max():.2e}")


@pytest.mark.parametrize("cfg_index,Z,n_iter", [(3, 1000, 200), (1, 32, 120)])
def test_long_fixed_count(oracle_lib, B, cfg_index, Z, n_iter):
    """Fixed-count posterior comparison well past 50 iterations (stalled frames of config 3's structure: errors do not
    accumulate; config 1: converged frames settle, the chaotic ones are reported against their floor)."""
    cfg, base, Z, fr = W.make_config(cfg_index, Z=Z, n_frames=4 if cfg_index != 1 else None)
    err, floor = assert_parity(oracle_lib, B, base, Z, fr.llr, fr.syndrome, n_iter, f"cfg{cfg_index}/Z{Z}")
    print(f"cfg{cfg_index} Z={Z} iter {n_iter}: max err {err.max():.2e}")


def test_config4_batch_sampled_frames(oracle_lib, B):
    """Config 4 in the launch configuration bench.py times (64 frames, early stop on); the oracle checks sampled
    frames one by one, and frame independence (bit-identical alone vs in the batch) covers the rest."""
    cfg, base, Z, fr = W.make_config(4, n_frames=64)
    n_iter = 12
    code = B.QCLDPCCode(base, Z)
    d_llr = torch.from_numpy(fr.llr).cuda()
    d_syn = torch.from_numpy(fr.syndrome).cuda()
    out = code.decode(d_llr, d_syn, n_iter, 1, want_posterior=True)
    torch.cuda.synchronize()
    post = out.posterior.cpu().numpy()
    hard = out.hard.cpu().numpy()
    assert (out.iters.cpu().numpy() == n_iter).all() and (out.passed.cpu().numpy() == 0).all()
    sample = np.array([0, 9, 18, 27, 37, 45, 54, 63])
    ref = oracle_lib.decode(base, Z, fr.llr[sample], fr.syndrome[sample], n_iter, 1)
    assert (ref.passed == 0).all() and (ref.iters == n_iter).all()
    case = PC.compare_fixed(oracle_lib, base, Z, fr.llr[sample], fr.syndrome[sample], n_iter, "cfg4 batch",
                            hard[sample], post[sample], frame_ids=sample)
    assert case.ok and not any(f.unpinned for f in case.frames), case.failures()
    print("cfg4 sampled frames: max err", max(f.err for f in case.frames))
    for f in (0, 37, 63):
        one = code.decode(d_llr[f:f + 1], d_syn[f:f + 1], n_iter, 1, want_posterior=True)
        torch.cuda.synchronize()
        assert torch.equal(one.posterior[0], out.posterior[f]) and torch.equal(one.hard[0], out.hard[f])
    # frame independence inside the batch, for EVERY frame: the batch reversed gives the reversed outputs bit for bit
    rev = code.decode(d_llr.flip(0).contiguous(), d_syn.flip(0).contiguous(), n_iter, 1, want_posterior=True)
    torch.cuda.synchronize()
    assert torch.equal(rev.posterior.flip(0), out.posterior) and torch.equal(rev.hard.flip(0), out.hard)


def assert_stop_parity(sp, n_frames):
    """north_star: "with early stop enabled the frame-error rate must be statistically consistent with the oracle".
    Both sides decode the SAME inputs, so the comparison is per frame: discordant pass flags per point must lie inside
    the binomial 95 % band around zero disagreement (expected 0, at most 1 of 32), every word the GPU
    reports as decoded must satisfy H x = s, and frames decoded on both sides must give the same word."""
    print(f"{sp.label}: FER gpu {sp.fer_gpu:.3f} oracle {sp.fer_oracle:.3f}; discordant pass flags "
          f"{sp.discordant_pass}/{n_frames}, discordant iteration counts {sp.discordant_iters}/{n_frames}, "
          f"iters_gpu - iters_oracle histogram {sp.diff_hist}")
    lo, hi = PC.binomial_band_95(n_frames, sp.fer_oracle)
    assert lo <= sp.fer_gpu <= hi, f"{sp.label}: GPU FER {sp.fer_gpu} outside the 95 % band [{lo:.3f}, {hi:.3f}]"
    assert sp.discordant_pass <= 1, f"{sp.label}: {sp.discordant_pass} discordant pass flags"
    assert sp.gpu_words_valid and sp.hard_mismatch_frames == 0
    assert sp.discordant_iters <= max(1, n_frames // 16), f"{sp.label}: iteration counts differ on {sp.discordant_iters} frames"


@pytest.mark.parametrize("snr_point", [0, 1, 2, 3, 4, 5])
def test_config5_fer_vs_oracle(oracle_lib, B, snr_point):
    """Config 5 as specified (32 frames per point, six SNR points, max 300 iterations, early stop on) on its base
    graph lifted by Z = 2000 (the oracle finishes 192 frames in minutes): per-frame pass flags and iteration counts."""
    cfg, base, Z, fr = W.make_config(5, snr_point=snr_point, Z=2000)
    assert fr.llr.shape[0] == 32 and cfg.max_iter == 300
    hard, iters, passed, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, want_posterior=False)
    sp = PC.compare_stop(oracle_lib, base, Z, fr.llr, fr.syndrome, cfg.max_iter, f"cfg5 Z=2000 point {snr_point}",
                         hard, iters, passed)
    assert_stop_parity(sp, 32)


@pytest.mark.parametrize("snr_point", [3, 4, 5])
def test_config5_full_size_sampled(oracle_lib, B, snr_point):
    """Config 5 at full Z = 10,000 inside the benched batch of 32 frames: the oracle decodes 4 sampled frames of the
    waterfall points one by one (the frames run concurrently on the host cores)."""
    cfg, base, Z, fr = W.make_config(5, snr_point=snr_point)
    sample = np.array([0, 11, 21, 31])
    hard, iters, passed, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, want_posterior=False)
    sp = PC.compare_stop(oracle_lib, base, Z, fr.llr[sample], fr.syndrome[sample], cfg.max_iter,
                         f"cfg5 full size point {snr_point} frames {sample.tolist()}", hard[sample], iters[sample],
                         passed[sample])
    print(f"  batch of 32: gpu pass {int(passed.sum())}/32, iterations {iters.min()}..{iters.max()}")
    assert sp.discordant_pass == 0 and sp.discordant_iters == 0 and sp.gpu_words_valid and sp.hard_mismatch_frames == 0


# ------------------------------------------------------------------------------------ pins applied to the GPU
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_gpu_exact_map_on_trees(B, seed):
    """The CUDA path against brute-force bitwise MAP directly (no oracle involved): exact on cycle-free codes as
    long as no message reaches the clamp."""
    rng = np.random.default_rng(seed)
    base = random_tree_code(rng, n_target=15, max_check_deg=5)
    m, n = base.shape
    H = dense_h(base, 1)
    Q = rng.normal(0.0, 1.5, size=n).astype(np.float32)
    s = rng.integers(0, 2, size=m, dtype=np.uint8)
    want = bitwise_map_llr(H, s, Q)
    hard, iters, passed, post = gpu_decode(B, base, 1, Q[None], s[None], 2 * n, 0)
    np.testing.assert_allclose(post[0], want, rtol=2e-5, atol=2e-5)
    decided = np.abs(want) > HARD_MIN
    np.testing.assert_array_equal(hard[0][decided], (want < 0).astype(np.uint8)[decided])


def test_gpu_syndrome_codeword_equivalence_bit_exact(B):
    cfg, base, Z, fr = W.make_config(1, n_frames=4)
    sign = (1.0 - 2.0 * fr.x.astype(np.float32))
    h1, i1, p1, post1 = gpu_decode(B, base, Z, fr.llr, fr.syndrome, 20, 0)
    h2, i2, p2, post2 = gpu_decode(B, base, Z, fr.llr * sign, np.zeros_like(fr.syndrome), 20, 0)
    np.testing.assert_array_equal(post1, post2 * sign)
    np.testing.assert_array_equal(h1 ^ fr.x, h2)
    np.testing.assert_array_equal(p1, p2)


@pytest.mark.parametrize("A", [25.0, 1e4])
def test_gpu_noiseless_limit_and_max_iter_zero(B, A):
    cfg, base, Z, fr = W.make_config(1, n_frames=3)
    llr = (A * (1.0 - 2.0 * fr.x.astype(np.float32))).astype(np.float32)
    hard, iters, passed, post = gpu_decode(B, base, Z, llr, fr.syndrome, 10, 1)
    np.testing.assert_array_equal(hard, fr.x)
    np.testing.assert_array_equal(iters, 1)
    np.testing.assert_array_equal(passed, 1)
    assert np.isfinite(post).all() and (np.sign(post) == np.sign(llr)).all()
    hard, iters, passed, post = gpu_decode(B, base, Z, llr, fr.syndrome, 0, 1)
    np.testing.assert_array_equal(hard, fr.x)
    np.testing.assert_array_equal(iters, 0)
    np.testing.assert_array_equal(passed, 1)
    np.testing.assert_array_equal(post, llr)
    # max_iter = 0 on a noisy frame: decisions from the channel alone, pass by direct check
    hard, iters, passed, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, 0, 0)
    np.testing.assert_array_equal(hard, (fr.llr < 0).astype(np.uint8))
    np.testing.assert_array_equal(passed.astype(bool), (W.syndrome_of(base, Z, hard) == fr.syndrome).all(axis=1))


@pytest.mark.parametrize("k", range(8))
def test_gpu_decision_tie_rule(oracle_lib, B, k):
    """P:361 (reading S4) through the C ABI: posteriors that are exactly zero decide bit 0 (tests/helpers.tie_cases:
    a variable without checks at Q = +0.0 / -0.0, and a variable between two clamped degree-1 checks at Q = -/+60)."""
    base, Z, llr, syn, max_iter, ties = tie_cases()[k]
    ref = oracle_lib.decode(base, Z, llr[None], syn[None], max_iter, 0)
    hard, iters, passed, post = gpu_decode(B, base, Z, llr[None], syn[None], max_iter, 0)
    assert (post[0, ties] == 0.0).all()
    assert (hard[0, ties] == 0).all()
    np.testing.assert_array_equal(hard, ref.hard)
    np.testing.assert_array_equal(passed, ref.passed)
    if max_iter > 0 and base.shape[1] == 1 and syn[0] == 0:
        below = (llr - np.float32(1e-3))
        hard, iters, passed, post = gpu_decode(B, base, Z, below[None], syn[None], max_iter, 0)
        assert (post[0] < 0).all() and (hard[0] == 1).all()


def test_gpu_frame_independence_and_permutation(B):
    cfg, base, Z, fr = W.make_config(1)
    h, i, p, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, 30, 1)
    perm = np.random.default_rng(7).permutation(len(fr.llr))
    h2, i2, p2, post2 = gpu_decode(B, base, Z, fr.llr[perm], fr.syndrome[perm], 30, 1)
    np.testing.assert_array_equal(post[perm], post2)
    np.testing.assert_array_equal(h[perm], h2)
    np.testing.assert_array_equal(i[perm], i2)
    h3, i3, p3, post3 = gpu_decode(B, base, Z, fr.llr[5:6], fr.syndrome[5:6], 30, 1)
    np.testing.assert_array_equal(post[5], post3[0])
    assert i[5] == i3[0] and p[5] == p3[0]


# ------------------------------------------------------------------------------------------- degenerate codes
def _random_code(rng, mb, nb, Z, density):
    base = np.full((mb, nb), -1, dtype=np.int32)
    mask = rng.random((mb, nb)) < density
    base[mask] = rng.integers(0, Z, size=int(mask.sum()))
    return base


@pytest.mark.parametrize("case", ["irregular", "dv_up_to_30", "dv_up_to_64", "many_rows_global_tables",
                                  "two_deg1_in_a_row", "identity", "zero_column", "deg1_check", "Z1"])
def test_degenerate_and_general_codes(oracle_lib, B, case):
    rng = np.random.default_rng(abs(hash(case)) % 2 ** 31 if False else sum(map(ord, case)))
    n_iter = 6
    if case == "irregular":
        Z, base = 37, _random_code(rng, 6, 12, 37, 0.4)
    elif case == "dv_up_to_30":
        Z, base = 19, _random_code(rng, 30, 8, 19, 0.8)
    elif case == "dv_up_to_64":
        Z, base = 7, _random_code(rng, 64, 5, 7, 0.9)
    elif case == "many_rows_global_tables":     # > 128 base rows and > 256 edges: tables read from global memory
        Z, base = 5, _random_code(rng, 150, 60, 5, 0.06)
    elif case == "two_deg1_in_a_row":
        Z = 11
        base = np.full((3, 6), -1, dtype=np.int32)
        base[0, [0, 1, 2, 3]] = [1, 5, 0, 7]    # columns 2 and 3 are both degree 1 in row 0
        base[1, [0, 1, 4]] = [2, 3, 4]
        base[2, [0, 1, 5]] = [9, 10, 6]
    elif case == "identity":                    # every column degree 1, one per row: everything is absorbed
        Z = 9
        base = np.full((4, 4), -1, dtype=np.int32)
        base[np.arange(4), np.arange(4)] = [0, 3, 8, 1]
    elif case == "zero_column":
        Z, base = 13, _random_code(rng, 4, 7, 13, 0.5)
        base[:, 2] = -1
    elif case == "deg1_check":                  # a check with a single (active) variable: |m| = clamp
        Z = 8
        base = np.full((3, 3), -1, dtype=np.int32)
        base[0, 0] = 3
        base[1, [0, 1, 2]] = [1, 2, 5]
        base[2, [1, 2]] = [0, 7]
    else:
        Z, base = 1, _random_code(rng, 7, 12, 1, 0.35)
    mb, nb = base.shape
    F = 3
    llr = rng.normal(0.4, 1.2, size=(F, nb * Z)).astype(np.float32)
    syn = rng.integers(0, 2, size=(F, mb * Z), dtype=np.uint8)
    for it in (0, 1, n_iter):
        assert_parity(oracle_lib, B, base, Z, llr, syn, it, case)
    ref = oracle_lib.decode(base, Z, llr, syn, 25, 1)
    hard, iters, passed, post = gpu_decode(B, base, Z, llr, syn, 25, 1)
    np.testing.assert_array_equal(passed, ref.passed)
    np.testing.assert_array_equal(iters, ref.iters)


def test_decode_host_matches_device_path(B, monkeypatch):
    cfg, base, Z, fr = W.make_config(1)
    code = B.QCLDPCCode(base, Z)
    h, i, p, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, 30, 1)
    out = code.decode_host(fr.llr, fr.syndrome, 30, 1, want_posterior=True)
    np.testing.assert_array_equal(out.hard, h)
    np.testing.assert_array_equal(out.iters, i)
    np.testing.assert_array_equal(out.passed, p)
    np.testing.assert_array_equal(out.posterior, post)
    out2 = code.decode_host(fr.llr, fr.syndrome, 30, 1, want_posterior=False)
    np.testing.assert_array_equal(out2.hard, h)
    assert B.qcldpc_last_launch_count() > 0
    # a batch whose frames all stop early: same outputs from both paths, and with the host-driven loop
    # (QCLDPC_LOOP=stream) the host path ends the launch sequence once nothing is live while the device-pointer path
    # enqueues all max_iter iterations (with the default graph loop both end on the device:
    # test_device_loop_stops_issuing_when_the_batch_has_stopped)
    conv = np.nonzero(p)[0][:6]
    h2, i2, p2, post2 = gpu_decode(B, base, Z, fr.llr[conv], fr.syndrome[conv], 400, 1)
    out3 = code.decode_host(fr.llr[conv], fr.syndrome[conv], 400, 1, want_posterior=True)
    assert p2.all() and i2.max() < 64
    np.testing.assert_array_equal(out3.hard, h2)
    np.testing.assert_array_equal(out3.iters, i2)
    np.testing.assert_array_equal(out3.passed, p2)
    np.testing.assert_array_equal(out3.posterior, post2)
    monkeypatch.setenv("QCLDPC_LOOP", "stream")
    code_s = B.QCLDPCCode(base, Z)
    monkeypatch.delenv("QCLDPC_LOOP")
    PC.gpu_decode(B, code_s, Z, fr.llr[conv], fr.syndrome[conv], 400, 1)
    n_dev = B.qcldpc_last_launch_count()
    out4 = code_s.decode_host(fr.llr[conv], fr.syndrome[conv], 400, 1, want_posterior=True)
    n_host = B.qcldpc_last_launch_count()
    np.testing.assert_array_equal(out4.iters, i2)
    np.testing.assert_array_equal(out4.posterior, post2)
    assert n_host < n_dev // 3


def test_decode_host_check_from_iter(oracle_lib, B):
    """qcldpc_decode_host_ex: the early-termination scheduling on the host-buffer path."""
    cfg, base, Z, fr = W.make_config(1)
    code = B.QCLDPCCode(base, Z)
    for check_from in (1, 9, 60):
        ref = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, check_from=check_from)
        out = code.decode_host(fr.llr, fr.syndrome, cfg.max_iter, 1, want_posterior=True, check_from_iter=check_from)
        np.testing.assert_array_equal(out.iters, ref.iters)
        np.testing.assert_array_equal(out.passed, ref.passed)
        dev = gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, check_from_iter=check_from)
        np.testing.assert_array_equal(out.hard, dev[0])
        np.testing.assert_array_equal(out.posterior, dev[3])
    with pytest.raises(ValueError):
        code.decode_host(fr.llr.astype(np.float64), fr.syndrome, 5, 0)        # wrong dtype must not be read as fp32
    with pytest.raises(ValueError):
        code.decode_host(fr.llr[:, ::2], fr.syndrome, 5, 0)                     # non-contiguous


@pytest.mark.parametrize("max_iter", [14, 15, 25, 26, 27, 37, 38, 39, 49, 61, 120])
def test_device_loop_matches_stream_loop_and_oracle(oracle_lib, B, max_iter, monkeypatch):
    """The iteration loop as a graph WHILE node (default) against one launch per iteration from the host
    (QCLDPC_LOOP=stream, read at handle creation) and against the oracle, for budgets on both sides of every body
    boundary (pre-loop 2..13 iterations, bodies of 12), early stop on and off."""
    cfg, base, Z, fr = W.make_config(1)
    llr = np.concatenate([fr.llr, 25.0 * (1.0 - 2.0 * fr.x[:2].astype(np.float32))])   # + two noiseless frames
    syn = np.concatenate([fr.syndrome, fr.syndrome[:2]])
    code_g = B.QCLDPCCode(base, Z)
    monkeypatch.setenv("QCLDPC_LOOP", "stream")
    code_s = B.QCLDPCCode(base, Z)
    monkeypatch.delenv("QCLDPC_LOOP")
    for early in (1, 0):
        g = PC.gpu_decode(B, code_g, Z, llr, syn, max_iter, early)
        assert B.qcldpc_last_loop_mode() == 1
        s_ = PC.gpu_decode(B, code_s, Z, llr, syn, max_iter, early)
        assert B.qcldpc_last_loop_mode() == 0
        for a, b in zip(g, s_):
            np.testing.assert_array_equal(a, b)
        ref = oracle_lib.decode(base, Z, llr, syn, max_iter, early)
        # past ~50 iterations the two chaotic frames of config 1 stop (or not) on rounding noise: frames on which the
        # oracle's own float instantiation disagrees with its double one are compared between the two loops only
        ref32 = oracle_lib.decode(base, Z, llr, syn, max_iter, early, precision=32)
        stable = (ref32.iters == ref.iters) & (ref32.passed == ref.passed)
        assert stable.sum() >= len(stable) - 2
        np.testing.assert_array_equal(g[1][stable], ref.iters[stable])
        np.testing.assert_array_equal(g[2][stable], ref.passed[stable])
        ok = ref.passed.astype(bool) & stable
        np.testing.assert_array_equal(g[0][ok], ref.hard[ok])


def test_device_loop_stops_issuing_when_the_batch_has_stopped(B):
    """qcldpc_decode only enqueues, yet a batch whose frames have all stopped must not pay for max_iter launches: the
    WHILE loop ends on the device.  Also: a second call with the same arguments re-launches the cached graph."""
    cfg, base, Z, fr = W.make_config(1)
    code = B.QCLDPCCode(base, Z)
    h, i, p, post = gpu_decode(B, base, Z, fr.llr, fr.syndrome, 50, 1)
    conv = np.nonzero(p)[0][:6]
    d_llr = torch.from_numpy(fr.llr[conv]).cuda()
    d_syn = torch.from_numpy(fr.syndrome[conv]).cuda()
    ws = torch.empty(code.workspace_bytes(len(conv)), dtype=torch.uint8, device="cuda")
    out = code.decode(d_llr, d_syn, 4000, 1, want_posterior=True, workspace=ws)
    assert B.qcldpc_last_loop_mode() == 1
    issued = code.iterations_issued(len(conv), ws)
    iters = out.iters.cpu().numpy()
    assert out.passed.cpu().numpy().all() and iters.max() < 64
    np.testing.assert_array_equal(iters, i[conv])
    # the last check that can stop a frame runs two launches after its iteration; the loop looks at the count of live
    # frames once per body of 12, and the first 2..13 iterations run before the loop
    assert iters.max() + 2 <= issued <= iters.max() + 2 + 12 + 13, (issued, iters.max())
    out2 = code.decode(d_llr, d_syn, 4000, 1, want_posterior=True, workspace=ws, out=out)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(out2.iters.cpu().numpy(), iters)
    np.testing.assert_array_equal(out2.posterior.cpu().numpy()[:, :64], post[conv][:, :64])
    # a batch that never stops issues exactly max_iter iterations
    stuck = np.nonzero(p == 0)[0][:2]
    d_llr2 = torch.from_numpy(fr.llr[stuck]).cuda()
    d_syn2 = torch.from_numpy(fr.syndrome[stuck]).cuda()
    ws2 = torch.empty(code.workspace_bytes(len(stuck)), dtype=torch.uint8, device="cuda")
    code.decode(d_llr2, d_syn2, 77, 1, want_posterior=False, workspace=ws2)
    assert code.iterations_issued(len(stuck), ws2) == 77


def test_decode_inside_a_callers_graph_capture(B):
    """A caller that captures its stream into a CUDA graph of its own gets the per-iteration launches as nodes of that
    graph (no graph launched inside a capture); replaying the captured graph reproduces the plain decode."""
    cfg, base, Z, fr = W.make_config(1)
    code = B.QCLDPCCode(base, Z)
    d_llr = torch.from_numpy(fr.llr).cuda()
    d_syn = torch.from_numpy(fr.syndrome).cuda()
    ws = torch.empty(code.workspace_bytes(len(fr.llr)), dtype=torch.uint8, device="cuda")
    ref = code.decode(d_llr, d_syn, 30, 1, want_posterior=True)
    torch.cuda.synchronize()
    out = B.DecodeResult(torch.zeros_like(ref.hard), torch.zeros_like(ref.iters), torch.zeros_like(ref.passed),
                         torch.zeros_like(ref.posterior))
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        code.decode(d_llr, d_syn, 30, 1, want_posterior=True, workspace=ws, out=out)
        assert B.qcldpc_last_loop_mode() == 0
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out.hard, ref.hard) and torch.equal(out.iters, ref.iters)
    assert torch.equal(out.passed, ref.passed) and torch.equal(out.posterior, ref.posterior)


def test_gpu_argument_errors(B):
    cfg, base, Z, fr = W.make_config(1, n_frames=2)
    code = B.QCLDPCCode(base, Z)
    d_llr = torch.from_numpy(fr.llr).cuda()
    d_syn = torch.from_numpy(fr.syndrome).cuda()
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.QCLDPCError) as ei:
        code.decode(d_llr, d_syn, 5, 0, workspace=small)
    assert ei.value.status == -3
    with pytest.raises(B.QCLDPCError) as ei:
        code.decode(d_llr, d_syn, -1, 0)
    assert ei.value.status == -1
    with pytest.raises(ValueError):
        code.decode(d_llr[:, :-1], d_syn, 5, 0)


@pytest.mark.gpu
@pytest.mark.parametrize("which", ["config1_exact", "ensemble_generic"])
def test_gpu_no_writes_outside_the_buffers(B, which):
    """compute-sanitizer is not available on the GPU pool: guard bands instead.  Every buffer handed to the C ABI sits
    inside a larger allocation whose surroundings are filled with a pattern; nothing outside may change, and the
    result must equal the plain call's."""
    if which == "config1_exact":
        cfg, base, Z, fr = W.make_config(1)
        code = B.QCLDPCCode(base, Z)
        llr, syn = fr.llr, fr.syndrome
    else:
        spec = W.paper_ensemble_spec(400, 50)
        ens = W.make_paper_ensemble(spec)
        fr = W.make_frames_sparse(*ens, 50, W.sigma_for_gap(0.02, 2.0), 5, 31337)
        code = B.QCLDPCCode.from_sparse(*ens, 50)
        llr, syn = fr.llr, fr.syndrome
    F, n, m = llr.shape[0], code.n, code.m
    G = 4096                                               # guard bytes (a multiple of 256: keeps the alignment)

    def guarded(nbytes, dtype):
        raw = torch.full((G + nbytes + G,), 0xAB, dtype=torch.uint8, device="cuda")
        return raw, raw[G:G + nbytes].view(dtype)

    need = code.workspace_bytes(F)
    need_al = (need + 255) // 256 * 256
    ws_raw, ws = guarded(need_al, torch.uint8)
    hard_raw, hard = guarded(F * n, torch.uint8)
    it_raw, iters = guarded(F * 4, torch.int32)
    ps_raw, passed = guarded((F + 255) // 256 * 256, torch.uint8)
    po_raw, post = guarded(F * n * 4, torch.float32)
    out = B.DecodeResult(hard.view(F, n), iters, passed[:F], post.view(F, n))
    d_llr, d_syn = torch.from_numpy(llr).cuda(), torch.from_numpy(syn).cuda()
    for early in (0, 1):
        code.decode(d_llr, d_syn, 30, early, want_posterior=True, workspace=ws, out=out)
        torch.cuda.synchronize()
        ref = code.decode(d_llr, d_syn, 30, early, want_posterior=True)
        torch.cuda.synchronize()
        assert torch.equal(out.hard, ref.hard) and torch.equal(out.iters, ref.iters)
        assert torch.equal(out.posterior, ref.posterior) and torch.equal(out.passed, ref.passed)
        for raw, body in ((ws_raw, need_al), (hard_raw, F * n), (it_raw, F * 4), (ps_raw, (F + 255) // 256 * 256),
                          (po_raw, F * n * 4)):
            assert bool((raw[:G] == 0xAB).all()) and bool((raw[G + body:] == 0xAB).all())


@pytest.mark.gpu
@pytest.mark.parametrize("max_iter", [1, 2, 3, 4, 5, 12, 13, 14])
def test_early_stop_with_small_iteration_budgets(oracle_lib, B, max_iter):
    """The early-exit check of iteration T rides two launches behind pass T: budgets around that lag, and frames that
    pass exactly at max_iter - 2, max_iter - 1 and max_iter, must give the oracle's flags, counts and outputs."""
    cfg, base, Z, fr = W.make_config(1)
    llr = np.concatenate([fr.llr, 25.0 * np.sign(fr.llr[:2])])             # two noiseless frames: pass at iteration 1
    # noiseless copies of frames 0, 1 with the signs of the TRUE words
    llr[-2:] = 25.0 * (1.0 - 2.0 * fr.x[:2].astype(np.float32))
    syn = np.concatenate([fr.syndrome, fr.syndrome[:2]])
    ref = oracle_lib.decode(base, Z, llr, syn, max_iter, 1)
    hard, iters, passed, post = gpu_decode(B, base, Z, llr, syn, max_iter, 1)
    np.testing.assert_array_equal(passed, ref.passed)
    np.testing.assert_array_equal(iters, ref.iters)
    assert iters[-1] == 1 and iters[-2] == 1 and passed[-2:].all()
    ok = ref.passed.astype(bool)
    np.testing.assert_array_equal(hard[ok], ref.hard[ok])
    assert rel_err(post, ref.posterior).max() <= TOL


@pytest.mark.gpu
def test_gpu_two_streams_share_one_handle(B):
    """include/qcldpc.h: the handle is immutable and may be used concurrently from several streams with distinct
    workspaces.  Two decodes of different frames enqueued on two streams must equal the same decodes run alone."""
    cfg, base, Z, fr = W.make_config(3, n_frames=2, Z=1000)
    code = B.QCLDPCCode(base, Z)
    d_llr = torch.from_numpy(fr.llr).cuda()
    d_syn = torch.from_numpy(fr.syndrome).cuda()
    alone = [code.decode(d_llr[k:k + 1], d_syn[k:k + 1], 60, 1, want_posterior=True) for k in range(2)]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = []
    for rep in range(3):
        outs = []
        for k, st in enumerate(streams):
            st.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(st):
                outs.append(code.decode(d_llr[k:k + 1], d_syn[k:k + 1], 60, 1, want_posterior=True, stream=st))
        torch.cuda.synchronize()
        for k in range(2):
            assert torch.equal(outs[k].hard, alone[k].hard) and torch.equal(outs[k].iters, alone[k].iters)
            assert torch.equal(outs[k].posterior, alone[k].posterior) and torch.equal(outs[k].passed, alone[k].passed)


@pytest.mark.gpu
@pytest.mark.parametrize("seed", list(range(16)))
def test_random_codes_against_oracle(oracle_lib, B, seed):
    """Random base matrices (any row and column degree up to the supported 64, degree-0 and degree-1 rows and columns,
    several degree-1 columns in a row), random lifting sizes around the tile sizes of both kernel families, 1-9
    frames (one and two frames per thread), fixed iterations and early stop."""
    rng = np.random.default_rng(9000 + seed)
    Z = int(rng.choice([1, 2, 3, 7, 21, 31, 32, 33, 50, 63, 64, 65, 127, 128, 129, 200, 257]))
    mb = int(rng.integers(2, 13))
    nb = int(rng.integers(mb, mb + 15))
    base = _random_code(rng, mb, nb, Z, float(rng.choice([0.15, 0.3, 0.5, 0.8])))
    if seed % 4 == 0:                                      # a degree-1 diagonal on the right, like the paper's codes
        k = min(mb, nb // 2)
        base[:, nb - k:] = -1
        base[np.arange(k), nb - k + np.arange(k)] = 0
    n_frames = int(rng.integers(1, 10))
    n, m = nb * Z, mb * Z
    x = rng.integers(0, 2, size=(n_frames, n), dtype=np.uint8)
    syn = W.syndrome_of(base, Z, x)
    sigma = float(rng.choice([0.5, 0.8, 1.2]))
    llr = (2.0 * ((1.0 - 2.0 * x) + sigma * rng.standard_normal((n_frames, n))) / sigma ** 2).astype(np.float32)
    n_iter = int(rng.integers(1, 26))
    assert_parity(oracle_lib, B, base, Z, llr, syn, n_iter, f"random seed {seed}")
    ref = oracle_lib.decode(base, Z, llr, syn, 40, 1)
    hard, iters, passed, post = gpu_decode(B, base, Z, llr, syn, 40, 1)
    ref32 = oracle_lib.decode(base, Z, llr, syn, 40, 1, precision=32)
    stable = (ref32.iters == ref.iters) & (ref32.passed == ref.passed)   # frames whose stop does not hinge on rounding
    np.testing.assert_array_equal(passed[stable], ref.passed[stable])
    np.testing.assert_array_equal(iters[stable], ref.iters[stable])
    ok = stable & ref.passed.astype(bool)
    np.testing.assert_array_equal(hard[ok], ref.hard[ok])
    np.testing.assert_array_equal(W.syndrome_of(base, Z, hard[passed.astype(bool)]), syn[passed.astype(bool)])
