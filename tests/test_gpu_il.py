"""GPU tests of the frame-interleaved kernel family (csrc/pass_il.cuh: groups of 32 frames, lane = frame), the path of
batched decodes of the paper's own ensemble (NEXT-1).  Against the oracle, and bit for bit against the generic family
(QCLDPC_IL=0): a frame's result must not depend on the kernel family that decodes it."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1702_07740_b200 import workloads as W  # noqa: E402
from tests import parity_cases as PC  # noqa: E402

TOL = 1e-3


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_1702_07740_b200 import binding
    return binding


def handles(B, monkeypatch, ens, q, force=False):
    """(interleaved family, generic family) handles of one code; force: interleaved for every batch size."""
    if force:
        monkeypatch.setenv("QCLDPC_IL", "2")
    il = B.QCLDPCCode.from_sparse(*ens, q)
    monkeypatch.setenv("QCLDPC_IL", "0")
    gen = B.QCLDPCCode.from_sparse(*ens, q)
    monkeypatch.delenv("QCLDPC_IL")
    return il, gen


def decode(code, llr, syn, max_iter, early):
    out = code.decode(torch.from_numpy(llr).cuda(), torch.from_numpy(syn).cuda(), max_iter, early, want_posterior=True)
    torch.cuda.synchronize()
    return out.hard.cpu().numpy(), out.iters.cpu().numpy(), out.passed.cpu().numpy(), out.posterior.cpu().numpy()


@pytest.mark.parametrize("nb,q,n_iter,F", [(400, 50, 15, 32), (800, 21, 10, 32), (400, 7, 12, 64), (400, 50, 6, 27)])
def test_il_paper_ensemble_fixed_iterations(oracle_lib, B, monkeypatch, nb, q, n_iter, F):
    spec = W.paper_ensemble_spec(nb, q)
    ens = W.make_paper_ensemble(spec)
    fr = W.make_frames_sparse(*ens, q, W.sigma_for_gap(0.02, 0.3), F, 4242)
    il, gen = handles(B, monkeypatch, ens, q)
    got = decode(il, fr.llr, fr.syndrome, n_iter, 0)
    ref = oracle_lib.decode_sparse(*ens, q, fr.llr, fr.syndrome, n_iter, 0)
    err = np.abs(got[3] - ref.posterior) / np.maximum(1.0, np.abs(ref.posterior))
    assert err.max() <= TOL, err.max()
    decided = np.abs(ref.posterior) > 1e-2
    np.testing.assert_array_equal(got[0][decided], ref.hard[decided])
    np.testing.assert_array_equal(got[2], ref.passed)
    assert (got[1] == n_iter).all()
    for a, b in zip(got, decode(gen, fr.llr, fr.syndrome, n_iter, 0)):       # the generic family: bit for bit
        np.testing.assert_array_equal(a, b)


@pytest.mark.parametrize("max_iter", [0, 1, 2, 3, 13, 40, 80])
def test_il_early_stop_mixed_batch(oracle_lib, B, monkeypatch, max_iter):
    """32 frames, converging and not, mixed in the lanes of one group; budgets around the two-launch lag of the check
    and on both sides of the graph loop; flags, counts and the words of decoded frames against the oracle, everything
    against the generic family."""
    spec = W.paper_ensemble_spec(400, 21)
    ens = W.make_paper_ensemble(spec)
    hi = W.make_frames_sparse(*ens, 21, W.sigma_for_gap(0.02, 3.0), 20, 555)
    lo = W.make_frames_sparse(*ens, 21, W.sigma_for_gap(0.02, 0.3), 12, 556)
    order = np.random.default_rng(1).permutation(32)
    llr = np.concatenate([hi.llr, lo.llr])[order]
    syn = np.concatenate([hi.syndrome, lo.syndrome])[order]
    il, gen = handles(B, monkeypatch, ens, 21)
    got = decode(il, llr, syn, max_iter, 1)
    for a, b in zip(got, decode(gen, llr, syn, max_iter, 1)):
        np.testing.assert_array_equal(a, b)
    ref = oracle_lib.decode_sparse(*ens, 21, llr, syn, max_iter, 1)
    np.testing.assert_array_equal(got[2], ref.passed)
    np.testing.assert_array_equal(got[1], ref.iters)
    ok = ref.passed.astype(bool)
    if max_iter >= 40:
        assert 0 < ok.sum() < 32
    np.testing.assert_array_equal(got[0][ok], ref.hard[ok])
    np.testing.assert_array_equal(W.syndrome_of_sparse(*ens, 21, got[0][ok]), syn[ok])
    assert (np.abs(got[3][ok] - ref.posterior[ok]) <= TOL * np.maximum(1.0, np.abs(ref.posterior[ok]))).all()


def test_il_frame_independence(B, monkeypatch):
    """A frame alone (generic family), in a group of 32 and in the second, ragged group of 59 frames gives the same
    outputs bit for bit, also after its lane neighbours have stopped."""
    spec = W.paper_ensemble_spec(400, 50)
    ens = W.make_paper_ensemble(spec)
    hi = W.make_frames_sparse(*ens, 50, W.sigma_for_gap(0.02, 3.0), 30, 77)
    lo = W.make_frames_sparse(*ens, 50, W.sigma_for_gap(0.02, 0.3), 29, 78)
    order = np.random.default_rng(2).permutation(59)
    llr = np.concatenate([hi.llr, lo.llr])[order]
    syn = np.concatenate([hi.syndrome, lo.syndrome])[order]
    il, gen = handles(B, monkeypatch, ens, 50)
    for early in (0, 1):
        b59 = decode(il, llr, syn, 30, early)
        b32 = decode(il, llr[:32], syn[:32], 30, early)
        for a, b in zip(b59, b32):
            np.testing.assert_array_equal(a[:32], b)
        for f in (0, 7, 31, 32, 45, 58):
            alone = decode(gen, llr[f:f + 1], syn[f:f + 1], 30, early)
            for a, b in zip(b59, alone):
                np.testing.assert_array_equal(a[f], b[0])


@pytest.mark.parametrize("q,F", [(50, 32), (21, 59), (7, 40)])
def test_il_asynchronous_variant_equals_register_variant(B, monkeypatch, q, F):
    """Long columns run the asynchronous variant by default (messages in tensor memory, loads as a cp.async ring);
    QCLDPC_ILA=0 selects the variant with register loads and messages in shared memory, QCLDPC_ILA=1 / 3 other ring
    depths.  Same outputs bit for bit, fixed count and early stop, ragged last group included."""
    spec = W.paper_ensemble_spec(400, q)
    ens = W.make_paper_ensemble(spec)
    hi = W.make_frames_sparse(*ens, q, W.sigma_for_gap(0.02, 3.0), F // 2, 91)
    lo = W.make_frames_sparse(*ens, q, W.sigma_for_gap(0.02, 0.3), F - F // 2, 92)
    llr, syn = np.concatenate([hi.llr, lo.llr]), np.concatenate([hi.syndrome, lo.syndrome])
    default = B.QCLDPCCode.from_sparse(*ens, q)
    others = []
    for depth in ("0", "1", "3"):
        monkeypatch.setenv("QCLDPC_ILA", depth)
        others.append(B.QCLDPCCode.from_sparse(*ens, q))
    monkeypatch.delenv("QCLDPC_ILA")
    for early, it in ((0, 12), (1, 40)):
        ref = decode(default, llr, syn, it, early)
        for other in others:
            for a, b in zip(ref, decode(other, llr, syn, it, early)):
                np.testing.assert_array_equal(a, b)


def test_il_two_decodes_at_once_on_two_streams(B):
    """Two batched decodes in flight at once (two streams, a workspace each): their CTAs share the multiprocessors'
    tensor memory, registers and shared memory; each must give what it gives alone."""
    spec = W.paper_ensemble_spec(400, 50)
    ens = W.make_paper_ensemble(spec)
    code = B.QCLDPCCode.from_sparse(*ens, 50)
    fa = W.make_frames_sparse(*ens, 50, W.sigma_for_gap(0.02, 3.0), 32, 1201)
    fb = W.make_frames_sparse(*ens, 50, W.sigma_for_gap(0.02, 0.3), 64, 1202)
    ins = [(torch.from_numpy(f.llr).cuda(), torch.from_numpy(f.syndrome).cuda()) for f in (fa, fb)]
    alone = [code.decode(l, s, 60, 1, want_posterior=True) for l, s in ins]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for _ in range(3):
        both = []
        for (l, s), st in zip(ins, streams):
            with torch.cuda.stream(st):
                both.append(code.decode(l, s, 60, 1, want_posterior=True, stream=st))
        torch.cuda.synchronize()
        for got, ref in zip(both, alone):
            for a, b in zip(got, ref):
                assert torch.equal(a, b)


def _random_code(rng, mb, nb, Z, density):
    base = np.full((mb, nb), -1, dtype=np.int32)
    mask = rng.random((mb, nb)) < density
    base[mask] = rng.integers(0, Z, size=int(mask.sum()))
    return base


@pytest.mark.parametrize("seed", list(range(12)))
def test_il_random_codes_against_oracle(oracle_lib, B, monkeypatch, seed):
    """The interleaved family forced onto random base matrices (any row and column degree up to 64, empty and
    degree-1 rows and columns, several degree-1 columns in a row) and batch sizes that leave lanes empty."""
    rng = np.random.default_rng(7000 + seed)
    Z = int(rng.choice([1, 2, 3, 7, 21, 31, 32, 33, 50, 64, 65, 130]))
    mb = int(rng.integers(2, 13))
    nb = int(rng.integers(mb, mb + 15))
    base = _random_code(rng, mb, nb, Z, float(rng.choice([0.15, 0.3, 0.5, 0.8])))
    if seed % 4 == 0:
        k = min(mb, nb // 2)
        base[:, nb - k:] = -1
        base[np.arange(k), nb - k + np.arange(k)] = 0
    if seed == 5:                                              # long columns: four partial sums
        base = _random_code(rng, 40, 6, Z, 0.9)
        mb, nb = base.shape
    F = int(rng.choice([1, 5, 31, 32, 33, 40]))
    r, c = np.nonzero(base >= 0)
    ens = (r.astype(np.int32), c.astype(np.int32), base[r, c].astype(np.int32), mb, nb)
    x = rng.integers(0, 2, size=(F, nb * Z), dtype=np.uint8)
    syn = W.syndrome_of(base, Z, x)
    sigma = float(rng.choice([0.5, 0.8, 1.2]))
    llr = (2.0 * ((1.0 - 2.0 * x) + sigma * rng.standard_normal(x.shape)) / sigma ** 2).astype(np.float32)
    il, gen = handles(B, monkeypatch, ens, Z, force=True)
    n_iter = int(rng.integers(1, 20))
    for early, it in ((0, n_iter), (1, 40), (0, 0)):
        got = decode(il, llr, syn, it, early)
        for a, b in zip(got, decode(gen, llr, syn, it, early)):
            np.testing.assert_array_equal(a, b)
    case = PC.compare_fixed(oracle_lib, base, Z, llr, syn, n_iter, f"il random {seed}", *[decode(il, llr, syn, n_iter, 0)[k] for k in (0, 3)])
    assert case.ok, case.failures()


def test_il_full_size_sampled(oracle_lib, B):
    """The paper's q = 50 code at full size (n = 1e6), 32 frames in one group -- the launch shape bench.py --ensemble 50
    times -- at the paper's operating point: sampled frames against the oracle after 10 iterations."""
    spec = W.paper_ensemble_spec(20000, 50)
    ens = W.make_paper_ensemble(spec)
    sigma = (2.0 ** (2.0 * 0.02 / 0.99) - 1.0) ** -0.5
    fr = W.make_frames_sparse(*ens, 50, sigma, 32, 31415)
    code = B.QCLDPCCode.from_sparse(*ens, 50)
    got = decode(code, fr.llr, fr.syndrome, 10, 1)
    sample = np.array([0, 13, 31])
    ref = oracle_lib.decode_sparse(*ens, 50, fr.llr[sample], fr.syndrome[sample], 10, 1)
    err = np.abs(got[3][sample] - ref.posterior) / np.maximum(1.0, np.abs(ref.posterior))
    assert err.max() <= TOL, err.max()
    decided = np.abs(ref.posterior) > 1e-2
    np.testing.assert_array_equal(got[0][sample][decided], ref.hard[decided])
    np.testing.assert_array_equal(got[2][sample], ref.passed)
    np.testing.assert_array_equal(got[1][sample], ref.iters)
