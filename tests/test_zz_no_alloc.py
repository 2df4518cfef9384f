"""GPU test of qcldpc_decode_static (include/qcldpc.h): the decode for callers that cannot allocate device memory.  Its
workspace is a 16 MiB device array inside the library, shared by every call on a GPU and never cleared between calls, so
the outputs of calls IN A ROW are compared with the existing path's (qcldpc_decode_ex with a workspace of the caller's) on
the same inputs, within the tolerance of the parity tests (tests/parity_cases.py: |dL| <= 1e-3 max(1, |L|), hard bits
where |L| > 1e-2; flags and iteration counts exactly).

This file sorts last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1702_07740_b200 import workloads as W  # noqa: E402
from tests import parity_cases as PC  # noqa: E402


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_1702_07740_b200 import binding
    return binding


def _outputs(B, F, n, posterior=True):
    """Output buffers the caller owns, filled with garbage that no decode produces."""
    return B.DecodeResult(torch.full((F, n), 7, dtype=torch.uint8, device="cuda"),
                          torch.full((F,), -5, dtype=torch.int32, device="cuda"),
                          torch.full((F,), 9, dtype=torch.uint8, device="cuda"),
                          torch.full((F, n), float("nan"), dtype=torch.float32, device="cuda") if posterior else None)


def _same(got, ref):
    """decode_static's outputs against the existing path's, both DecodeResults on the device."""
    post, post_ref = got.posterior.cpu().numpy(), ref.posterior.cpu().numpy().astype(np.float64)
    assert np.isfinite(post).all()
    err = PC.rel_err(post, post_ref)
    assert err.max() <= PC.TOL, err.max()
    decided = np.abs(post_ref) > PC.HARD_MIN
    np.testing.assert_array_equal(got.hard.cpu().numpy()[decided], ref.hard.cpu().numpy()[decided])
    np.testing.assert_array_equal(got.iters.cpu().numpy(), ref.iters.cpu().numpy())
    np.testing.assert_array_equal(got.passed.cpu().numpy(), ref.passed.cpu().numpy())


def _case(B, cfg_index, Z, n_frames, first_frame):
    cfg, base, Z, fr = W.make_config(cfg_index, n_frames=n_frames, Z=Z, first_frame=first_frame)
    return base, Z, torch.from_numpy(fr.llr).cuda(), torch.from_numpy(fr.syndrome).cuda()


@pytest.mark.parametrize("cfg_index,Z,n_frames", [(1, None, 16), (2, 1000, 2)])
def test_decode_static_matches_decode_on_calls_in_a_row(B, cfg_index, Z, n_frames):
    """Three calls in a row on one stream, nothing in between: frames A with a fixed count, other frames B with early
    stop, frames A again.  Each must equal the existing path on the same inputs: a call may not see what the previous one
    left in the shared array."""
    base, Z, llr_a, syn_a = _case(B, cfg_index, Z, n_frames, 0)
    _, _, llr_b, syn_b = _case(B, cfg_index, Z, n_frames, n_frames)
    code = B.QCLDPCCode(base, Z)
    assert code.workspace_bytes(n_frames) <= B.qcldpc_static_workspace_bytes()
    n = base.shape[1] * Z
    out_a, out_b, out_a2 = (_outputs(B, n_frames, n) for _ in range(3))
    code.decode_static(llr_a, syn_a, 30, 0, out_a)
    code.decode_static(llr_b, syn_b, 60, 1, out_b)
    code.decode_static(llr_a, syn_a, 30, 0, out_a2)
    torch.cuda.synchronize()
    assert B.qcldpc_last_loop_mode() == 0                         # plain launches: no graph was built
    _same(out_a, code.decode(llr_a, syn_a, 30, 0, want_posterior=True))
    _same(out_b, code.decode(llr_b, syn_b, 60, 1, want_posterior=True))
    torch.cuda.synchronize()
    for x, y in zip(out_a, out_a2):                               # the same inputs twice: the same bits
        assert torch.equal(x, y)
    assert (out_a.iters == 30).all()


def test_decode_static_frame_interleaved_family(B):
    """A batch of the paper's own ensemble (small: 400 base columns, q = 7, 32 frames) takes the frame-interleaved
    kernels with their messages in tensor memory; its workspace fits the static array.  Two calls in a row, then one
    captured into the caller's graph, against the existing path."""
    spec = W.paper_ensemble_spec(400, 7)
    ens = W.make_paper_ensemble(spec)
    code = B.QCLDPCCode.from_sparse(*ens, 7)
    F = 32
    assert code.workspace_bytes(F) <= B.qcldpc_static_workspace_bytes()
    fa = W.make_frames_sparse(*ens, 7, W.sigma_for_gap(0.02, 3.0), F, 4711)
    fb = W.make_frames_sparse(*ens, 7, W.sigma_for_gap(0.02, 0.3), F, 4712)
    llr_a, syn_a = torch.from_numpy(fa.llr).cuda(), torch.from_numpy(fa.syndrome).cuda()
    llr_b, syn_b = torch.from_numpy(fb.llr).cuda(), torch.from_numpy(fb.syndrome).cuda()
    out_a, out_b = _outputs(B, F, code.n), _outputs(B, F, code.n)
    code.decode_static(llr_a, syn_a, 40, 1, out_a)
    code.decode_static(llr_b, syn_b, 15, 0, out_b)
    torch.cuda.synchronize()
    ref_a = code.decode(llr_a, syn_a, 40, 1, want_posterior=True)
    _same(out_a, ref_a)
    _same(out_b, code.decode(llr_b, syn_b, 15, 0, want_posterior=True))
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        code.decode_static(llr_a, syn_a, 40, 1, out_a)
    for t in out_a:
        t.zero_()
    g.replay()
    torch.cuda.synchronize()
    _same(out_a, ref_a)


def test_decode_static_rejects_what_does_not_fit(B):
    cfg, base, Z, fr = W.make_config(1, n_frames=1)
    code = B.QCLDPCCode(base, Z)
    F = 256
    assert code.workspace_bytes(F) > B.qcldpc_static_workspace_bytes()
    llr = torch.zeros((F, base.shape[1] * Z), dtype=torch.float32, device="cuda")
    syn = torch.zeros((F, base.shape[0] * Z), dtype=torch.uint8, device="cuda")
    out = _outputs(B, F, base.shape[1] * Z, posterior=False)
    with pytest.raises(B.QCLDPCError) as e:
        code.decode_static(llr, syn, 5, 0, out)
    assert e.value.status == -3                                   # QCLDPC_ERR_WORKSPACE
    assert str(code.workspace_bytes(F)) in str(e.value) and str(B.qcldpc_static_workspace_bytes()) in str(e.value)
    torch.cuda.synchronize()
    assert (out.iters == -5).all() and (out.hard == 7).all()      # nothing ran


def test_decode_static_under_the_callers_graph_capture(B):
    """torch captures in the `global` error mode, in which a cudaMalloc on any thread fails and invalidates the capture:
    a decode_static captured into the caller's graph and replayed twice shows that the call allocates nothing."""
    base, Z, llr, syn = _case(B, 1, None, 16, 0)
    code = B.QCLDPCCode(base, Z)
    n = base.shape[1] * Z
    out = _outputs(B, 16, n)
    code.decode_static(llr, syn, 20, 1, out)                      # warm-up: modules loaded, the array's address known
    torch.cuda.synchronize()
    ref = code.decode(llr, syn, 20, 1, want_posterior=True)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        code.decode_static(llr, syn, 20, 1, out)
    for _ in range(2):
        for t in out:
            t.zero_()
        g.replay()
        torch.cuda.synchronize()
        _same(out, ref)
