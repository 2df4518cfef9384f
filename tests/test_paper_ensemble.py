"""NEXT-1: the paper's own multi-edge ensemble as a workload, and the sparse base-matrix entry points.
CPU part: generator pins against what the paper prints, sparse == dense for the oracle and the harness."""
from __future__ import annotations

import numpy as np
import pytest

from paper_1702_07740_b200 import workloads as W


def _triplets(base):
    r, c = np.nonzero(base >= 0)
    return r.astype(np.int32), c.astype(np.int32), base[r, c].astype(np.int32)


def test_ensemble_counts_match_the_papers_printed_numbers():
    """P:292-296 (Omega, Psi), P:302 (H is 9.8e5 x 1e6), P:328 (q = 21: n = 1.008e6 keeps rate 0.02; q = 50: n = 1e6,
    rate 0.01995), P:499 (connections: 3,337,494 random / 160,185 q = 21 / 66,747 q = 50; the few missing edges are
    parallel edges the paper's sampler dropped, ours re-draws them)."""
    s21 = W.paper_ensemble_spec(48000, 21)
    assert s21.n == 1_008_000 and s21.mb / s21.nb == pytest.approx(0.98, abs=1e-12)        # rate exactly 0.02
    assert (s21.rows_t3, s21.rows_t7) == (17 * 48000 // 1600, 3 * 48000 // 320)             # reading G1 (swapped)
    assert abs(s21.base_edges - 160_185) <= 20 and s21.base_edges == 160_200
    s50 = W.paper_ensemble_spec(20000, 50)
    assert s50.n == 1_000_000
    assert 1.0 - s50.mb / s50.nb == pytest.approx(0.01995, abs=1e-4)                        # "R_code = 0.01995"
    assert abs(s50.base_edges - 66_747) <= 5 and s50.base_edges == 66_750
    assert abs(s50.base_edges * 50 - 3_337_494) <= 10                                        # the random code's count
    # socket balance per 1e6 columns: printed Psi does not balance type 1, the swapped one does (G1)
    vn1 = 22_500 * 2 + 17_500 * 3
    assert vn1 == 97_500 and 9_375 * 3 + 10_625 * 7 == 102_500 and 10_625 * 3 + 9_375 * 7 == 97_500
    assert 40_000 * 57 == 600_000 * 2 + 360_000 * 3                                          # type 2 balances as printed


@pytest.mark.parametrize("nb,q", [(400, 50), (800, 21), (20000, 50)])
def test_ensemble_graph_satisfies_the_degree_distribution(nb, q):
    spec = W.paper_ensemble_spec(nb, q)
    rows, cols, shifts, mb, nbb = W.make_paper_ensemble(spec)
    assert (mb, nbb) == (spec.mb, spec.nb) and len(rows) == spec.base_edges
    key = rows.astype(np.int64) * nb + cols
    assert len(np.unique(key)) == len(key)                                                   # one circulant per block
    nc, n_top = spec.n_core2 + spec.n_core3, spec.rows_t3 + spec.rows_t7
    cdeg, rdeg = np.bincount(cols, minlength=nb), np.bincount(rows, minlength=mb)
    assert (cdeg[:spec.n_core2] == 59).all() and (cdeg[spec.n_core2:nc] == 60).all() and (cdeg[nc:] == 1).all()
    assert (rdeg[:spec.rows_t3] == 3).all() and (rdeg[spec.rows_t3:n_top] == 7).all()
    assert (rdeg[n_top:n_top + spec.rows_l2] == 3).all() and (rdeg[n_top + spec.rows_l2:] == 4).all()
    top = rows < n_top
    assert (cols[top] < nc).all()                                                            # type 1: core x top only
    d1 = cols >= nc
    assert (rows[d1] - n_top == cols[d1] - nc).all() and (shifts[d1] == 0).all()             # unshifted diagonal
    assert shifts.min() >= 0 and shifts.max() < q
    # same structure for another q, different shifts
    r2, c2, p2, _, _ = W.make_paper_ensemble(W.paper_ensemble_spec(nb, q + 1))
    assert (r2 == rows).all() and (c2 == cols).all() and (p2[~d1] != shifts[~d1]).any()


def test_sparse_and_dense_forms_agree(oracle_lib):
    """Oracle and harness: a code given by its non-zero blocks is the same code as its dense base matrix."""
    cfg, base, Z, fr = W.make_config(1, n_frames=3)
    r, c, p = _triplets(base)
    perm = np.random.default_rng(5).permutation(len(r))                                     # any order
    mb, nb = base.shape
    np.testing.assert_array_equal(W.syndrome_of_sparse(r[perm], c[perm], p[perm], mb, nb, Z, fr.x), fr.syndrome)
    np.testing.assert_array_equal(oracle_lib.syndrome_sparse(r, c, p, mb, nb, Z, fr.x), fr.syndrome)
    a = oracle_lib.decode(base, Z, fr.llr, fr.syndrome, 12, 0)
    b = oracle_lib.decode_sparse(r[perm], c[perm], p[perm], mb, nb, Z, fr.llr, fr.syndrome, 12, 0)
    np.testing.assert_array_equal(a.posterior, b.posterior)
    np.testing.assert_array_equal(a.hard, b.hard)
    with pytest.raises(RuntimeError):                                                        # repeated block
        oracle_lib.decode_sparse(np.r_[r, r[:1]], np.r_[c, c[:1]], np.r_[p, p[:1]], mb, nb, Z, fr.llr, fr.syndrome,
                                 1, 0)


def test_ensemble_decodes_at_high_snr(oracle_lib):
    """Sanity of the workload: the reduced ensemble converges well above threshold and stalls near it."""
    spec = W.paper_ensemble_spec(400, 50)
    rows, cols, shifts, mb, nb = W.make_paper_ensemble(spec)
    hi = W.make_frames_sparse(rows, cols, shifts, mb, nb, 50, W.sigma_for_gap(0.02, 4.0), 2, 777)
    out = oracle_lib.decode_sparse(rows, cols, shifts, mb, nb, 50, hi.llr, hi.syndrome, 60, 1)
    assert out.passed.all() and (out.iters < 60).all()
    np.testing.assert_array_equal(oracle_lib.syndrome_sparse(rows, cols, shifts, mb, nb, 50, out.hard), hi.syndrome)


# ---------------------------------------------------------------------------------------------------- GPU (C ABI)
TOL = 1e-3


def _gpu_decode(code, llr, syn, max_iter, early_stop):
    import torch
    out = code.decode(torch.from_numpy(llr).cuda(), torch.from_numpy(syn).cuda(), max_iter, early_stop,
                      want_posterior=True)
    torch.cuda.synchronize()
    return out.hard.cpu().numpy(), out.iters.cpu().numpy(), out.passed.cpu().numpy(), out.posterior.cpu().numpy()


@pytest.mark.gpu
def test_gpu_sparse_create_equals_dense_create():
    from paper_1702_07740_b200 import binding as B
    cfg, base, Z, fr = W.make_config(1)
    r, c, p = _triplets(base)
    perm = np.random.default_rng(3).permutation(len(r))
    dense = _gpu_decode(B.QCLDPCCode(base, Z), fr.llr, fr.syndrome, 20, 0)
    sparse = _gpu_decode(B.QCLDPCCode.from_sparse(r[perm], c[perm], p[perm], base.shape[0], base.shape[1], Z),
                         fr.llr, fr.syndrome, 20, 0)
    for a, b in zip(dense, sparse):
        np.testing.assert_array_equal(a, b)
    with pytest.raises(B.QCLDPCError):
        B.QCLDPCCode.from_sparse(np.r_[r, r[:1]], np.r_[c, c[:1]], np.r_[p, p[:1]], base.shape[0], base.shape[1], Z)


@pytest.mark.gpu
@pytest.mark.parametrize("nb,q,n_iter", [(400, 50, 15), (800, 21, 10), (400, 7, 12)])
def test_gpu_paper_ensemble_fixed_iterations(oracle_lib, nb, q, n_iter):
    """Parity on the paper's ensemble (core degree 59/60, lower checks with 2 or 3 core edges, top checks of degree
    3 and 7) at reduced block length, near threshold: posterior and hard bits against the oracle."""
    from paper_1702_07740_b200 import binding as B
    spec = W.paper_ensemble_spec(nb, q)
    rows, cols, shifts, mb, nbb = W.make_paper_ensemble(spec)
    fr = W.make_frames_sparse(rows, cols, shifts, mb, nbb, q, W.sigma_for_gap(0.02, 0.3), 3, 4242)
    ref = oracle_lib.decode_sparse(rows, cols, shifts, mb, nbb, q, fr.llr, fr.syndrome, n_iter, 0)
    hard, iters, passed, post = _gpu_decode(B.QCLDPCCode.from_sparse(rows, cols, shifts, mb, nbb, q), fr.llr,
                                            fr.syndrome, n_iter, 0)
    err = np.abs(post - ref.posterior) / np.maximum(1.0, np.abs(ref.posterior))
    assert err.max() <= TOL, err.max()
    decided = np.abs(ref.posterior) > 1e-2
    np.testing.assert_array_equal(hard[decided], ref.hard[decided])
    np.testing.assert_array_equal(passed, ref.passed)
    assert (iters == n_iter).all()


@pytest.mark.gpu
def test_gpu_paper_ensemble_early_stop(oracle_lib):
    from paper_1702_07740_b200 import binding as B
    spec = W.paper_ensemble_spec(400, 50)
    rows, cols, shifts, mb, nb = W.make_paper_ensemble(spec)
    fr = W.make_frames_sparse(rows, cols, shifts, mb, nb, 50, W.sigma_for_gap(0.02, 3.0), 6, 999)
    ref = oracle_lib.decode_sparse(rows, cols, shifts, mb, nb, 50, fr.llr, fr.syndrome, 80, 1)
    hard, iters, passed, post = _gpu_decode(B.QCLDPCCode.from_sparse(rows, cols, shifts, mb, nb, 50), fr.llr,
                                            fr.syndrome, 80, 1)
    np.testing.assert_array_equal(passed, ref.passed)
    np.testing.assert_array_equal(iters, ref.iters)
    ok = ref.passed.astype(bool)
    assert ok.any()
    np.testing.assert_array_equal(hard[ok], ref.hard[ok])
    np.testing.assert_array_equal(W.syndrome_of_sparse(rows, cols, shifts, mb, nb, 50, hard[ok]), fr.syndrome[ok])


def _mixed_rows_code(rng, nc, kinds, q):
    """Test input only: nc core columns; `kinds` = [(core edges, has degree-1 column, count)] rows in that order, core
    sockets drawn without repetition inside a row.  Rows with a degree-1 column and 2 / 3 / more core edges are the
    pair / triple / gen rows of the generic kernel; rows without one report the parity (counter edges)."""
    rows, cols, r, n_abs = [], [], 0, 0
    for n_core, has_abs, count in kinds:
        for _ in range(count):
            for c in rng.choice(nc, size=n_core, replace=False):
                rows.append(r); cols.append(int(c))
            if has_abs:
                rows.append(r); cols.append(nc + n_abs); n_abs += 1
            r += 1
    rows, cols = np.asarray(rows, np.int32), np.asarray(cols, np.int32)
    return rows, cols, rng.integers(0, q, size=len(rows)).astype(np.int32), r, nc + n_abs


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["triples only", "all kinds", "triples across chunks", "long columns", "tiny q"])
@pytest.mark.parametrize("n_frames", [1, 5, 26])
def test_gpu_row_kinds_of_the_generic_kernel(oracle_lib, case, n_frames):
    """Every chunk body of the generic pass (pair, triple, gen, mixed), with the boundaries between the edge classes of
    a column falling at different places of the 4- and 8-edge chunks, one and two frames per thread, and (26 frames) six
    frames of q = 5 or three of q = 33 side by side in a tile."""
    from paper_1702_07740_b200 import binding as B
    rng = np.random.default_rng(sum(map(ord, case)))
    nc, q, sigma, kinds = {
        "triples only": (6, 33, 2.0, [(3, True, 40)]),
        "all kinds": (9, 70, 3.2, [(2, False, 3), (3, False, 2), (7, False, 2), (4, True, 5), (3, True, 30), (2, True, 25)]),
        "triples across chunks": (5, 50, 2.0, [(5, False, 1), (3, True, 21), (2, True, 9)]),
        "long columns": (4, 130, 4.5, [(3, False, 2), (4, False, 3), (3, True, 60), (2, True, 20), (1, True, 3)]),
        "tiny q": (7, 5, 3.2, [(2, False, 2), (3, True, 35), (2, True, 14)]),
    }[case]
    rows, cols, shifts, mb, nb = _mixed_rows_code(rng, nc, kinds, q)
    assert np.bincount(cols[cols < nc], minlength=nc).max() <= 64
    code = B.QCLDPCCode.from_sparse(rows, cols, shifts, mb, nb, q)
    # fixed iterations near the code's limit (messages of every size), early stop well inside it (no marginal frames)
    for n_iter, early, sg in ((7, 0, sigma), (40, 1, 0.6 * sigma)):
        fr = W.make_frames_sparse(rows, cols, shifts, mb, nb, q, sg, n_frames, 31337)
        ref = oracle_lib.decode_sparse(rows, cols, shifts, mb, nb, q, fr.llr, fr.syndrome, n_iter, early)
        hard, iters, passed, post = _gpu_decode(code, fr.llr, fr.syndrome, n_iter, early)
        np.testing.assert_array_equal(passed, ref.passed)
        np.testing.assert_array_equal(iters, ref.iters)
        assert early == 0 or (ref.passed.all() and ref.iters.max() < 40)
        err = np.abs(post - ref.posterior) / np.maximum(1.0, np.abs(ref.posterior))
        assert err.max() <= TOL, (case, n_iter, err.max())
        decided = np.abs(ref.posterior) > 1e-2
        np.testing.assert_array_equal(hard[decided], ref.hard[decided])


@pytest.mark.gpu
def test_gpu_generic_kernel_frame_independence():
    """Batched decodes carry two frames per thread in the generic kernel, single frames one: a frame's outputs must not
    depend on the batch (bit for bit), also when its pair partner stops early or is missing (odd batch)."""
    from paper_1702_07740_b200 import binding as B
    spec = W.paper_ensemble_spec(400, 21)
    rows, cols, shifts, mb, nb = W.make_paper_ensemble(spec)
    code = B.QCLDPCCode.from_sparse(rows, cols, shifts, mb, nb, 21)
    hi = W.make_frames_sparse(rows, cols, shifts, mb, nb, 21, W.sigma_for_gap(0.02, 3.0), 8, 555)
    lo = W.make_frames_sparse(rows, cols, shifts, mb, nb, 21, W.sigma_for_gap(0.02, 0.3), 5, 556)
    order = [0, 1, 8, 2, 3, 9, 10, 4, 5, 6, 11, 7, 12]                                # converging and not, mixed
    llr13, syn13 = np.concatenate([hi.llr, lo.llr])[order], np.concatenate([hi.syndrome, lo.syndrome])[order]
    # 7 frames: two frames per thread; 13 frames: also three frames side by side in a tile (q = 21 in 64 lanes), the
    # last CTA row with a single frame
    for n in (7, 13):
        llr, syn = llr13[:n], syn13[:n]
        for early in (0, 1):
            batch = _gpu_decode(code, llr, syn, 40, early)
            assert early == 0 or (0 < batch[2].sum() < n)                            # some stop early, some do not
            for f in range(n):
                alone = _gpu_decode(code, llr[f:f + 1], syn[f:f + 1], 40, early)
                for a_, b_ in zip(batch, alone):
                    np.testing.assert_array_equal(a_[f], b_[0])


def test_rate10_standin_structure():
    """NEXT-2 stand-in (the paper does not print that code's degree distribution): size and shape only."""
    rows, cols, shifts, mb, nb = W.make_rate10_standin()
    assert nb * 512 == 2 ** 20 and abs((1.0 - mb / nb) - 0.1) < 1e-3                  # n = 2^20, rate 1/10
    nc, n_top = (nb + 2) // 5, nb // 10
    cdeg, rdeg = np.bincount(cols, minlength=nb), np.bincount(rows, minlength=mb)
    assert set(cdeg[:nc]) <= {10, 11} and (cdeg[nc:] == 1).all()
    assert rdeg[:n_top].min() >= 2 and (rdeg[n_top:] == 3).all()
    key = rows.astype(np.int64) * nb + cols
    assert len(np.unique(key)) == len(key)
    d1 = cols >= nc
    assert (rows[d1] - n_top == cols[d1] - nc).all() and (shifts[d1] == 0).all()


@pytest.mark.gpu
def test_gpu_rate10_standin_reduced(oracle_lib):
    from paper_1702_07740_b200 import binding as B
    rows, cols, shifts, mb, nb = W.make_rate10_standin(200, 64)
    fr = W.make_frames_sparse(rows, cols, shifts, mb, nb, 64, 0.161 ** -0.5, 5, 2020)
    for early, n_iter in ((0, 20), (1, 100)):
        ref = oracle_lib.decode_sparse(rows, cols, shifts, mb, nb, 64, fr.llr, fr.syndrome, n_iter, early)
        hard, iters, passed, post = _gpu_decode(B.QCLDPCCode.from_sparse(rows, cols, shifts, mb, nb, 64), fr.llr,
                                                fr.syndrome, n_iter, early)
        np.testing.assert_array_equal(passed, ref.passed)
        np.testing.assert_array_equal(iters, ref.iters)
        if early == 0:
            err = np.abs(post - ref.posterior) / np.maximum(1.0, np.abs(ref.posterior))
            assert err.max() <= TOL, err.max()
            decided = np.abs(ref.posterior) > 1e-2
            np.testing.assert_array_equal(hard[decided], ref.hard[decided])


@pytest.mark.gpu
def test_gpu_paper_ensemble_full_size(oracle_lib):
    """The paper's q = 50 code at full size (n = 1e6, 66,750 base blocks, 3.34 M edges), one frame at the paper's
    operating point (beta = 0.99, SNR 0.0284): posterior and hard bits after 12 iterations against the oracle."""
    from paper_1702_07740_b200 import binding as B
    spec = W.paper_ensemble_spec(20000, 50)
    rows, cols, shifts, mb, nb = W.make_paper_ensemble(spec)
    sigma = (2.0 ** (2.0 * 0.02 / 0.99) - 1.0) ** -0.5
    fr = W.make_frames_sparse(rows, cols, shifts, mb, nb, 50, sigma, 1, 31415)
    ref = oracle_lib.decode_sparse(rows, cols, shifts, mb, nb, 50, fr.llr, fr.syndrome, 12, 0)
    hard, iters, passed, post = _gpu_decode(B.QCLDPCCode.from_sparse(rows, cols, shifts, mb, nb, 50), fr.llr,
                                            fr.syndrome, 12, 0)
    err = np.abs(post - ref.posterior) / np.maximum(1.0, np.abs(ref.posterior))
    assert err.max() <= TOL, err.max()
    decided = np.abs(ref.posterior) > 1e-2
    np.testing.assert_array_equal(hard[decided], ref.hard[decided])
    np.testing.assert_array_equal(passed, ref.passed)
