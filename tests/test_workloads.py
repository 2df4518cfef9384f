"""The seeded generators produce the structure BASELINE.json states (CPU only)."""
import numpy as np
import pytest

from paper_1702_07740_b200 import workloads as W
from tests.helpers import dense_h


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_base_matrix_structure(idx):
    cfg = W.CONFIGS[idx]
    sp = cfg.code
    base = W.make_base_matrix(sp)
    assert base.shape == (sp.mb, sp.nb) and base.dtype == np.int32
    assert base.min() >= -1 and base.max() < sp.Z
    nz = base >= 0
    core = nz[:, :sp.n_core]
    assert (core[:sp.top_rows].sum(axis=0) == sp.top_deg).all()
    assert (core[sp.top_rows:].sum(axis=0) == sp.low_deg).all()
    assert (core[sp.top_rows:].sum(axis=1) == 2).all()          # every lower row: exactly 2 core edges
    assert (core[:sp.top_rows].sum(axis=1) >= 2).all()          # S11
    d1 = nz[:, sp.n_core:]
    assert (d1.sum(axis=0) == 1).all() and not d1[:sp.top_rows].any()
    for j in range(sp.n_core, sp.nb):
        assert base[j - sp.n_core + sp.top_rows, j] == 0        # unshifted diagonal
    assert sp.n == sp.nb * sp.Z and abs((1 - sp.mb / sp.nb) - sp.rate) < 1e-12
    np.testing.assert_array_equal(base, W.make_base_matrix(sp))  # deterministic
    assert int(nz[:, :sp.n_core].sum()) == sp.n_core * (sp.top_deg + sp.low_deg)


def test_sizes_match_survey_table():
    # SURVEY.md §8 size table: n, m, E_core, E_d1
    want = {1: (2560, 2304, 5632, 2048), 2: (1000000, 900000, 2200000, 800000),
            3: (1000000, 980000, 2100000, 900000), 5: (1000000, 950000, 2100000, 900000)}
    for idx, (n, m, ec, ed) in want.items():
        sp = W.CONFIGS[idx].code
        assert (sp.n, sp.m) == (n, m)
        assert sp.n_core * (sp.top_deg + sp.low_deg) * sp.Z == ec
        assert (sp.nb - sp.n_core) * sp.Z == ed
    assert W.CONFIGS[4].code == W.CONFIGS[3].code and W.CONFIGS[4].n_frames == 64


def test_scaled_spec_keeps_graph():
    sp = W.CONFIGS[3].code
    a = W.make_base_matrix(sp) >= 0
    b = W.make_base_matrix(W.scaled_spec(sp, 64)) >= 0
    np.testing.assert_array_equal(a, b)


def test_frames_are_seeded_and_consistent():
    cfg, base, Z, fr = W.make_config(1)
    assert fr.llr.dtype == np.float32 and fr.llr.shape == (16, 2560) and fr.syndrome.shape == (16, 2304)
    H = dense_h(base, Z).astype(np.int64)
    np.testing.assert_array_equal((fr.x.astype(np.int64) @ H.T) % 2, fr.syndrome)
    _, _, _, fr2 = W.make_config(1, n_frames=3, first_frame=5)
    np.testing.assert_array_equal(fr2.llr, fr.llr[5:8])
    np.testing.assert_array_equal(fr2.syndrome, fr.syndrome[5:8])
    # LLR ~ N(+-2/sigma^2, 4/sigma^2) with the sign of the transmitted bit
    mu = 2 / fr.sigma ** 2
    z = fr.llr * (1 - 2.0 * fr.x)
    assert abs(z.mean() - mu) < 5 * (2 / fr.sigma) / np.sqrt(z.size)
    assert abs(z.std() - 2 / fr.sigma) < 0.02
