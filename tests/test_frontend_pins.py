"""Pins of the NEXT-4 oracle (oracle/frontend.py) against things other than itself (CPU only, -m "not gpu").

LLR front end (P:344 Step 1): hand-computed symbols; the d = 2 variance against its closed form
2 sigma^2_Z / ||X||^2; the BIAWGN recipe of the workloads; and the property that DEFINES Q_v in Step 1 -- Q_v is the
log-likelihood ratio ln P(C_v = 0 | R_v) / P(C_v = 1 | R_v) of the channel of Eq. 1 -- checked by simulation, which is
what settles reading G5 (norm vs squared norm).
Bit packing: numpy.packbits.  CRC-32 (reading G7): the standard check value, zlib on random strings, linearity."""
import zlib

import numpy as np
import pytest

from oracle import frontend as FE


def test_llr_hand_computed_symbols():
    # d = 1: R = 1.5, X = 2, sigma_Z^2 = 4.  Squared norm (Eq. 1): sigma_N^2 = 4 / 4 = 1, Q = 3.  As printed: 4 / 2, Q = 1.5
    assert FE.llr_init([[1.5]], [[2.0]], [4.0], 1, 2)[0, 0] == 3.0
    assert FE.llr_init([[1.5]], [[-2.0]], [4.0], 1, 2)[0, 0] == 3.0          # a norm: the sign of X does not matter
    assert FE.llr_init([[1.5]], [[2.0]], [4.0], 1, 1)[0, 0] == 1.5
    assert FE.llr_init([[-0.25]], [[0.5]], [2.0], 1, 2)[0, 0] == -0.0625      # 2 * -0.25 * 0.25 / 2
    # d = 0 ignores X; one sigma per frame
    q = FE.llr_init([[1.0, -2.0], [1.0, -2.0]], None, [0.5, 4.0], 0)
    np.testing.assert_array_equal(q, [[4.0, -8.0], [0.5, -1.0]])
    # d = 2: X = (3, 4): a = 7/25, b = 1/25, a^2 + b^2 = 50/625 = 0.08; sigma_Z^2 = 0.5: sigma_N^2 = 0.04
    q = FE.llr_init([[1.0, -2.0]], [[3.0, 4.0]], [0.5], 2)
    np.testing.assert_allclose(q, [[50.0, -100.0]], rtol=1e-15)
    # X = (1, 1): a = 1, b = 0: the pair sees sigma_Z^2 itself
    np.testing.assert_array_equal(FE.llr_init([[0.5, 0.25]], [[1.0, 1.0]], [2.0], 2), [[0.5, 0.25]])
    # X = 0: infinite noise variance, the symbol carries nothing
    assert FE.llr_init([[1.5]], [[0.0]], [4.0], 1, 2)[0, 0] == 0.0
    with pytest.raises(ValueError):
        FE.llr_init([[1.0, 2.0, 3.0]], [[1.0, 2.0, 3.0]], [1.0], 2)
    with pytest.raises(ValueError):
        FE.llr_init([[1.0]], [[1.0]], [1.0], 4)


def test_llr_d2_closed_form_and_uniform_variance():
    """the variance is uniform over the pair and (a^2 + b^2) sigma_Z^2 = 2 sigma_Z^2 / (X_1^2 + X_2^2)."""
    rng = np.random.default_rng(1)
    X = rng.standard_normal((3, 64))
    R = rng.standard_normal((3, 64))
    s2 = np.array([0.3, 1.0, 7.5])
    q = FE.llr_init(R, X, s2, 2)
    nrm2 = np.repeat(X[:, 0::2] ** 2 + X[:, 1::2] ** 2, 2, axis=1)
    np.testing.assert_allclose(q, 2.0 * R * nrm2 / (2.0 * s2[:, None]), rtol=1e-13)


def test_llr_dim0_is_the_workload_recipe():
    from paper_1702_07740_b200 import workloads as W
    cfg, base, Z, fr = W.make_config(1, n_frames=2)
    rng = np.random.default_rng(W.frame_seed_base(1))                       # frame 0 again, by the documented recipe
    x = rng.integers(0, 2, size=base.shape[1] * Z, dtype=np.uint8)
    y = (1.0 - 2.0 * x.astype(np.float64)) + fr.sigma * rng.standard_normal(x.size)
    q = FE.llr_init(y[None], None, [fr.sigma ** 2], 0)
    np.testing.assert_array_equal(q[0].astype(np.float32), fr.llr[0])


def _calibration_z(Q, C, edges):
    """Largest |z| over bins of Q of (observed fraction of C = 1) - (mean of 1 / (1 + e^Q)): zero mean if Q is the LLR."""
    worst = 0.0
    for lo, hi in zip(edges[:-1], edges[1:]):
        sel = (Q >= lo) & (Q < hi)
        k = int(sel.sum())
        if k < 2000:
            continue
        p = 1.0 / (1.0 + np.exp(Q[sel]))
        z = (C[sel].mean() - p.mean()) / np.sqrt((p * (1 - p)).mean() / k)
        worst = max(worst, abs(float(z)))
    return worst


def test_reading_g5_squared_norm_makes_q_the_llr():
    """Step 1 defines Q_v = ln P(C_v = 0 | R_v) / P(C_v = 1 | R_v).  On the channel of Eq. 1 (Y = X + Z,
    M = (-1)^C Y, R = M / X with X known to Alice) a true LLR is calibrated: among symbols with Q_v near q the fraction
    with C_v = 1 is 1 / (1 + e^q).  sigma^2_N = sigma^2_Z / ||X||^2 passes; the printed sigma^2_Z / ||X|| does not."""
    rng = np.random.default_rng(2)
    n, s2 = 600000, 1.5
    C = rng.integers(0, 2, n)
    X = rng.standard_normal(n)
    Y = X + np.sqrt(s2) * rng.standard_normal(n)
    R = ((-1.0) ** C) * Y / X
    edges = np.arange(-3.0, 3.01, 0.5)
    z2 = _calibration_z(FE.llr_init(R[None], X[None], [s2], 1, 2)[0], C, edges)
    z1 = _calibration_z(FE.llr_init(R[None], X[None], [s2], 1, 1)[0], C, edges)
    assert z2 < 4.5, z2
    assert z1 > 10.0, z1
    # d = 2, complex form of Eq. 2: R = M X^-1 with U = (+-1, +-1); the printed a_i, b_i are calibrated
    n2 = n // 2
    C2 = rng.integers(0, 2, (n2, 2))
    Xc = rng.standard_normal(n2) + 1j * rng.standard_normal(n2)
    Zc = np.sqrt(s2) * (rng.standard_normal(n2) + 1j * rng.standard_normal(n2))
    U = (-1.0) ** C2[:, 0] + 1j * (-1.0) ** C2[:, 1]
    Rc = U * (Xc + Zc) / Xc
    Rp = np.stack([Rc.real, Rc.imag], axis=1).reshape(1, -1)
    Xp = np.stack([Xc.real, Xc.imag], axis=1).reshape(1, -1)
    zq = _calibration_z(FE.llr_init(Rp, Xp, [s2], 2)[0], C2.reshape(-1), edges)
    assert zq < 4.5, zq


def test_pack_bits_against_numpy():
    rng = np.random.default_rng(3)
    hard = rng.integers(0, 2, size=(4, 203), dtype=np.uint8)
    for n_bits in (0, 1, 7, 8, 9, 64, 200, 203):
        np.testing.assert_array_equal(FE.pack_bits(hard, n_bits), np.packbits(hard[:, :n_bits], axis=1))
    # only bit 0 of an input byte counts
    np.testing.assert_array_equal(FE.pack_bits(hard | 0xFE, 203), np.packbits(hard, axis=1))
    assert FE.pack_bits(np.array([[1, 0, 0, 0, 0, 0, 0, 0, 1]], np.uint8), 9).tolist() == [[0x80, 0x80]]


def test_crc32_check_value_and_zlib():
    assert FE.crc32(b"123456789") == 0xCBF43926                             # the catalogue check value of CRC-32
    assert FE.crc32(b"") == 0
    rng = np.random.default_rng(4)
    for L in (1, 2, 3, 4, 5, 8, 31, 32, 33, 255, 256, 1000, 2496):
        d = rng.integers(0, 256, L, dtype=np.uint8).tobytes()
        assert FE.crc32(d) == zlib.crc32(d), L
    # affine over GF(2): crc(a ^ b ^ c) = crc(a) ^ crc(b) ^ crc(c) for equal lengths
    a, b, c = (rng.integers(0, 256, 77, dtype=np.uint8) for _ in range(3))
    assert FE.crc32((a ^ b ^ c).tobytes()) == FE.crc32(a.tobytes()) ^ FE.crc32(b.tobytes()) ^ FE.crc32(c.tobytes())


def test_frame_crc_layout():
    """Fig. 7: k information bits = (k - 32) message bits + 32 CRC bits, then parity.  Reading G8."""
    rng = np.random.default_rng(5)
    k_bits = 20000                                                          # rate 0.02, n = 1e6
    msg = rng.integers(0, 256, (3, (k_bits - 32) // 8), dtype=np.uint8)
    frames = np.zeros((3, k_bits // 8 + 5), dtype=np.uint8)
    frames[:, :msg.shape[1]] = msg
    for f in range(3):
        frames[f, msg.shape[1]:msg.shape[1] + 4] = np.frombuffer(zlib.crc32(msg[f].tobytes()).to_bytes(4, "big"), np.uint8)
    frames[2, 17] ^= 0x10                                                   # one flipped message bit
    crc, ok = FE.frame_crc(frames, k_bits)
    assert ok.tolist() == [1, 1, 0]
    assert crc[0] == zlib.crc32(msg[0].tobytes()) and crc[2] != zlib.crc32(msg[2].tobytes())
    with pytest.raises(ValueError):
        FE.frame_crc(frames, 20001)
