"""GPU parity of the NEXT-4 steps (LLR front end, bit packing, CRC-32) against oracle/frontend.py, through the C ABI.

Tolerances.  qcldpc_llr_init works in IEEE single precision in the printed order, the oracle in double on the same fp32
inputs: d = 0 is one rounding (2 R / sigma^2), d = 1 three (||X||^2, sigma_Z^2 / ., 2 R / .), d = 2 about twelve (a, b from
sums and quotients, a^2 + b^2, the products): relative error <= 2^-24 per rounding, so 4 / 4 / 16 units of 2^-24 are
asserted (2.4e-7, 2.4e-7, 9.5e-7), with an absolute floor for results that underflow.  Packing and CRC are bit-exact."""
import zlib

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import frontend as FE  # noqa: E402
from paper_1702_07740_b200 import workloads as W  # noqa: E402

ULP = 2.0 ** -24


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_1702_07740_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("dim,power,units", [(0, 2, 4), (1, 2, 4), (1, 1, 4), (2, 2, 16)])
@pytest.mark.parametrize("n", [2, 6, 1000, 4098, 100003 * 2])
def test_llr_init_matches_oracle(B, dim, power, units, n):
    """Several tiles and a ragged tail (n not a multiple of 4 takes the scalar path), 3 frames with their own sigma."""
    rng = np.random.default_rng(n + 10 * dim + power)
    F = 3
    X = rng.standard_normal((F, n)).astype(np.float32)
    C = rng.integers(0, 2, (F, n))
    s2 = np.array([0.3, 35.2, 1.0], dtype=np.float32)
    Y = X + np.sqrt(s2)[:, None] * rng.standard_normal((F, n)).astype(np.float32)
    R = (((-1.0) ** C) * Y / X).astype(np.float32)
    want = FE.llr_init(R, X, s2, dim, power)
    got = B.llr_init(dev(R), dev(X) if dim else None, dev(s2), dim, power).cpu().numpy().astype(np.float64)
    fin = np.isfinite(want)                                  # R = M / X overflows where X is tiny: both sides give inf
    np.testing.assert_array_equal(got[~fin], want[~fin])
    err = np.abs(got[fin] - want[fin]) / np.maximum(np.abs(want[fin]), 1e-30)
    assert err.max() <= units * ULP, err.max()


def test_llr_init_special_values_and_errors(B):
    R = np.array([[1.5, -2.0, 0.0, 3.0]], np.float32)
    X = np.array([[0.0, -0.0, 2.0, np.inf]], np.float32)
    s2 = np.array([4.0], np.float32)
    for dim, p in ((1, 2), (1, 1)):
        want = FE.llr_init(R, X, s2, dim, p)
        got = B.llr_init(dev(R), dev(X), dev(s2), dim, p).cpu().numpy()
        np.testing.assert_array_equal(got[:, :3], want[:, :3].astype(np.float32))
        np.testing.assert_array_equal(np.signbit(got[:, :3]), np.signbit(want[:, :3]))   # X = 0: Q = +-0 with R's sign
        assert np.isinf(got[0, 3]) and np.isinf(want[0, 3])
    with pytest.raises(B.QCLDPCError):
        B.llr_init(dev(R[:, :3]), dev(X[:, :3]), dev(s2), 2)                              # d = 2 needs an even n
    with pytest.raises(B.QCLDPCError):
        B.llr_init(dev(R), dev(X), dev(s2), 4)                                             # d = 4: not in the paper
    with pytest.raises(B.QCLDPCError):
        B.llr_init(dev(R), None, dev(s2), 1)


def test_llr_init_feeds_the_decoder_like_the_workload_recipe(B):
    """dim = 0 on y = (1 - 2x) + noise reproduces the LLRs of the workload generator to the last bit but one: the
    generator rounds 2 y / sigma^2 once from double, the kernel rounds y and sigma^2 to fp32 first."""
    cfg, base, Z, fr = W.make_config(1, n_frames=2)
    y = (fr.llr.astype(np.float64) * fr.sigma ** 2 / 2.0).astype(np.float32)
    s2 = np.full(2, fr.sigma ** 2, dtype=np.float32)
    got = B.llr_init(dev(y), None, dev(s2), 0).cpu().numpy()
    np.testing.assert_allclose(got, fr.llr, rtol=4 * ULP, atol=0)


@pytest.mark.parametrize("n,n_bits", [(8, 8), (64, 64), (1000, 1000), (1000, 333), (1003, 1003), (1003, 17), (4096, 0),
                                      (2560, 256), (1000000, 20000), (1000000, 1000000)])
def test_pack_bits_bit_exact(B, n, n_bits):
    rng = np.random.default_rng(n + n_bits)
    F = 3 if n < 1000000 else 2
    hard = rng.integers(0, 2, (F, n), dtype=np.uint8)
    if n_bits == 0:
        with_zero = B.pack_bits(dev(hard), 0)
        assert tuple(with_zero.shape) == (F, 0)
        return
    want = FE.pack_bits(hard, n_bits) if n_bits <= 20000 else np.packbits(hard[:, :n_bits], axis=1)
    np.testing.assert_array_equal(B.pack_bits(dev(hard), n_bits).cpu().numpy(), want)
    np.testing.assert_array_equal(B.pack_bits(dev(hard | 0xFE), n_bits).cpu().numpy(), want)   # only bit 0 counts


def test_pack_bits_unaligned_base_pointer(B):
    """A view whose rows are not 8-byte aligned takes the byte path."""
    rng = np.random.default_rng(9)
    raw = rng.integers(0, 2, 3 + 2 * 1000, dtype=np.uint8)
    d = dev(raw)[3:].view(2, 1000)
    np.testing.assert_array_equal(B.pack_bits(d, 1000).cpu().numpy(), FE.pack_bits(raw[3:].reshape(2, 1000), 1000))


@pytest.mark.parametrize("k_bits", [32, 40, 64, 2080, 20000, 100000, 800008])
def test_crc32_check_bit_exact(B, k_bits):
    """Message lengths of 0, 1, 4 bytes, one byte per thread and a ragged last chunk, the paper's k = 20,000,
    and long messages; frames with a good CRC, a flipped message bit and a flipped CRC bit."""
    rng = np.random.default_rng(k_bits)
    F = 5
    nmsg = (k_bits - 32) // 8
    frames = rng.integers(0, 256, (F, k_bits // 8 + 3), dtype=np.uint8)
    for f in range(F):
        frames[f, nmsg:nmsg + 4] = np.frombuffer(zlib.crc32(frames[f, :nmsg].tobytes()).to_bytes(4, "big"), np.uint8)
    if nmsg:
        frames[1, nmsg // 2] ^= 0x04
    frames[3, nmsg + 2] ^= 0x80
    crc, ok = B.crc32_check(dev(frames), k_bits)
    want_crc, want_ok = FE.frame_crc(frames, k_bits) if k_bits <= 20000 else (
        np.array([zlib.crc32(r[:nmsg].tobytes()) for r in frames], dtype=np.uint32),
        np.array([1, 0 if nmsg else 1, 1, 0, 1], dtype=np.uint8))
    np.testing.assert_array_equal(crc.cpu().numpy().astype(np.uint32), want_crc)
    np.testing.assert_array_equal(ok.cpu().numpy(), want_ok)
    assert want_ok.tolist() == [1, 0 if nmsg else 1, 1, 0, 1]


def test_crc32_check_value(B):
    frame = np.frombuffer(b"123456789" + (0xCBF43926).to_bytes(4, "big"), np.uint8)[None]
    crc, ok = B.crc32_check(dev(frame.copy()), 8 * 13)
    assert int(crc[0]) == 0xCBF43926 and int(ok[0]) == 1
    with pytest.raises(B.QCLDPCError):
        B.crc32_check(dev(frame.copy()), 8 * 13 + 1)
    with pytest.raises(B.QCLDPCError):
        B.crc32_check(dev(frame.copy()), 8 * 14)                                          # longer than a row


def test_frontend_decode_pack_crc_chain(B):
    """The whole adjacent path on device: R, X -> LLR (d = 1) -> decode -> packed bits -> CRC verdict.  The word's first
    k bits are message + CRC (Fig. 7); in syndrome form any word is legal, s = H x; high SNR, so the decoder returns x."""
    cfg, base, Z, fr0 = W.make_config(1, n_frames=1)
    n = base.shape[1] * Z
    k_bits = 256                                                            # rate 0.1 of n = 2560
    rng = np.random.default_rng(11)
    F = 4
    x = rng.integers(0, 2, (F, n), dtype=np.uint8)
    for f in range(F):
        msg = np.packbits(x[f, :k_bits - 32])
        x[f, k_bits - 32:k_bits] = np.unpackbits(np.frombuffer(zlib.crc32(msg.tobytes()).to_bytes(4, "big"), np.uint8))
    syn = W.syndrome_of(base, Z, x)
    s2 = np.full(F, 0.05, np.float32)
    X = rng.standard_normal((F, n)).astype(np.float32)
    X = np.where(np.abs(X) < 0.3, np.float32(0.3) * np.sign(X) + (X == 0), X).astype(np.float32)   # keep |X| away from 0
    Y = X + np.sqrt(0.05) * rng.standard_normal((F, n)).astype(np.float32)
    R = (((-1.0) ** x) * Y / X).astype(np.float32)
    code = B.QCLDPCCode(base, Z)
    llr = B.llr_init(dev(R), dev(X), dev(s2), 1, 2)
    out = code.decode(llr, dev(syn), 50, 1, want_posterior=False)
    packed = B.pack_bits(out.hard, k_bits)
    crc, ok = B.crc32_check(packed, k_bits)
    torch.cuda.synchronize()
    assert out.passed.cpu().numpy().all()
    np.testing.assert_array_equal(out.hard.cpu().numpy(), x)
    assert ok.cpu().numpy().all()
    want_crc, want_ok = FE.frame_crc(FE.pack_bits(x, k_bits), k_bits)
    np.testing.assert_array_equal(crc.cpu().numpy().astype(np.uint32), want_crc)
    # a frame whose CRC field does not belong to its message is caught
    x2 = x.copy(); x2[0, 5] ^= 1
    _, ok2 = B.crc32_check(B.pack_bits(dev(x2), k_bits), k_bits)
    assert ok2.cpu().numpy().tolist() == [0, 1, 1, 1]
