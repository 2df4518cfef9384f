"""ORACLE -- test infrastructure, NOT product code.  The steps either side of the decoder:

  llr_init    Step 1 of Algorithm 1: sigma^2_{N_v} <- sigma^2_Z / ||X_v||,  Q_v <- 2 R_v / sigma^2_{N_v}, with the
              per-symbol noise variance of the d = 1 scheme or of the d = 2 scheme (a_i, b_i).
  pack_bits   the decoded word as bits (Step 5, keeps the first k of them), most significant bit first.
  crc32 / frame_crc_ok   the 32-bit CRC of the message part of a frame (Fig. 7; N_CRC = 32).

Plain numpy in double precision, written to be checked against the paper by eye; nothing here is shared with the CUDA
path.  Only tests/ may import this module.  Readings:
  G5  P:97 and P:344 print sigma^2_N = sigma^2_Z / ||X_v|| (a norm), while Eq. 1, from which the sentence is
      derived, has the noise term Z_i / X_i, whose variance is sigma^2_Z / X_i^2, and the d = 2 formula of P:120 gives
      (a_i^2 + b_i^2) sigma^2_Z = 2 sigma^2_Z / ||X||^2 -- a squared norm as well.  norm_power = 2 (the variance that
      Eq. 1 implies; the default) or 1 (as printed).  Pin: only norm_power = 2 makes Q_v the log-likelihood ratio that
      Step 1 says it is (tests/test_frontend_pins.py).
  G7  the paper names no CRC polynomial: CRC-32 of IEEE 802.3 (polynomial 0x04C11DB7, bit-reflected, initial value and
      final XOR 0xFFFFFFFF), the code everyone calls "CRC-32"; check value 0xCBF43926 for the ASCII string "123456789".
  G8  bit order: bit v of a frame is bit 7 - (v mod 8) of byte v // 8 (most significant first); the CRC field holds the
      CRC value as a 32-bit big-endian number in the 32 bits that follow the message (Fig. 7: message, CRC, parity).
"""
from __future__ import annotations

import numpy as np

CRC32_POLY = 0x104C11DB7      # x^32 + x^26 + x^23 + x^22 + x^16 + x^12 + x^11 + x^10 + x^8 + x^7 + x^5 + x^4 + x^2 + x + 1


def llr_init(R, X, sigma2_z, dim: int = 1, norm_power: int = 2) -> np.ndarray:
    """Q [F][n] in double from R [F][n], X [F][n], sigma2_z [F] (P:344 Step 1).

    dim = 0   no side information: sigma^2_N = sigma^2_Z for every symbol (X is ignored; the BIAWGN recipe of
              BASELINE.json, LLR = 2 y / sigma^2)
    dim = 1   sigma^2_{N_v} = sigma^2_Z / ||X_v||^norm_power                       (reading G5)
    dim = 2   symbols in successive pairs (R_{2i-1}, R_{2i}), i = 1..n/2:
              a_i = (X_{2i-1} + X_{2i}) / (X_{2i-1}^2 + X_{2i}^2),  b_i = (X_{2i} - X_{2i-1}) / (X_{2i-1}^2 + X_{2i}^2),
              sigma^2_{N(2i-1)} = sigma^2_{N(2i)} = (a_i^2 + b_i^2) sigma^2_Z
    then Q_v = 2 R_v / sigma^2_{N_v}."""
    R = np.asarray(R, dtype=np.float64)
    s2 = np.asarray(sigma2_z, dtype=np.float64).reshape(-1, 1)
    with np.errstate(divide="ignore", invalid="ignore"):
        if dim == 0:
            s2n = np.broadcast_to(s2, R.shape)
        elif dim == 1:
            X = np.asarray(X, dtype=np.float64)
            norm = np.abs(X)
            s2n = s2 / (norm if norm_power == 1 else norm * norm)
        elif dim == 2:
            X = np.asarray(X, dtype=np.float64)
            if R.shape[1] % 2:
                raise ValueError("d = 2 needs an even number of symbols")
            x1, x2 = X[:, 0::2], X[:, 1::2]
            den = x1 * x1 + x2 * x2
            a = (x1 + x2) / den
            b = (x2 - x1) / den
            s2n = np.repeat((a * a + b * b) * s2, 2, axis=1)
        else:
            raise ValueError("dim must be 0, 1 or 2 (the d = 4 and d = 8 noise terms are not in the paper, P:120)")
        return 2.0 * R / s2n


def pack_bits(hard, n_bits: int) -> np.ndarray:
    """The first n_bits of every frame of hard [F][n] (0/1 bytes; only bit 0 counts) as ceil(n_bits / 8) bytes, most
    significant bit first (reading G8); the unused low bits of the last byte are zero.  Written out bit by bit."""
    hard = np.asarray(hard, dtype=np.uint8)
    F = hard.shape[0]
    out = np.zeros((F, (n_bits + 7) // 8), dtype=np.uint8)
    for v in range(n_bits):
        out[:, v // 8] |= (hard[:, v] & 1) << (7 - v % 8)
    return out


def crc32(data: bytes) -> int:
    """CRC-32 (reading G7) from its definition as a polynomial remainder over GF(2): the message bits, least
    significant bit of every byte first, with the first 32 of them complemented (the initial value), followed by 32
    zero bits, are divided by the generator polynomial; the complemented remainder, bit-reflected, is the CRC."""
    bits = np.unpackbits(np.frombuffer(bytes(data), dtype=np.uint8), bitorder="little").astype(np.uint8)
    work = np.concatenate([bits, np.zeros(32, dtype=np.uint8)])
    work[:32] ^= 1                                                           # initial value 0xFFFFFFFF
    gen = np.array([(CRC32_POLY >> (32 - j)) & 1 for j in range(33)], dtype=np.uint8)   # x^32 first
    for i in range(len(bits)):                                               # long division, one quotient bit at a time
        if work[i]:
            work[i:i + 33] ^= gen
    rem = work[len(bits):] ^ 1                                               # final XOR 0xFFFFFFFF
    return int(sum(int(b) << j for j, b in enumerate(rem)))                  # first remainder bit is bit 0 (reflected)


def frame_crc(packed, k_bits: int):
    """(crc [F] uint32 of the message part, ok [F] uint8) of packed frames [F][>= k_bits / 8] (Fig. 7): the k
    information bits are k - 32 message bits followed by the 32 CRC bits; ok = the computed CRC equals the stored one."""
    if k_bits % 8 or k_bits < 32:
        raise ValueError("k_bits must be a multiple of 8 and at least 32")
    packed = np.asarray(packed, dtype=np.uint8)
    nmsg = (k_bits - 32) // 8
    crc = np.array([crc32(row[:nmsg].tobytes()) for row in packed], dtype=np.uint32)
    stored = np.array([int.from_bytes(row[nmsg:nmsg + 4].tobytes(), "big") for row in packed], dtype=np.uint32)
    return crc, (crc == stored).astype(np.uint8)
