"""Pins for the oracle's samplers (pins P4-P5).  CPU only.

The stream bytes every sampler consumes are re-derived here through OpenSSL
(python `cryptography`), not through the oracle's AES, so a wrong offset, byte
order or tag shows up; the distributions are checked against closed forms."""
from math import comb

import numpy as np
import pytest

import oracle as O

pytest.importorskip("cryptography.hazmat.primitives.ciphers")
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes  # noqa: E402


def stream(seed: int, tag: int, attempt: int, inst: int, nbytes: int) -> np.ndarray:
    key = seed.to_bytes(8, "little") + bytes(8)
    iv = ((tag << 56) + (attempt << 32) + inst).to_bytes(8, "big") + bytes(8)
    ks = Cipher(algorithms.AES(key), modes.CTR(iv)).encryptor().update(bytes(nbytes))
    return np.frombuffer(ks, dtype=np.uint8)


def words(seed, tag, attempt, inst, count):
    return stream(seed, tag, attempt, inst, 2 * count).view("<u2").astype(np.uint32)


# ---------------------------------------------------------------- O4 uniform

def test_p4_power_of_two_modulus_is_the_raw_le16_stream():
    for seed, tag, inst in [(1, O.TAG_A, 0), (2, O.TAG_S, 3), (4, O.TAG_S, 31)]:
        got = O.sample_uniform(0, 4096, seed, tag, inst, 65536)
        assert np.array_equal(got, words(seed, tag, 0, inst, 4096))
    # q = 2^12: T = 65536, value = c mod 4096
    got = O.sample_uniform(0, 1000, 9, O.TAG_A, 0, 4096)
    assert np.array_equal(got, words(9, O.TAG_A, 0, 0, 1000) % 4096)


def test_p4_any_subrange_equals_slice():
    full = O.sample_uniform(0, 5000, 3, O.TAG_A, 0, 65521)
    for first, count in [(0, 1), (1, 7), (7, 2), (8, 8), (13, 2000), (4999, 1)]:
        assert np.array_equal(O.sample_uniform(first, count, 3, O.TAG_A, 0, 65521), full[first:first + count])


@pytest.mark.parametrize("q", [65536, 65521, 40000, 17])
def test_p4_strided_draw_is_the_openssl_stream_at_those_positions(q):
    # a column of a row-major matrix: elements first + r*stride, re-derived through OpenSSL with an
    # independent walk over the attempt streams (not through orc_sample_uniform)
    first, stride, count = 5, 37, 700
    pos = first + stride * np.arange(count)
    N = int(pos[-1]) + 1
    T = q * (65536 // q)
    want = np.zeros(count, np.uint32)
    pending = np.arange(count)
    a = 0
    while pending.size:
        c = words(7, O.TAG_A, a, 0, N)[pos[pending]]
        ok = c < T
        want[pending[ok]] = c[ok] % q
        pending = pending[~ok]
        a += 1
    got = O.sample_uniform_strided(first, stride, count, 7, O.TAG_A, 0, q)
    assert np.array_equal(got, want)
    assert np.array_equal(got, O.sample_uniform(0, N, 7, O.TAG_A, 0, q)[pos])


@pytest.mark.parametrize("q", [3, 17, 251, 40000, 65521])
def test_p4_rejection_follows_attempt_streams(q):
    N = 1 << 15
    got = O.sample_uniform(0, N, 3, O.TAG_A, 5, q).astype(np.uint32)
    assert got.max() < q
    T = q * (65536 // q)
    # independent walk over attempt streams a = 0,1,2,... at the SAME element position
    want = np.zeros(N, np.uint32)
    pending = np.arange(N)
    a = 0
    while pending.size:
        c = words(3, O.TAG_A, a, 5, N)[pending]
        ok = c < T
        want[pending[ok]] = c[ok] % q
        pending = pending[~ok]
        a += 1
        assert a < 64
    assert np.array_equal(got, want)
    if q == 40000:
        assert a > 3       # rejection really happened repeatedly (P(reject) = 0.39)


def test_p4_prime_modulus_rejection_count_and_uniformity():
    q, N = 65521, 1 << 22
    got = O.sample_uniform(0, N, 3, O.TAG_A, 0, q).astype(np.int64)
    c0 = words(3, O.TAG_A, 0, 0, N)
    rejected = int((c0 >= q).sum())
    expect = N * 15 / 65536                                  # 960 at N = 2^22
    assert abs(rejected - expect) < 5 * np.sqrt(expect)
    assert np.array_equal(got[c0 < q], c0[c0 < q])
    # chi-square over 256 equal-width buckets of [0, q)
    counts = np.bincount((got * 256) // q, minlength=256).astype(np.float64)
    exp = np.array([(((b + 1) * q + 255) // 256) - ((b * q + 255) // 256) for b in range(256)]) * (N / q)
    chi2 = float(((counts - exp) ** 2 / exp).sum())
    assert chi2 < 255 + 6 * np.sqrt(2 * 255)


# ---------------------------------------------------------------- O5 CBD

@pytest.mark.parametrize("eta", [1, 2, 3, 4, 8])
def test_p5_cbd_exhaustive_pmf_over_all_words(eta):
    q = 65536
    hist = {}
    for w in range(65536):
        x = O.cbd_from_word(w, q, eta)
        x = x - q if x > q // 2 else x
        hist[x] = hist.get(x, 0) + 1
    assert min(hist) == -eta and max(hist) == eta
    for x in range(-eta, eta + 1):
        # pmf C(2eta, eta+x)/2^(2eta), times 65536 words
        assert hist[x] == comb(2 * eta, eta + x) * 65536 // (1 << (2 * eta)), (eta, x)
    mean = sum(x * c for x, c in hist.items()) / 65536
    var = sum(x * x * c for x, c in hist.items()) / 65536
    assert mean == 0 and var == eta / 2


@pytest.mark.parametrize("q,eta", [(65536, 4), (65521, 8), (17, 3)])
def test_p5_cbd_stream_positions_and_mod_q(q, eta):
    N = 3000
    got = O.sample_cbd(0, N, 4, O.TAG_E, 2, q, eta).astype(np.int64)
    w = words(4, O.TAG_E, 0, 2, N)
    M = (1 << eta) - 1
    lo = np.array([bin(int(x) & M).count("1") for x in w])
    hi = np.array([bin((int(x) >> 8) & M).count("1") for x in w])
    assert np.array_equal(got, (lo - hi) % q)
    assert np.array_equal(O.sample_cbd(100, 50, 4, O.TAG_E, 2, q, eta), got[100:150])
    # sign convention: low byte counts positive
    assert O.cbd_from_word(0x0001, q, eta) == 1 and O.cbd_from_word(0x0100, q, eta) == q - 1


def test_p5_cbd_empirical_variance():
    got = O.sample_cbd(0, 1 << 18, 2, O.TAG_E, 0, 65536, 4).astype(np.int64)
    x = np.where(got > 32768, got - 65536, got)
    assert abs(x.mean()) < 0.02 and abs(x.var() - 2.0) < 0.03


# ---------------------------------------------------------------- O6 bits

def test_o6_bits_are_lsb_first_stream_bits():
    ks = stream(2, O.TAG_R, 0, 7, 512)
    assert np.array_equal(O.sample_bits(0, 4096, 2, O.TAG_R, 7), ks)
    allbits = np.unpackbits(ks, bitorder="little")
    for first, nbits in [(0, 1), (3, 5), (5, 8), (13, 257), (4000, 96), (8, 0)]:
        got = O.sample_bits(first, nbits, 2, O.TAG_R, 7)
        assert got.size == (nbits + 7) // 8
        assert np.array_equal(np.unpackbits(got, bitorder="little")[:nbits], allbits[first:first + nbits])
        if nbits % 8:
            assert got[-1] >> (nbits % 8) == 0          # padding bits are zero


def test_streams_of_different_objects_differ():
    a = O.sample_uniform(0, 64, 1, O.TAG_A, 0, 65536)
    assert not np.array_equal(a, O.sample_uniform(0, 64, 1, O.TAG_S, 0, 65536))
    assert not np.array_equal(a, O.sample_uniform(0, 64, 2, O.TAG_A, 0, 65536))
    assert not np.array_equal(O.sample_uniform(0, 64, 1, O.TAG_S, 0, 65536),
                              O.sample_uniform(0, 64, 1, O.TAG_S, 1, 65536))
