"""Pins for the oracle's AES-128 / CTR stream: the standard's
known answers (tests/golden/*.txt), the 64-bit carry, and an independent AES
(OpenSSL through python `cryptography`).  CPU only."""
import numpy as np
import pytest
from conftest import read_golden

import oracle as O

crypto = pytest.importorskip("cryptography.hazmat.primitives.ciphers")
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes  # noqa: E402


def openssl_ctr(key: bytes, iv: bytes, nbytes: int) -> bytes:
    return Cipher(algorithms.AES(key), modes.CTR(iv)).encryptor().update(bytes(nbytes))


def test_p1_fips197_known_answers():
    g = read_golden("aes128_fips197.txt")
    h = bytes.fromhex
    assert O.aes128_encrypt_block(h(g["c1_key"]), h(g["c1_plaintext"])) == h(g["c1_ciphertext"])
    assert O.aes128_encrypt_block(h(g["b_key"]), h(g["b_input"])) == h(g["b_output"])


def test_p2_sp800_38a_ctr_vector():
    g = read_golden("aes128_ctr_sp800_38a.txt")
    key, iv = bytes.fromhex(g["key"]), bytes.fromhex(g["initial_counter"])
    pt = b"".join(bytes.fromhex(x) for x in g["plaintext"])
    ct = b"".join(bytes.fromhex(x) for x in g["ciphertext"])
    ks = O.ctr_bytes(key, iv, 0, 64).tobytes()
    assert bytes(a ^ b for a, b in zip(ks, pt)) == ct


def test_p2_counter_carries_across_64_bits():
    g = read_golden("aes128_ctr_sp800_38a.txt")
    key, iv = bytes.fromhex(g["carry_key"]), bytes.fromhex(g["carry_iv"])
    ks = O.ctr_bytes(key, iv, 16, 16).tobytes()            # block 1 only
    assert ks == bytes.fromhex(g["carry_block1"])
    assert ks == O.aes128_encrypt_block(key, bytes.fromhex("00000000000000010000000000000000"))
    assert O.ctr_bytes(key, iv, 0, 48).tobytes() == openssl_ctr(key, iv, 48)
    # full 128-bit wrap: iv = 2^128 - 1, block 1 encrypts the all-zero counter
    ff = b"\xff" * 16
    assert O.ctr_bytes(key, ff, 16, 16).tobytes() == O.aes128_encrypt_block(key, bytes(16))


@pytest.mark.parametrize("seed", range(6))
def test_ctr_matches_openssl_random_keys(seed):
    rng = np.random.default_rng(seed)
    key, iv = rng.bytes(16), rng.bytes(16)
    n = int(rng.integers(1, 700))
    assert O.ctr_bytes(key, iv, 0, n).tobytes() == openssl_ctr(key, iv, n)


def test_p3_any_offset_is_a_slice_of_the_stream():
    rng = np.random.default_rng(7)
    key, iv = rng.bytes(16), rng.bytes(16)
    whole = O.ctr_bytes(key, iv, 0, 1000)
    for a, b in [(0, 1), (1, 15), (15, 2), (16, 16), (17, 300), (333, 667), (999, 1), (5, 0)]:
        assert np.array_equal(O.ctr_bytes(key, iv, a, b), whole[a:a + b])
    # far offsets (beyond 2^32 blocks) agree with OpenSSL started at the advanced counter
    off_blocks = (1 << 36) + 12345
    adv = (int.from_bytes(iv, "big") + off_blocks) % (1 << 128)
    assert (O.ctr_bytes(key, iv, 16 * off_blocks + 3, 61).tobytes()
            == openssl_ctr(key, adv.to_bytes(16, "big"), 64)[3:])


def test_o3_seed_key_and_object_iv_layout():
    assert O.seed_key(0x0807060504030201) == bytes([1, 2, 3, 4, 5, 6, 7, 8]) + bytes(8)
    assert O.seed_key(5) == bytes([5]) + bytes(15)
    # BE64(tag*2^56 + attempt*2^32 + inst) || 0^8
    assert O.object_iv(1, 0, 0) == bytes([1]) + bytes(15)
    assert O.object_iv(4, 0x010203, 0x0a0b0c0d) == bytes([4, 1, 2, 3, 0x0a, 0x0b, 0x0c, 0x0d]) + bytes(8)
    for tag, att, inst in [(2, 0, 31), (5, 7, 0xffffffff), (15, 0xffffff, 1)]:
        want = ((tag << 56) + (att << 32) + inst).to_bytes(8, "big") + bytes(8)
        assert O.object_iv(tag, att, inst) == want
