"""Pins for the oracle's keygen / encaps / decaps (pins P6-P8, P10).
CPU only.  Expected values come from the hand-worked golden example, python big
integers, numpy int64 matrix products (a library routine on a special case),
algebraic identities and exhaustive enumeration -- never from the CUDA path."""
import numpy as np
import pytest
from conftest import read_golden

import oracle as O
from paper_2606_01211_b200 import workloads as W


def pack_bits(bits) -> np.ndarray:
    return np.packbits(np.asarray(bits, dtype=np.uint8).ravel(), bitorder="little")


def unpack_bits(packed, n) -> np.ndarray:
    return np.unpackbits(np.asarray(packed, dtype=np.uint8), bitorder="little")[:n]


def rows(text):
    return np.array([[int(x) for x in r.split()] for r in text.split(";")])


# ---------------------------------------------------------------- golden hand example

def test_hand_worked_example_eq1_and_regev_formulas():
    g = read_golden("lwe_hand_example.txt")
    q, n, m, k = (int(g[x]) for x in "qnmk")
    A, R, U = rows(g["A"]), rows(g["R"]), rows(g["U"])
    s, e, b, mu, v, d, bits = (rows(g[x])[0] for x in ("s", "e", "b", "mu", "v", "d", "bits"))
    assert A.shape == (m, n) and R.shape == (m, k) and U.shape == (n, k)
    assert np.array_equal(O.keygen(A, s, e, q), b)
    Ugot, vgot = O.encaps(A, b, pack_bits(R), pack_bits(mu), k, q)
    assert np.array_equal(Ugot, U) and np.array_equal(vgot, v)
    out, dgot = O.decaps(U, v, s, q, return_d=True)
    assert np.array_equal(dgot, d)
    assert np.array_equal(unpack_bits(out, k), bits)


# ---------------------------------------------------------------- P6 keygen

def brute_keygen(A, s, e, q):
    """independent: python big integers, one reduction at the very end"""
    m, n = A.shape
    return np.array([(sum(int(A[i, j]) * int(s[j]) for j in range(n)) + int(e[i])) % q for i in range(m)])


@pytest.mark.parametrize("q", [17, 3329, 65521, 65536])
@pytest.mark.parametrize("m,n", [(8, 4), (5, 7), (33, 16)])
def test_p6_keygen_brute_force(q, m, n):
    A, s, e = W.random_u16((m, n), q, 1), W.random_u16(n, q, 2), W.random_u16(m, q, 3)
    assert np.array_equal(O.keygen(A, s, e, q), brute_keygen(A, s, e, q))


def test_p6_keygen_extreme_values_do_not_overflow():
    for q in (65521, 65536):
        m, n = 4, 4096
        A = np.full((m, n), q - 1, np.uint16)
        s = np.full(n, q - 1, np.uint16)
        e = np.full(m, q - 1, np.uint16)
        want = (n * (q - 1) * (q - 1) + (q - 1)) % q
        assert np.all(O.keygen(A, s, e, q) == want)


@pytest.mark.parametrize("q", [65521, 65536])
def test_p6_keygen_linearity_and_special_vectors(q):
    m, n = 64, 48
    A = W.random_u16((m, n), q, 11)
    s1, s2 = W.random_u16(n, q, 12), W.random_u16(n, q, 13)
    e = W.random_u16(m, q, 14)
    zero_e, zero_s = np.zeros(m, np.uint16), np.zeros(n, np.uint16)
    s12 = ((s1.astype(np.int64) + s2) % q).astype(np.uint16)
    lhs = O.keygen(A, s12, zero_e, q).astype(np.int64)
    rhs = (O.keygen(A, s1, zero_e, q).astype(np.int64) + O.keygen(A, s2, zero_e, q)) % q
    assert np.array_equal(lhs, rhs)
    assert np.array_equal(O.keygen(A, zero_s, e, q), e)                  # s = 0 -> b = e
    for j in (0, 5, n - 1):                                               # s = e_j -> column j (+ e)
        u = zero_s.copy()
        u[j] = 1
        assert np.array_equal(O.keygen(A, u, e, q), (A[:, j].astype(np.int64) + e) % q)
    ones = np.ones(n, np.uint16)                                          # s = 1 -> row sums
    assert np.array_equal(O.keygen(A, ones, zero_e, q), A.astype(np.int64).sum(axis=1) % q)
    # a transposed operand would fail this: non-square A against int64 matmul
    assert np.array_equal(O.keygen(A, s1, e, q), (A.astype(np.int64) @ s1.astype(np.int64) + e) % q)


# ---------------------------------------------------------------- P8 encaps alone

@pytest.mark.parametrize("q", [17, 65521, 65536])
def test_p8_encaps_matches_int64_matmul_and_single_matvecs(q):
    m, n, k = 40, 24, 16
    A, b = W.random_u16((m, n), q, 21), W.random_u16(m, q, 22)
    R = (W.random_bytes(m * k, 23) & 1).reshape(m, k)
    mu = W.random_bytes(k, 24) & 1
    U, v = O.encaps(A, b, pack_bits(R), pack_bits(mu), k, q)
    A64, R64 = A.astype(np.int64), R.astype(np.int64)
    assert np.array_equal(U, (A64.T @ R64) % q)
    assert np.array_equal(v, (b.astype(np.int64) @ R64 + mu.astype(np.int64) * (q // 2)) % q)
    # batched == 256 (here k) independent single-bit encryptions:
    # column c of U is the mat-vec A^T r_c, done with the KEYGEN routine on A^T
    At = np.ascontiguousarray(A.T)
    for c in (0, 7, k - 1):
        col = O.keygen(At, R[:, c].astype(np.uint16), np.zeros(n, np.uint16), q)
        assert np.array_equal(U[:, c], col)
    # row-restricted variant agrees with the full one
    pick = np.array([0, 3, n - 1, 3], np.uint32)
    assert np.array_equal(O.encaps_rows(A, pack_bits(R), pick, k, q), U[pick])
    assert np.array_equal(O.encaps_v(b, pack_bits(R), pack_bits(mu), k, q), v)


@pytest.mark.parametrize("q", [65521, 65536])
def test_p8_encaps_one_hot_and_all_ones_R(q):
    m, n, k = 16, 8, 8
    A, b = W.random_u16((m, n), q, 31), W.random_u16(m, q, 32)
    mu = np.array([1, 0, 1, 1, 0, 0, 1, 0], np.uint8)
    R = np.zeros((m, k), np.uint8)
    R[5, 3] = 1                                     # single 1: column 3 picks row 5 of A
    U, v = O.encaps(A, b, pack_bits(R), pack_bits(mu), k, q)
    assert np.array_equal(U[:, 3], A[5, :])
    assert int(v[3]) == (int(b[5]) + (q // 2)) % q
    assert not U[:, [0, 1, 2, 4, 5, 6, 7]].any()
    assert np.array_equal(np.delete(v, 3), (np.delete(mu, 3).astype(np.int64) * (q // 2)) % q)
    R[:] = 1                                        # all ones: column sums of A, sum of b
    U, v = O.encaps(A, b, pack_bits(R), pack_bits(mu), k, q)
    assert np.array_equal(U, np.repeat((A.astype(np.int64).sum(axis=0) % q)[:, None], k, axis=1))
    assert np.array_equal(v, (int(b.astype(np.int64).sum()) + mu.astype(np.int64) * (q // 2)) % q)


def test_s11_encoding_constant():
    # floor(q/2): 32768 for q = 2^16, 32760 for q = 65521
    for q, half in ((65536, 32768), (65521, 32760)):
        v = O.encaps_v(np.zeros(8, np.uint16), np.zeros(8, np.uint8), np.array([0x01], np.uint8), 8, q)
        assert v.tolist() == [half, 0, 0, 0, 0, 0, 0, 0]


# ---------------------------------------------------------------- P10 rounding

@pytest.mark.parametrize("q", [65536, 65521, 17, 16, 2, 3])
def test_p10_rounding_exhaustive(q):
    for d in range(q):
        assert O.round_bit(d, q) == (1 if (4 * d >= q and 4 * d < 3 * q) else 0), (q, d)


def test_p10_pow2_rounding_is_a_shift():
    d = np.arange(65536)
    want = ((d + (1 << 14)) >> 15) & 1
    got = np.array([O.round_bit(int(x), 65536) for x in d])
    assert np.array_equal(got, want)


def test_o9_decaps_brute_force_and_sign():
    q, n, k = 65521, 12, 16
    U, v, s = W.random_u16((n, k), q, 41), W.random_u16(k, q, 42), W.random_u16(n, q, 43)
    out, d = O.decaps(U, v, s, q, return_d=True)
    want = np.array([(int(v[c]) - sum(int(U[j, c]) * int(s[j]) for j in range(n))) % q for c in range(k)])
    assert np.array_equal(d, want)
    assert np.array_equal(unpack_bits(out, k), [(1 if (4 * x >= q and 4 * x < 3 * q) else 0) for x in want])


# ---------------------------------------------------------------- P7 noise identity + round trip

def kem_from_seed(w: W.Workload, n=None, m=None, inst=0):
    """One instance of workload `w` (optionally at reduced n, m), every object drawn
    from the seeded AES-CTR streams (O3-O6)."""
    n, m = n or w.n, m or w.m
    A = O.sample_uniform(0, m * n, w.seed, O.TAG_A, 0, w.q).reshape(m, n)
    s = O.sample_uniform(0, n, w.seed, O.TAG_S, inst, w.q)
    e = O.sample_cbd(0, m, w.seed, O.TAG_E, inst, w.q, w.eta)
    Rbits = O.sample_bits(0, m * w.k, w.seed, O.TAG_R, inst)
    mubits = O.sample_bits(0, w.k, w.seed, O.TAG_MU, inst)
    return A, s, e, Rbits, mubits


@pytest.mark.parametrize("w,n,m", [(W.C1, None, None), (W.C3, 96, 192), (W.C4, 64, 128), (W.C2, 128, 256)])
def test_p7_noise_identity_and_every_bit_recovered(w, n, m):
    A, s, e, Rbits, mubits = kem_from_seed(w, n, m, inst=1)
    m_, n_ = A.shape
    q, k = w.q, w.k
    b = O.keygen(A, s, e, q)
    U, v = O.encaps(A, b, Rbits, mubits, k, q)
    out, d = O.decaps(U, v, s, q, return_d=True)
    assert np.array_equal(out, mubits)                                  # decaps recovers every bit
    # (v - U^T s - mu*floor(q/2)) mod q == e^T R mod q, exactly
    R = unpack_bits(Rbits, m_ * k).reshape(m_, k).astype(np.int64)
    mu = unpack_bits(mubits, k).astype(np.int64)
    e_signed = np.where(e.astype(np.int64) > q // 2, e.astype(np.int64) - q, e.astype(np.int64))
    noise = e_signed @ R
    assert np.array_equal((d.astype(np.int64) - mu * (q // 2)) % q, noise % q)
    assert np.abs(noise).max() <= m_ * w.eta and np.abs(noise).max() < q // 4


def test_c1_full_size_roundtrip_is_deterministically_correct():
    # S16: |e^T R| <= m*eta = 2048 < q/4 for C1, so recovery cannot fail
    w = W.C1
    for inst in (0, 3):
        A, s, e, Rbits, mubits = kem_from_seed(w, inst=inst)
        b = O.keygen(A, s, e, w.q)
        U, v = O.encaps(A, b, Rbits, mubits, w.k, w.q)
        assert np.array_equal(O.decaps(U, v, s, w.q), mubits)


def test_wrong_secret_does_not_decapsulate():
    w = W.C1
    A, s, e, Rbits, mubits = kem_from_seed(w, 64, 128)
    b = O.keygen(A, s, e, w.q)
    U, v = O.encaps(A, b, Rbits, mubits, w.k, w.q)
    s_bad = W.random_u16(s.shape, w.q, 99)
    wrong = unpack_bits(O.decaps(U, v, s_bad, w.q), w.k) != unpack_bits(mubits, w.k)
    assert 64 < wrong.sum() < 192                                       # ~half the bits flip


# ---------------------------------------------------------------- O11: FO re-encryption check (Alg. 5)

def fo_case(w, n, m, inst=0):
    A, s, e, Rbits, mubits = kem_from_seed(w, n, m, inst=inst)
    b = O.keygen(A, s, e, w.q)
    U, v = O.encaps(A, b, Rbits, mubits, w.k, w.q)
    return A, s, b, Rbits, mubits, U, v


@pytest.mark.parametrize("w,n,m", [(W.C1, 64, 128), (W.C3, 96, 192)])
def test_o11_honest_ciphertext_is_accepted_and_decrypts(w, n, m):
    A, s, b, Rbits, mubits, U, v = fo_case(w, n, m)
    out, ok = O.decaps_fo(A, b, U, v, s, Rbits, w.q)
    assert ok == 1 and np.array_equal(out, mubits)


@pytest.mark.parametrize("w,n,m", [(W.C1, 64, 128), (W.C3, 96, 192)])
def test_o11_any_change_of_the_ciphertext_is_rejected(w, n, m):
    """Alg. 5 l.4: c' = c fails for a tampered c -- both for a change too small to alter m' (the re-encryption
    of the SAME message differs from the tampered c in that element) and for one that flips a bit of m'."""
    A, s, b, Rbits, mubits, U, v = fo_case(w, n, m)
    q, k = w.q, w.k
    # +1 on one element of v: d moves by 1, far from the threshold -> m' unchanged, verdict 0
    v1 = v.copy(); v1[7] = (int(v1[7]) + 1) % q
    out, ok = O.decaps_fo(A, b, U, v1, s, Rbits, q)
    assert ok == 0 and np.array_equal(out, mubits)
    # +floor(q/2)+3 on one element of v: that bit of m' flips, and v' = b^T R + m'*floor(q/2) is 3 (or 2, odd q) away
    v2 = v.copy(); v2[200] = (int(v2[200]) + q // 2 + 3) % q
    out, ok = O.decaps_fo(A, b, U, v2, s, Rbits, q)
    flipped = unpack_bits(out, k) != unpack_bits(mubits, k)
    assert ok == 0 and flipped.sum() == 1 and flipped[200]
    # one element of U (first, last, middle), +1: rejected
    for (j, c) in ((0, 0), (n - 1, k - 1), (n // 2, 17)):
        U1 = U.copy(); U1[j, c] = (int(U1[j, c]) + 1) % q
        _, ok = O.decaps_fo(A, b, U1, v, s, Rbits, q)
        assert ok == 0, (j, c)
    # wrong coins: the re-encryption does not reproduce c
    R_bad = Rbits.copy(); R_bad[5] ^= 0x10
    out, ok = O.decaps_fo(A, b, U, v, s, R_bad, q)
    assert ok == 0 and np.array_equal(out, mubits)


def test_o11_coins_are_an_input_exact_half_shift_is_a_valid_ciphertext():
    """The reading taken (S19): the coins R are an INPUT of the check (the paper derives them
    through hashes that are outside the hot path).  Then, for q = 2^16, v + q/2 in one position is exactly the
    encryption of the message with that bit flipped under the same coins, so the check accepts it and m' differs
    in that bit -- binding the coins to m is the hash layer's job.  Pins the verdict to 'c' == c', nothing more."""
    w = W.C1
    A, s, b, Rbits, mubits, U, v = fo_case(w, 64, 128)
    v2 = v.copy(); v2[31] = (int(v2[31]) + w.q // 2) % w.q
    out, ok = O.decaps_fo(A, b, U, v2, s, Rbits, w.q)
    flipped = unpack_bits(out, w.k) != unpack_bits(mubits, w.k)
    assert ok == 1 and flipped.sum() == 1 and flipped[31]
