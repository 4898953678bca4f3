"""Pins of the oracle's q > 65536 functions (N2 on Table 1's q = 65537 rows; readings S23-S25 of
DESIGN.md section 3): uint32 residues, 32-bit-word uniform sampler, int8 small objects.  Nothing here calls the CUDA path.

What fixes each function: the stream re-derived through OpenSSL (python `cryptography`), python big-integer brute
force, reduction to the already pinned uint16 functions for q <= 65536, the special case 2^16 = -1 (mod 65537),
the exact noise identity, and full key recovery on the paper's n = 8192 parameter set."""
import numpy as np
import pytest

import oracle as O

pytest.importorskip("cryptography.hazmat.primitives.ciphers")
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes  # noqa: E402

F4 = 65537


def stream(seed: int, tag: int, attempt: int, inst: int, nbytes: int) -> np.ndarray:
    key = seed.to_bytes(8, "little") + bytes(8)
    iv = ((tag << 56) + (attempt << 32) + inst).to_bytes(8, "big") + bytes(8)
    ks = Cipher(algorithms.AES(key), modes.CTR(iv)).encryptor().update(bytes(nbytes))
    return np.frombuffer(ks, dtype=np.uint8)


def words32(seed, tag, attempt, inst, count):
    return stream(seed, tag, attempt, inst, 4 * count).view("<u4").astype(np.uint64)


def centred(x, q):
    x = np.asarray(x).astype(np.int64)
    return np.where(x > q // 2, x - q, x)


# ---------------------------------------------------------------- O4w: uniform mod q on 32-bit words

@pytest.mark.parametrize("q", [F4, 65539, 100003, 3 << 29, (1 << 31) - 1, 12289])
def test_o4w_follows_the_attempt_streams_of_32_bit_words(q):
    """an independent walk over the attempt streams through OpenSSL; q = 3 * 2^29 rejects 25 % of the words"""
    N, seed, inst = 1 << 13, 5, 7
    T = q * ((1 << 32) // q)
    want = np.zeros(N, np.uint64)
    pending = np.arange(N)
    a = 0
    while pending.size:
        c = words32(seed, O.TAG_A, a, inst, N)[pending]
        ok = c < T
        want[pending[ok]] = c[ok] % q
        pending = pending[~ok]
        a += 1
    got = O.sample_uniform32(0, N, seed, O.TAG_A, inst, q)
    assert got.max() < q
    assert np.array_equal(got.astype(np.uint64), want)
    if q == 3 << 29:
        assert a >= 3, "no rejection was exercised"


def test_o4w_subrange_strided_and_uniformity():
    full = O.sample_uniform32(0, 6000, 3, O.TAG_A, 0, F4)
    for first, count in [(0, 1), (1, 7), (3, 2), (4, 4), (13, 2000), (5999, 1)]:
        assert np.array_equal(O.sample_uniform32(first, count, 3, O.TAG_A, 0, F4), full[first:first + count])
    pos = 5 + 37 * np.arange(150)
    assert np.array_equal(O.sample_uniform32_strided(5, 37, 150, 3, O.TAG_A, 0, F4), full[pos])
    # the block-wise walk of the contiguous sampler against the element-wise definition, rejection included
    for q in (F4, 3 << 29):
        assert np.array_equal(O.sample_uniform32(3, 3001, 13, O.TAG_A, 2, q),
                              O.sample_uniform32_strided(3, 1, 3001, 13, O.TAG_A, 2, q))
    # chi-square over 257 buckets of 255 values (65535 = 257 * 255; the two top values 65535, 65536 left out)
    big = O.sample_uniform32(0, 1 << 20, 11, O.TAG_A, 0, F4)
    assert big.max() == F4 - 1 or big.max() < F4
    assert (big == F4 - 1).sum() < 60                        # expected 16, the value only a 17-bit type can hold
    inside = big[big < 65535]
    counts = np.bincount(inside // 255, minlength=257).astype(np.float64)
    exp = inside.size / 257
    chi2 = ((counts - exp) ** 2 / exp).sum()
    assert chi2 < 256 + 5 * np.sqrt(2 * 256)


# ---------------------------------------------------------------- O5s: signed CBD

@pytest.mark.parametrize("eta", [1, 3, 4, 8])
def test_o5s_is_o5_before_the_reduction(eta):
    q = 3329
    z = O.sample_cbd_s8(40, 3000, 9, O.TAG_S, 2, eta)
    assert z.min() >= -eta and z.max() <= eta and (z < 0).any() and (z > 0).any()
    assert np.array_equal(z.astype(np.int64) % q, O.sample_cbd(40, 3000, 9, O.TAG_S, 2, q, eta).astype(np.int64))
    # sign convention: low byte counts up, high byte counts down (O5)
    w = stream(9, O.TAG_S, 0, 2, 2 * 3040).view("<u2")[40:]
    M = (1 << eta) - 1
    pc = lambda x: np.array([bin(int(v)).count("1") for v in x])  # noqa: E731
    assert np.array_equal(z, pc(w & M) - pc((w >> 8) & M))


# ---------------------------------------------------------------- O7w / O14w / O9w: brute force and reductions

def brute_keygen(A, s, e, q):
    m, n = A.shape
    return [(sum(int(A[i, j]) * int(s[j]) for j in range(n)) + int(e[i])) % q for i in range(m)]


def brute_encaps(A, t, R, E1, e2, mub, q):
    m, n = A.shape
    k = R.shape[1]
    U = [[(sum(int(A[i, j]) * int(R[i, c]) for i in range(m)) + int(E1[j, c])) % q for c in range(k)] for j in range(n)]
    v = [(sum(int(t[i]) * int(R[i, c]) for i in range(m)) + int(e2[c]) + int(mub[c]) * (q // 2)) % q for c in range(k)]
    return U, v


def small_case(q, m, n, k, seed):
    rng = np.random.default_rng(seed)
    A = rng.integers(0, q, (m, n), dtype=np.uint64).astype(np.uint32)
    A[0, 0] = q - 1                                           # the value a uint16 cannot hold (q = 65537: 65536)
    A[m - 1, n - 1] = q - 1
    s = rng.integers(-3, 4, n).astype(np.int8)
    e = rng.integers(-12, 13, m).astype(np.int8)
    R = rng.integers(-12, 13, (m, k)).astype(np.int8)
    E1 = rng.integers(-12, 13, (n, k)).astype(np.int8)
    e2 = rng.integers(-3, 4, k).astype(np.int8)
    mubits = rng.integers(0, 256, k // 8).astype(np.uint8)
    return A, s, e, R, E1, e2, mubits


@pytest.mark.parametrize("q", [F4, 65539, 100003, 131071])
def test_o7w_o14w_o9w_python_big_integer_brute_force(q):
    m, n, k = 12, 12, 8
    A, s, e, R, E1, e2, mubits = small_case(q, m, n, k, q)
    mub = np.unpackbits(mubits, bitorder="little")[:k]
    t = O.keygen_w(A, s, e, q)
    assert t.tolist() == brute_keygen(A, s, e, q)
    U, v = O.encaps_pv_w(A, t, R, E1, e2, mubits, q)
    Ub, vb = brute_encaps(A, t, R, E1, e2, mub, q)
    assert U.tolist() == Ub and v.tolist() == vb
    out, d = O.decaps_w(U, v, s, q, return_d=True)
    dw = [(int(v[c]) - sum(int(U[j, c]) * int(s[j]) for j in range(n))) % q for c in range(k)]
    assert d.tolist() == dw
    bits = [1 if (4 * x >= q and 4 * x < 3 * q) else 0 for x in dw]
    assert np.unpackbits(out, bitorder="little")[:k].tolist() == bits


@pytest.mark.parametrize("q", [3329, 12289, 65521, 65536])
def test_wide_functions_reduce_to_the_uint16_ones_for_small_moduli(q):
    m, n, k = 40, 24, 16
    A, s, e, R, E1, e2, mubits = small_case(q, m, n, k, 7 * q)
    res = lambda x: (x.astype(np.int64) % q).astype(np.uint16)  # noqa: E731
    t = O.keygen_w(A, s, e, q)
    assert np.array_equal(t, O.keygen(A.astype(np.uint16), res(s), res(e), q))
    U, v = O.encaps_pv_w(A, t, R, E1, e2, mubits, q)
    U16, v16 = O.encaps_pv(A.astype(np.uint16), t.astype(np.uint16), R, E1, e2, mubits, q)
    assert np.array_equal(U, U16) and np.array_equal(v, v16)
    out, d = O.decaps_w(U, v, s, q, return_d=True)
    out16, d16 = O.decaps(U16, v16, res(s), q, return_d=True)
    assert np.array_equal(out, out16) and np.array_equal(d, d16)


def test_two_to_the_sixteen_is_minus_one_mod_65537():
    """A = 65536 everywhere: t_i = e_i - sum_j s_j and U_jc = E1_jc - sum_i R_ic (mod 65537) -- the top bit of a 17-bit
    residue weighs -1; a path that drops or mis-weighs it fails here."""
    q, m, n, k = F4, 48, 32, 16
    _, s, e, R, E1, e2, mubits = small_case(q, m, n, k, 3)
    A = np.full((m, n), 65536, np.uint32)
    t = O.keygen_w(A, s, e, q)
    assert np.array_equal(t.astype(np.int64), (e.astype(np.int64) - int(s.astype(np.int64).sum())) % q)
    U, v = O.encaps_pv_w(A, t, R, E1, e2, mubits, q)
    colsum = R.astype(np.int64).sum(axis=0)
    assert np.array_equal(U.astype(np.int64), (E1.astype(np.int64) - colsum[None, :]) % q)
    # linearity of keygen in s (e = 0)
    s2 = np.roll(s, 5)
    z = np.zeros(m, np.int8)
    A2 = small_case(q, m, n, k, 4)[0]
    lhs = O.keygen_w(A2, (s.astype(np.int64) + s2).astype(np.int8), z, q).astype(np.int64)
    rhs = (O.keygen_w(A2, s, z, q).astype(np.int64) + O.keygen_w(A2, s2, z, q)) % q
    assert np.array_equal(lhs, rhs)


def test_o9w_rounding_exhaustive_for_65537():
    """U = 0, v = d: every d in [0, 65537) against the rational rule 1 iff q/4 <= d < 3q/4 (S12; no ties, q odd)"""
    q, n = F4, 8
    s = np.ones(n, np.int8)
    k = 1 << 10
    U = np.zeros((n, k), np.uint32)
    for d0 in range(0, q, k):
        d = np.arange(d0, d0 + k) % q
        out, dd = O.decaps_w(U, d.astype(np.uint32), s, q, return_d=True)
        assert np.array_equal(dd, d)
        want = ((4 * d >= q) & (4 * d < 3 * q)).astype(np.uint8)
        assert np.array_equal(np.unpackbits(out, bitorder="little")[:k], want)


# ---------------------------------------------------------------- the paper's parameter set n = 8192

def table1_row(n):
    """(n, q, sigma, kappa, eta) of Table 1 from the text fixture"""
    from conftest import GOLDEN
    for line in (GOLDEN / "paper_table1_params.txt").read_text().splitlines():
        r = line.split("#", 1)[0].split()
        if r and int(r[0]) == n:
            return int(r[0]), int(r[1]), float(r[2]), int(r[3]), int(r[4])
    raise KeyError(n)


def draw_instance(n, q, sigma, kappa, eta, k, seed, inst):
    s = O.sample_cbd_s8(0, n, seed, O.TAG_S, inst, eta)
    e = O.sample_gauss(0, n, seed, O.TAG_E, inst, sigma)
    R = O.sample_gauss(0, n * k, seed, O.TAG_RG, inst, sigma).reshape(n, k)
    E1 = O.sample_gauss(0, n * k, seed, O.TAG_E1, inst, sigma).reshape(n, k)
    e2 = O.sample_cuniform(0, k, seed, O.TAG_E2, inst, kappa)
    mubits = O.sample_bits(0, k, seed, O.TAG_MU, inst)
    return s, e, R, E1, e2, mubits


def noise_identity(U, v, s, e, R, E1, e2, mubits, q):
    k = v.size
    mub = np.unpackbits(mubits, bitorder="little")[:k].astype(np.int64)
    ss = s.astype(np.int64)
    Us = U.astype(np.int64).T @ ss                            # exact in int64: |U^T s| < 2^17 * 8 * n < 2^63
    lhs = (v.astype(np.int64) - Us - mub * (q // 2)) % q
    rhs = (e.astype(np.int64) @ R.astype(np.int64) + e2.astype(np.int64) - ss @ E1.astype(np.int64)) % q
    return np.array_equal(lhs, rhs)


def test_noise_identity_and_key_recovery_at_q_65537_small_n():
    n, q, sigma, kappa, eta = 1024, F4, 1.2, 2, 3
    k, seed = 256, 31
    A = O.sample_uniform32(0, n * n, seed, O.TAG_A, 0, q).reshape(n, n)
    for inst in (0, 5):
        s, e, R, E1, e2, mubits = draw_instance(n, q, sigma, kappa, eta, k, seed, inst)
        t = O.keygen_w(A, s, e, q)
        U, v = O.encaps_pv_w(A, t, R, E1, e2, mubits, q)
        assert noise_identity(U, v, s, e, R, E1, e2, mubits, q)
        assert np.array_equal(O.decaps_w(U, v, s, q), mubits)


def test_table1_row_n8192_bits_recovered():
    """Table 1 row 5 (n = 8192, q = 65537, sigma = 1.2, e2 in [-2, 2], eta = 3) on the oracle.  The k = 256
    columns of an instance are independent of one another, so the first 32 of them (message bits 0..31, the matching
    columns of R, E1, e2) are the same computation at an eighth of the cost: the exact noise identity and
    decaps(encaps(mu)) == mu on those columns, with all n^2 elements of A (1024 of them equal to 65536) in play."""
    n, q, sigma, kappa, eta = table1_row(8192)
    assert (q, sigma, kappa, eta) == (F4, 1.2, 2, 3)
    k, kk, seed, inst = 256, 32, 8, 0
    A = O.sample_uniform32(0, n * n, seed, O.TAG_A, 0, q).reshape(n, n)
    assert (A == 65536).sum() > 500                            # ~1024 entries only a 17-bit type can hold
    s, e, R, E1, e2, mubits = draw_instance(n, q, sigma, kappa, eta, k, seed, inst)
    R, E1, e2, mubits = np.ascontiguousarray(R[:, :kk]), np.ascontiguousarray(E1[:, :kk]), e2[:kk], mubits[: kk // 8]
    t = O.keygen_w(A, s, e, q)
    U, v = O.encaps_pv_w(A, t, R, E1, e2, mubits, q)
    assert noise_identity(U, v, s, e, R, E1, e2, mubits, q)
    assert np.array_equal(O.decaps_w(U, v, s, q), mubits)
