"""Pins of the oracle's N2 functions (the paper's own PKE variant: Gaussian e, r, e1; centred-uniform e2; CBD-3 secret;
square A; Table 1).  Nothing here calls the CUDA path."""
import numpy as np
import pytest
from scipy import integrate, stats

import oracle as O
from paper_2606_01211_b200 import workloads as W

SIGMAS = [1.0, 1.2, 1.7, 2.3]                      # every sigma of Table 1


# ---------------------------------------------------------------- O12: rounded Gaussian through a 16-bit CDT

@pytest.mark.parametrize("sigma", SIGMAS)
def test_o12_table_is_the_rounded_gaussian_cdf(sigma):
    """C[j] = round(65536 * P(round(sigma N) <= j - 12)), against scipy's normal CDF (its own implementation, not
    libm's erfc) and against numerical integration of the density."""
    cdt = O.gauss_cdt(sigma).astype(np.int64)
    assert np.all(np.diff(cdt) >= 0) and cdt[0] == 0 and cdt[-1] == 65536
    for j in range(2 * O.GAUSS_TAU):
        edge = (j - O.GAUSS_TAU + 0.5) / sigma
        assert abs(cdt[j] - 65536 * stats.norm.cdf(edge)) <= 0.5 + 1e-6, j
    j = O.GAUSS_TAU + 1                                # P(z <= 1) by quadrature of exp(-x^2/2)/sqrt(2 pi)
    area, _ = integrate.quad(lambda x: np.exp(-x * x / 2) / np.sqrt(2 * np.pi), -np.inf, 1.5 / sigma)
    assert abs(cdt[j] - 65536 * area) <= 0.5 + 1e-4


@pytest.mark.parametrize("sigma", SIGMAS)
def test_o12_integer_table_equals_the_60_digit_golden(sigma):
    """The INTEGER table itself, entry by entry, against tests/golden/gauss_cdt_table1.txt (written by
    make_gauss_cdt_golden.py with python `decimal` at 60 digits from a series for Phi: no libm, no oracle, no CUDA).
    The oracle and the CUDA host code both use libm's erfc in double; this pin fixes what they must produce."""
    from conftest import read_golden
    gold = [int(x) for x in read_golden("gauss_cdt_table1.txt")[f"sigma_{sigma}"].split()]
    assert len(gold) == 2 * O.GAUSS_TAU
    assert O.gauss_cdt(sigma).tolist() == gold


@pytest.mark.parametrize("sigma", SIGMAS)
def test_o12_exhaustive_histogram_symmetry_and_moments(sigma):
    """all 65536 words: the histogram IS the table's differences; it is the rounded-Gaussian pmf to 2^-16 per
    value, symmetric to one count, with mean 0 and variance sigma^2 + 1/12 (Sheppard) to 1e-3."""
    cdt = O.gauss_cdt(sigma)
    z = np.array([O.gauss_from_word(w, cdt) for w in range(65536)])
    vals, counts = np.unique(z, return_counts=True)
    hist = dict(zip(vals.tolist(), counts.tolist()))
    ext = np.concatenate([[0], cdt.astype(np.int64), [65536]])
    for zz in range(-O.GAUSS_TAU, O.GAUSS_TAU + 1):
        want = ext[zz + O.GAUSS_TAU + 1] - ext[zz + O.GAUSS_TAU]
        assert hist.get(zz, 0) == want, zz
        pmf = stats.norm.cdf((zz + 0.5) / sigma) - stats.norm.cdf((zz - 0.5) / sigma)
        assert abs(want / 65536 - pmf) <= 1.01 / 65536, zz
        assert abs(hist.get(zz, 0) - hist.get(-zz, 0)) <= 1, zz
    assert abs(z.mean()) < 2e-4
    assert abs(z.var() - (sigma * sigma + 1 / 12)) < 1e-3
    assert O.gauss_from_word(0, cdt) < 0 < O.gauss_from_word(65535, cdt)          # small words are the negative tail


def test_o12_stream_samples_follow_the_word_rule_and_both_encodings_agree():
    seed, inst, sigma, q = 21, 3, 1.7, 12289
    cdt = O.gauss_cdt(sigma)
    key, iv = O.seed_key(seed), O.object_iv(O.TAG_RG, 0, inst)
    ks = O.ctr_bytes(key, iv, 2 * 40, 2 * 500)
    words = ks[0::2].astype(np.uint32) | (ks[1::2].astype(np.uint32) << 8)         # LE16, elements 40..539
    z8 = O.sample_gauss(40, 500, seed, O.TAG_RG, inst, sigma)
    assert np.array_equal(z8, np.array([O.gauss_from_word(int(w), cdt) for w in words], np.int8))
    z16 = O.sample_gauss(40, 500, seed, O.TAG_RG, inst, sigma, q)
    assert np.array_equal(z16.astype(np.int64), z8.astype(np.int64) % q)
    assert np.array_equal(O.sample_gauss(0, 700, seed, O.TAG_RG, inst, sigma)[40:540], z8)     # offset reproducible
    big = O.sample_gauss(0, 1 << 18, seed, O.TAG_E1, 0, sigma).astype(np.float64)
    assert abs(big.mean()) < 0.02 and abs(big.var() - (sigma ** 2 + 1 / 12)) < 0.05


# ---------------------------------------------------------------- O13: centred uniform

@pytest.mark.parametrize("bound", [1, 2, 3])             # Table 1's k for e2
def test_o13_centred_uniform_range_rule_and_uniformity(bound):
    seed, inst, qq = 5, 2, 2 * bound + 1
    x = O.sample_cuniform(0, 1 << 16, seed, O.TAG_E2, inst, bound).astype(np.int64)
    assert x.min() == -bound and x.max() == bound
    counts = np.bincount(x + bound, minlength=qq)
    chi2 = ((counts - x.size / qq) ** 2 / (x.size / qq)).sum()
    assert chi2 < stats.chi2.ppf(1 - 1e-6, qq - 1)
    # attempt-0 words below T = q' floor(65536/q') are accepted as (c mod q') - bound
    ks = O.ctr_bytes(O.seed_key(seed), O.object_iv(O.TAG_E2, 0, inst), 0, 2 * 4096)
    c = ks[0::2].astype(np.int64) | (ks[1::2].astype(np.int64) << 8)
    T = qq * (65536 // qq)
    acc = c < T
    assert np.array_equal(x[:4096][acc], (c[acc] % qq) - bound)
    # rejected positions take the same position of attempt stream 1 (if that one is accepted)
    ks1 = O.ctr_bytes(O.seed_key(seed), O.object_iv(O.TAG_E2, 1, inst), 0, 2 * 4096)
    c1 = ks1[0::2].astype(np.int64) | (ks1[1::2].astype(np.int64) << 8)
    rej = (~acc) & (c1 < T)
    assert np.array_equal(x[:4096][rej], (c1[rej] % qq) - bound)


# ---------------------------------------------------------------- O14: Encrypt of the paper's PKE

def brute_encaps_pv(A, t, R, E1, e2, mu, q):
    m, n = A.shape
    k = len(e2)
    U = [[(sum(int(A[i][j]) * int(R[i][c]) for i in range(m)) + int(E1[j][c])) % q for c in range(k)] for j in range(n)]
    v = [(sum(int(t[i]) * int(R[i][c]) for i in range(m)) + int(e2[c]) + int(mu[c]) * (q // 2)) % q for c in range(k)]
    return np.array(U, np.uint16), np.array(v, np.uint16)


@pytest.mark.parametrize("q", [3329, 12289, 65521, 65536])
def test_o14_brute_force_with_python_integers(q):
    rng = np.random.default_rng(q)
    m, n, k = 9, 7, 16
    A, t = W.random_u16((m, n), q, 1), W.random_u16((m,), q, 2)
    R = rng.integers(-12, 13, (m, k)).astype(np.int8)
    E1 = rng.integers(-12, 13, (n, k)).astype(np.int8)
    e2 = rng.integers(-3, 4, k).astype(np.int8)
    mubits = W.random_bytes(k // 8, 3)
    mu = np.unpackbits(mubits, bitorder="little")[:k]
    U, v = O.encaps_pv(A, t, R, E1, e2, mubits, q)
    Ub, vb = brute_encaps_pv(A, t, R, E1, e2, mu, q)
    assert np.array_equal(U, Ub) and np.array_equal(v, vb)


def test_o14_reduces_to_the_binary_encaps():
    """R in {0,1}, E1 = 0, e2 = 0 is exactly O8 (BASELINE.json's Regev form)."""
    q, m, n, k = 65521, 48, 24, 32
    A, b = W.random_u16((m, n), q, 4), W.random_u16((m,), q, 5)
    Rbits, mubits = W.random_bytes(m * k // 8, 6), W.random_bytes(k // 8, 7)
    R = np.unpackbits(Rbits, bitorder="little")[: m * k].reshape(m, k).astype(np.int8)
    U, v = O.encaps_pv(A, b, R, np.zeros((n, k), np.int8), np.zeros(k, np.int8), mubits, q)
    U8, v8 = O.encaps(A, b, Rbits, mubits, k, q)
    assert np.array_equal(U, U8) and np.array_equal(v, v8)


def pv_instance(n, q, sigma, bound, k, seed, inst):
    A = O.sample_uniform(0, n * n, seed, O.TAG_A, 0, q).reshape(n, n)
    s = O.sample_cbd(0, n, seed, O.TAG_S, inst, q, 3)                                   # chi_3^n
    e = O.sample_gauss(0, n, seed, O.TAG_E, inst, sigma, q)
    R = O.sample_gauss(0, n * k, seed, O.TAG_RG, inst, sigma).reshape(n, k)
    E1 = O.sample_gauss(0, n * k, seed, O.TAG_E1, inst, sigma).reshape(n, k)
    e2 = O.sample_cuniform(0, k, seed, O.TAG_E2, inst, bound)
    mubits = O.sample_bits(0, k, seed, O.TAG_MU, inst)
    return A, s, e, R, E1, e2, mubits


@pytest.mark.parametrize("n,q,sigma,bound", [(512, 3329, 2.3, 3), (256, 12289, 2.3, 3)])
def test_o14_noise_identity_and_every_bit_recovered(n, q, sigma, bound):
    """Table 1's first parameter set and a smaller one: with t = A s + e,
    v - U^T s - mu floor(q/2) = e^T R + e2 - s^T E1 (mod q) exactly, and Decrypt (O9) returns every bit."""
    k = 256
    A, s, e, R, E1, e2, mubits = pv_instance(n, q, sigma, bound, k, seed=31, inst=2)
    t = O.keygen(A, s, e, q)
    U, v = O.encaps_pv(A, t, R, E1, e2, mubits, q)
    out, d = O.decaps(U, v, s, q, return_d=True)
    sgn = lambda x: np.where(x.astype(np.int64) > q // 2, x.astype(np.int64) - q, x.astype(np.int64))  # noqa: E731
    mu = np.unpackbits(mubits, bitorder="little")[:k].astype(np.int64)
    noise = sgn(e) @ R.astype(np.int64) + e2.astype(np.int64) - sgn(s) @ E1.astype(np.int64)
    assert np.array_equal((d.astype(np.int64) - mu * (q // 2)) % q, noise % q)
    assert np.abs(noise).max() < q // 4
    assert np.array_equal(out, mubits)


# ---------------------------------------------------------------- the paper's Table 1 as a fixture
def _table1_rows():
    from pathlib import Path
    rows = []
    for line in (Path(__file__).parent / "golden" / "paper_table1_params.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            n, q, sigma, kappa, eta, hard = line.split()
            rows.append((int(n), int(q), float(sigma), int(kappa), int(eta), int(hard)))
    return rows


def test_table1_rows_used_by_n2_are_the_papers():
    """workloads.PAPER_TABLE1 (what the N2 tests and bench.py run) is exactly the uint16-modulus part of the paper's
    Table 1, with the binomial eta = 3 secret of P:L70."""
    rows = _table1_rows()
    assert len(rows) == 9 and all(r[4] == 3 for r in rows)
    fit = [(n, q, s, kap) for n, q, s, kap, _, _ in rows if q <= 65536]
    assert fit == list(W.PAPER_TABLE1)
    assert all(q == 65537 for _, q, _, _, _, _ in rows[4:])


@pytest.mark.parametrize("row", range(4))
def test_table1_rows_decrypt_with_margin(row):
    """For every Table 1 row the library runs, the decryption noise e^T r + e2 - s^T e1 of the paper's PKE stays far
    inside the decoding threshold q/4 ("reliable decapsulation"): standard deviation from the closed-form
    variances of O5 (eta/2), O12 (sigma^2 + 1/12) and O13 (kappa(kappa+1)/3), margin in standard deviations."""
    n, q, sigma, kappa = W.PAPER_TABLE1[row]
    var_g = sigma * sigma + 1.0 / 12.0
    var = n * var_g * var_g + n * 1.5 * var_g + kappa * (kappa + 1) / 3.0        # e^T r  +  s^T e1  +  e2
    margin = (q / 4.0) / np.sqrt(var)
    assert margin > 4.0, (n, q, margin)
