"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(SURVEY 8(c) P11/P12): every object is drawn on the device from the config's seed exactly as
bench.py's step does, the oracle draws its own copy of whatever it needs from the same seed,
and the comparison is element by element on what the oracle can finish in seconds (C3: all of
it; C4/C5: sampled rows of b and U, all of v / mu') plus properties that hold at any size
(the noise identity v - U^T s - mu*floor(q/2) = e^T R over all k columns, every bit recovered,
stored A == regenerated A).  No oracle input comes from the GPU."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O  # noqa: E402
from paper_2606_01211_b200 import workloads as W  # noqa: E402


@pytest.fixture(scope="module")
def H():
    import gpu_helpers
    return gpu_helpers


def device_kem(H, c, w, inst0, batch, dA, regen_too=False):
    """bench.py's step on caller-owned buffers; returns the device tensors"""
    n, m, k = w.n, w.m, w.k
    s, e, b = H.dev_empty_u16(batch, n), H.dev_empty_u16(batch, m), H.dev_empty_u16(batch, m)
    Rbits, mubits = H.dev_empty_u8(batch, m * k // 8), H.dev_empty_u8(batch, k // 8)
    U, v, out = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k), H.dev_empty_u8(batch, k // 8)
    c.sample_kem(s, e, Rbits, mubits, w.seed, inst0, batch)          # the launch configuration bench.py times
    c.keygen(dA, 0, s, e, b, batch)
    g = dict(s=s, e=e, b=b, Rbits=Rbits, mubits=mubits, U=U, v=v, out=out)
    if regen_too:
        g["b_regen"] = H.dev_empty_u16(batch, m)
        c.keygen(None, w.seed, s, e, g["b_regen"], batch)
    c.encaps(dA, 0, b, Rbits, mubits, U, v, batch)
    c.decaps(U, v, s, out, batch)
    return g


def noise_identity_holds(w, U, v, s, e, Rbits, mubits):
    """(v - U^T s - mu*floor(q/2)) mod q == (e^T R) mod q for all k columns (P7), in exact integers"""
    q, k, m = w.q, w.k, e.size
    R = np.unpackbits(Rbits, bitorder="little")[: m * k].reshape(m, k).astype(np.int64)
    mu = np.unpackbits(mubits, bitorder="little")[:k].astype(np.int64)
    Us = (U.astype(np.uint64).T @ s.astype(np.uint64)) % np.uint64(q)           # < 2^16 * 2^16 * n < 2^64
    lhs = (v.astype(np.int64) - Us.astype(np.int64) - mu * (q // 2)) % q
    e_signed = np.where(e.astype(np.int64) > q // 2, e.astype(np.int64) - q, e.astype(np.int64))
    rhs = (e_signed @ R) % q
    return np.array_equal(lhs, rhs)


def test_c3_full_size_everything_against_the_oracle(H):
    """C3 (n=4096, m=8192, q=65521, eta=8): small enough for the oracle to compute every output."""
    w = W.C3
    n, m, k, q = w.n, w.m, w.k, w.q
    with H.make_ctx(w) as c:
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
        g = device_kem(H, c, w, 0, 1, dA, regen_too=True)
        A = H.host_u16(dA)
        got = {name: (H.host_u16(t) if t.dtype.itemsize == 2 else H.host_u8(t)) for name, t in g.items()}
    oi = H.OracleInstance(w, 0)
    assert np.array_equal(A, oi.A)
    assert np.array_equal(got["s"][0], oi.s) and np.array_equal(got["e"][0], oi.e)
    assert np.array_equal(got["Rbits"][0], oi.Rbits) and np.array_equal(got["mubits"][0], oi.mubits)
    b = O.keygen(oi.A, oi.s, oi.e, q)
    assert np.array_equal(got["b"][0], b) and np.array_equal(got["b_regen"][0], b)
    U, v = O.encaps(oi.A, b, oi.Rbits, oi.mubits, k, q)
    assert np.array_equal(got["v"][0], v)
    assert np.array_equal(got["U"][0], U)
    assert np.array_equal(got["out"][0], O.decaps(U, v, oi.s, q))
    assert np.array_equal(got["out"][0], oi.mubits)


def test_c4_bench_configuration_sampled_rows_and_invariants(H):
    """C4 exactly as bench.py launches it: 32 instances per call against one stored A (keygen as
    the tensor-core skinny GEMM, encaps as the CTA-pair tcgen05 GEMM with N = 8192 columns)."""
    w = W.C4
    n, m, k, q, Bt = w.n, w.m, w.k, w.q, w.batch
    inst0 = 64                                              # bench.py's third step on rank 0
    with H.make_ctx(w) as c:
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
        g = device_kem(H, c, w, inst0, Bt, dA)
        b, U, v, out = H.host_u16(g["b"]), H.host_u16(g["U"]), H.host_u16(g["v"]), H.host_u8(g["out"])
        s_g, e_g = H.host_u16(g["s"]), H.host_u16(g["e"])
        R_g, mu_g = H.host_u8(g["Rbits"]), H.host_u8(g["mubits"])
        # the same A, sampled: 3 random windows of the device copy against the oracle's stream
        A_dev_rows = {i: H.host_u16(dA[i]) for i in (0, 7777, m - 1)}
    for i, row in A_dev_rows.items():
        assert np.array_equal(row, O.sample_uniform(i * n, n, w.seed, O.TAG_A, 0, q))
    A = O.sample_uniform(0, m * n, w.seed, O.TAG_A, 0, q).reshape(m, n)
    rng = np.random.default_rng(404)
    for t in range(Bt):
        s = O.sample_uniform(0, n, w.seed, O.TAG_S, inst0 + t, q)
        e = O.sample_cbd(0, m, w.seed, O.TAG_E, inst0 + t, q, w.eta)
        Rbits = O.sample_bits(0, m * k, w.seed, O.TAG_R, inst0 + t)
        mubits = O.sample_bits(0, k, w.seed, O.TAG_MU, inst0 + t)
        assert np.array_equal(s_g[t], s) and np.array_equal(e_g[t], e), t
        assert np.array_equal(R_g[t], Rbits) and np.array_equal(mu_g[t], mubits), t
        assert np.array_equal(out[t], mubits), f"instance {t}: not every bit recovered"
        assert noise_identity_holds(w, U[t], v[t], s, e, Rbits, mubits), t
        if t in (0, 13, Bt - 1):                            # element-by-element on three instances
            bo = O.keygen(A, s, e, q)
            assert np.array_equal(b[t], bo), t
            assert np.array_equal(v[t], O.encaps_v(bo, Rbits, mubits, k, q)), t
            rows = np.unique(np.concatenate([[0, 1, 63, 64, 127, 128, n - 1], rng.integers(0, n, 41)])).astype(np.uint32)
            assert np.array_equal(U[t][rows], O.encaps_rows(A, Rbits, rows, k, q)), t


def test_c5_stored_and_regenerated_sampled_rows_columns_and_key_recovery(H):
    """C5 (n=32768, m=65536, A = 4 GiB): A stored on the device and regenerated (inside the keygen kernel;
    panel by panel for encaps) give the same b and the same U, v; the oracle recomputes 64 sampled rows of b (a row of A is a contiguous
    stream range) and 64 sampled rows of U x all 256 columns (row j of U needs column j of A, drawn
    by counter index: m AES blocks); the noise identity over all columns and full key recovery close
    the rest (BJ configs[4])."""
    import torch
    w = W.C5
    n, m, k, q = w.n, w.m, w.k, w.q
    rng = np.random.default_rng(505)
    brows = np.unique(np.concatenate([[0, 1, m - 1], rng.integers(0, m, 61)]))
    urows = np.unique(np.concatenate([[0, 1, 63, 64, n - 1], rng.integers(0, n, 59)]))
    with H.make_ctx(w) as c:
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
        g = device_kem(H, c, w, 0, 1, dA, regen_too=True)
        torch.cuda.synchronize()
        assert torch.equal(g["b"], g["b_regen"]), "stored A and regenerated A disagree (P11)"
        U_regen, v_regen = H.dev_empty_u16(1, n, k), H.dev_empty_u16(1, k)
        c.encaps(None, w.seed, g["b"], g["Rbits"], g["mubits"], U_regen, v_regen, 1)   # 64 panels of 1024 rows
        torch.cuda.synchronize()
        assert torch.equal(g["U"], U_regen) and torch.equal(g["v"], v_regen), "encaps: stored vs regenerated A (P11)"
        del U_regen
        b, U, v, out = H.host_u16(g["b"])[0], H.host_u16(g["U"])[0], H.host_u16(g["v"])[0], H.host_u8(g["out"])[0]
        s_g, e_g, R_g, mu_g = H.host_u16(g["s"])[0], H.host_u16(g["e"])[0], H.host_u8(g["Rbits"])[0], H.host_u8(g["mubits"])[0]
        A_dev_rows = H.host_u16(dA[torch.from_numpy(brows).cuda()])
        del dA
    s = O.sample_uniform(0, n, w.seed, O.TAG_S, 0, q)
    e = O.sample_cbd(0, m, w.seed, O.TAG_E, 0, q, w.eta)
    Rbits = O.sample_bits(0, m * k, w.seed, O.TAG_R, 0)
    mubits = O.sample_bits(0, k, w.seed, O.TAG_MU, 0)
    assert np.array_equal(s_g, s) and np.array_equal(e_g, e)
    assert np.array_equal(R_g, Rbits) and np.array_equal(mu_g, mubits)
    # sampled rows of b
    A_rows = np.stack([O.sample_uniform(int(i) * n, n, w.seed, O.TAG_A, 0, q) for i in brows])
    assert np.array_equal(A_dev_rows, A_rows)
    assert np.array_equal(b[brows], O.keygen(A_rows, s, e[brows], q))
    # sampled rows of U: A restricted to the sampled columns is an m x 64 matrix for the oracle
    A_cols = np.stack([O.sample_uniform_strided(int(j), n, m, w.seed, O.TAG_A, 0, q) for j in urows], axis=1)
    U_rows, _ = O.encaps(np.ascontiguousarray(A_cols), np.zeros(m, np.uint16), Rbits, mubits, k, q)
    assert np.array_equal(U[urows], U_rows)
    # everything else: exact identity over all columns + every bit recovered
    assert noise_identity_holds(w, U, v, s, e, Rbits, mubits)
    assert np.array_equal(out, mubits)
