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
    """C4 exactly as bench.py launches it, compared ELEMENT BY ELEMENT on 3 of the 32 instances (b and v in full, 48
    sampled rows of U); the other 29 instances rest on the exact noise identity over all columns plus full key
    recovery (an O(mk) check of the O(mnk) contraction).  32 instances per call against one stored A (keygen as
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


def test_c4_kem_host_real_size_instances_through_the_chunk_pipeline(H):
    """lwe_kem_host in the shape bench.py's e2e leg times: C4, 32 instances in pinned HOST buffers, KeyGen once for the
    batch, then chunks of 1, 1, 2, 4, 8, 16 instances through the copy-in / Encrypt + Decrypt / copy-out pipeline.  Inputs are numpy-seeded (not the method's draws);
    b and v of every instance in full, 24 sampled rows of U on 7 instances (at least one per chunk), the noise
    identity and the recovered bits on all 32."""
    import torch
    w = W.C4
    n, m, k, q, Bt = w.n, w.m, w.k, w.q, w.batch
    rng = np.random.default_rng(88)
    s = W.random_u16((Bt, n), q, 801)
    e_signed = rng.integers(-4, 5, (Bt, m))
    e = (e_signed % q).astype(np.uint16)
    Rbits = W.random_bytes(Bt * m * k // 8, 802).reshape(Bt, -1)
    mubits = W.random_bytes(Bt * k // 8, 803).reshape(Bt, -1)

    def pinned(a):
        return torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a).pin_memory()

    h_s, h_e, h_R, h_mu = pinned(s), pinned(e), pinned(Rbits), pinned(mubits)
    h_b = torch.zeros(Bt, m, dtype=torch.int16).pin_memory()
    h_U = torch.zeros(Bt, n, k, dtype=torch.int16).pin_memory()
    h_v = torch.zeros(Bt, k, dtype=torch.int16).pin_memory()
    h_out = torch.zeros(Bt, k // 8, dtype=torch.uint8).pin_memory()
    with H.make_ctx(w) as c:
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
        c.kem_host(dA, 0, h_s, h_e, h_R, h_mu, h_b, h_U, h_v, h_out, Bt)
    A = O.sample_uniform(0, m * n, w.seed, O.TAG_A, 0, q).reshape(m, n)
    gb, gU, gv, gout = (h_b.numpy().view(np.uint16), h_U.numpy().view(np.uint16), h_v.numpy().view(np.uint16), h_out.numpy())
    for t in range(Bt):
        bo = O.keygen(A, s[t], e[t], q)
        assert np.array_equal(gb[t], bo), ("b", t)
        assert np.array_equal(gv[t], O.encaps_v(bo, Rbits[t], mubits[t], k, q)), ("v", t)
        assert noise_identity_holds(w, gU[t], gv[t], s[t], e[t], Rbits[t], mubits[t]), t
        assert np.array_equal(gout[t], mubits[t]), f"instance {t}: not every bit recovered"
        if t in (0, 1, 3, 5, 10, 21, 31):                 # at least one instance of every chunk
            rows = np.unique(np.concatenate([[0, 64, n - 1], rng.integers(0, n, 21)])).astype(np.uint32)
            assert np.array_equal(gU[t][rows], O.encaps_rows(A, Rbits[t], rows, k, q)), ("U", t)


def test_paper_variant_n4096_batch32_as_bench_times_it(H):
    """N2 at the size bench.py's `paper_variant_n4096_B32` phase times (Table 1 row n = 4096, q = 12289, sigma = 1.7,
    e2 in [-3, 3], eta = 3): every object drawn on the device from the seed as the phase does; t and v in full and
    40 sampled rows of U element by element on 3 instances, the exact noise identity
    v - U^T s - mu floor(q/2) = e^T R + e2 - s^T E1 (mod q) and every recovered bit on all 32."""
    import torch
    n, q, sigma, bound = W.PAPER_TABLE1[3]
    k, Bt, seed = 256, 32, 6
    s8 = dict(dtype=torch.int8, device="cuda")
    from paper_2606_01211_b200 import binding as Bd
    with Bd.Context(n, n, k, q, 3, Bt) as c:
        dA = H.dev_empty_u16(n, n)
        c.sample_uniform(dA, 0, n * n, seed, W.TAG_A)
        s, e, t = H.dev_empty_u16(Bt, n), H.dev_empty_u16(Bt, n), H.dev_empty_u16(Bt, n)
        R, E1, e2 = torch.empty(Bt, n, k, **s8), torch.empty(Bt, n, k, **s8), torch.empty(Bt, k, **s8)
        mu, out = H.dev_empty_u8(Bt, k // 8), H.dev_empty_u8(Bt, k // 8)
        U, v = H.dev_empty_u16(Bt, n, k), H.dev_empty_u16(Bt, k)
        c.sample_cbd(s, 0, n, seed, W.TAG_S, 0, Bt)
        c.sample_gauss_u16(e, 0, n, seed, W.TAG_E, 0, Bt, sigma)
        c.sample_gauss_s8(R, 0, n * k, seed, W.TAG_RG, 0, Bt, sigma)
        c.sample_gauss_s8(E1, 0, n * k, seed, W.TAG_E1, 0, Bt, sigma)
        c.sample_cuniform_s8(e2, 0, k, seed, W.TAG_E2, 0, Bt, bound)
        c.sample_bits(mu, 0, k, seed, W.TAG_MU, 0, Bt)
        c.keygen(dA, 0, s, e, t, Bt)
        c.encaps_pv(dA, t, R, E1, e2, mu, U, v, Bt)
        c.decaps(U, v, s, out, Bt)
        gA, gt, gU, gv, gout = H.host_u16(dA), H.host_u16(t), H.host_u16(U), H.host_u16(v), H.host_u8(out)
    A = O.sample_uniform(0, n * n, seed, O.TAG_A, 0, q).reshape(n, n)
    assert np.array_equal(gA, A)
    rng = np.random.default_rng(4096)
    centred = lambda x: np.where(x.astype(np.int64) > q // 2, x.astype(np.int64) - q, x.astype(np.int64))  # noqa: E731
    for b in range(Bt):
        so = O.sample_cbd(0, n, seed, O.TAG_S, b, q, 3)
        eo = O.sample_gauss(0, n, seed, O.TAG_E, b, sigma, q)
        Ro = O.sample_gauss(0, n * k, seed, O.TAG_RG, b, sigma).reshape(n, k)
        E1o = O.sample_gauss(0, n * k, seed, O.TAG_E1, b, sigma).reshape(n, k)
        e2o = O.sample_cuniform(0, k, seed, O.TAG_E2, b, bound)
        muo = O.sample_bits(0, k, seed, O.TAG_MU, b)
        mub = np.unpackbits(muo, bitorder="little")[:k].astype(np.int64)
        # exact identity over all columns (python-size integers stay far below 2^63 here)
        ss, ee = centred(so), centred(eo)
        Us = (gU[b].astype(np.int64).T @ ss)
        lhs = (gv[b].astype(np.int64) - Us - mub * (q // 2)) % q
        rhs = (ee @ Ro.astype(np.int64) + e2o.astype(np.int64) - ss @ E1o.astype(np.int64)) % q
        assert np.array_equal(lhs, rhs), b
        assert np.array_equal(gout[b], muo), f"instance {b}: not every bit recovered"
        if b in (0, 17, Bt - 1):
            to = O.keygen(A, so, eo, q)
            assert np.array_equal(gt[b], to), b
            rows = np.unique(np.concatenate([[0, 63, 64, n - 1], rng.integers(0, n, 36)]))
            # rows of U = A^T R + E1: the oracle on the sampled columns of A (an n x |rows| matrix)
            Uo, vo = O.encaps_pv(np.ascontiguousarray(A[:, rows]), to, Ro, E1o[rows], e2o, muo, q)
            assert np.array_equal(gU[b][rows], Uo), b
            assert np.array_equal(gv[b], vo), b
