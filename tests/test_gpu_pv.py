"""GPU parity of N2 (the paper's own PKE variant): Gaussian / centred-uniform samplers and lwe_encaps_pv
against the oracle's O12-O14, bit for bit, and the whole KeyGen -> Encrypt -> Decrypt path from seeds on Table 1's first
parameter sets."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O  # noqa: E402
from paper_2606_01211_b200 import workloads as W  # noqa: E402


@pytest.fixture(scope="module")
def H():
    import gpu_helpers
    return gpu_helpers


def B():
    from paper_2606_01211_b200 import binding
    return binding


def dev_s8(H, a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int8)).cuda()


def empty_s8(*shape):
    import torch
    return torch.empty(*shape, dtype=torch.int8, device="cuda")


@pytest.mark.parametrize("sigma", [0.5, 1.0, 1.2, 1.7, 2.3, 2.8])      # 0.5 / 2.8: the limits the ABI accepts
@pytest.mark.parametrize("first,count,n_inst", [(0, 4096, 1), (40, 1000, 3), (8, 13, 2), (0, 1 << 16, 2)])
def test_gauss_samplers_match_oracle(H, sigma, first, count, n_inst):
    seed, q, inst0 = 77, 12289, 5
    with B().Context(64, 64, 256, q, 3, 1) as c:
        z8, z16 = empty_s8(n_inst, count), H.dev_empty_u16(n_inst, count)
        c.sample_gauss_s8(z8, first, count, seed, W.TAG_RG, inst0, n_inst, sigma)
        c.sample_gauss_u16(z16, first, count, seed, W.TAG_E, inst0, n_inst, sigma)
        g8, g16 = H.host_u8(z8.view(dtype=__import__("torch").uint8)).view(np.int8), H.host_u16(z16)
    for t in range(n_inst):
        assert np.array_equal(g8[t], O.sample_gauss(first, count, seed, O.TAG_RG, inst0 + t, sigma)), t
        assert np.array_equal(g16[t], O.sample_gauss(first, count, seed, O.TAG_E, inst0 + t, sigma, q)), t


@pytest.mark.parametrize("bound", [1, 2, 3, 127])
def test_cuniform_sampler_matches_oracle(H, bound):
    import torch
    seed, inst0, n_inst, first, count = 9, 2, 3, 5, 3001
    with B().Context(64, 64, 256, 3329, 3, 1) as c:
        out = empty_s8(n_inst, count)
        c.sample_cuniform_s8(out, first, count, seed, W.TAG_E2, inst0, n_inst, bound)
        g = H.host_u8(out.view(dtype=torch.uint8)).view(np.int8)
    for t in range(n_inst):
        assert np.array_equal(g[t], O.sample_cuniform(first, count, seed, O.TAG_E2, inst0 + t, bound)), t


@pytest.mark.parametrize("n,m,k,q,sigma,bound,inst0,n_inst", [
    (512, 512, 256, 3329, 2.3, 3, 0, 3), (264, 136, 128, 12289, 1.7, 2, 7, 2), (64, 64, 8, 65536, 0.5, 127, 1, 5),
    (1024, 1024, 256, 65537, 1.2, 2, 4, 2), (200, 72, 384, 65539, 2.8, 1, 0, 3)])
def test_sample_pke_equals_the_six_sampler_calls_and_the_oracle(H, n, m, k, q, sigma, bound, inst0, n_inst):
    """lwe_sample_pke (one launch) writes exactly what the six sampler calls write -- s (CBD), e, R, E1 (Gaussian), e2
    (centred uniform), mu (bits) -- on narrow (uint16 s, e) and wide (int8 s, e) contexts; each object against the
    oracle's own draw (O5 / O5s, O12, O13, O6)."""
    import torch
    seed, eta = 23, 3
    wide = q > 65536
    with B().Context(n, m, k, q, eta, n_inst) as c:
        s = empty_s8(n_inst, n) if wide else H.dev_empty_u16(n_inst, n)
        e = empty_s8(n_inst, m) if wide else H.dev_empty_u16(n_inst, m)
        R, E1, e2 = empty_s8(n_inst, m, k), empty_s8(n_inst, n, k), empty_s8(n_inst, k)
        mu = H.dev_empty_u8(n_inst, k // 8)
        for t_ in (s, e, R, E1, e2, mu):
            t_.fill_(0x55)
        c.sample_pke(s, e, R, E1, e2, mu, seed, inst0, n_inst, sigma, bound)
        torch.cuda.synchronize()
        as8 = lambda t_: t_.cpu().numpy().view(np.int8)  # noqa: E731
        gs = as8(s) if wide else H.host_u16(s)
        ge = as8(e) if wide else H.host_u16(e)
        gR, gE1, ge2, gmu = as8(R), as8(E1), as8(e2), H.host_u8(mu)
    for t in range(n_inst):
        i = inst0 + t
        if wide:
            assert np.array_equal(gs[t], O.sample_cbd_s8(0, n, seed, O.TAG_S, i, eta)), ("s", t)
            assert np.array_equal(ge[t], O.sample_gauss(0, m, seed, O.TAG_E, i, sigma)), ("e", t)
        else:
            assert np.array_equal(gs[t], O.sample_cbd(0, n, seed, O.TAG_S, i, q, eta)), ("s", t)
            assert np.array_equal(ge[t], O.sample_gauss(0, m, seed, O.TAG_E, i, sigma, q)), ("e", t)
        assert np.array_equal(gR[t].ravel(), O.sample_gauss(0, m * k, seed, O.TAG_RG, i, sigma)), ("R", t)
        assert np.array_equal(gE1[t].ravel(), O.sample_gauss(0, n * k, seed, O.TAG_E1, i, sigma)), ("E1", t)
        assert np.array_equal(ge2[t], O.sample_cuniform(0, k, seed, O.TAG_E2, i, bound)), ("e2", t)
        assert np.array_equal(gmu[t], O.sample_bits(0, k, seed, O.TAG_MU, i)), ("mu", t)


PV_SHAPES = [  # (n = m, k, q, batch)
    (256, 256, 3329, 1), (192, 256, 12289, 3), (200, 128, 12289, 3), (456, 256, 65521, 5), (1280, 256, 65536, 2),
    (64, 16, 3329, 2),
]


@pytest.mark.parametrize("path", [0, 1], ids=["tcgen05_pair", "simt"])
@pytest.mark.parametrize("n,k,q,batch", PV_SHAPES)
def test_encaps_pv_matches_oracle(H, path, n, k, q, batch):
    rng = np.random.default_rng(n + k)
    m = n
    A = W.random_u16((m, n), q, 71)
    t = W.random_u16((batch, m), q, 72)
    R = rng.integers(-12, 13, (batch, m, k)).astype(np.int8)
    E1 = rng.integers(-12, 13, (batch, n, k)).astype(np.int8)
    e2 = rng.integers(-3, 4, (batch, k)).astype(np.int8)
    mubits = W.random_bytes(batch * k // 8, 73).reshape(batch, -1)
    with B().Context(n, m, k, q, 3, batch) as c:
        c.set_option(B().OPT_ENCAPS_PATH, path)
        U, v = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k)
        U.fill_(-1)
        c.encaps_pv(H.dev(A), H.dev(t), dev_s8(H, R), dev_s8(H, E1), dev_s8(H, e2), H.dev(mubits), U, v, batch)
        gU, gv = H.host_u16(U), H.host_u16(v)
    for b in range(batch):
        Uo, vo = O.encaps_pv(A, t[b], R[b], E1[b], e2[b], mubits[b], q)
        assert np.array_equal(gv[b], vo), ("v", b)
        bad = np.argwhere(gU[b] != Uo)
        assert bad.size == 0, (f"U mismatch inst {b}: {len(bad)} entries, first {bad[:5].tolist()}")


@pytest.mark.parametrize("path", [0, 1], ids=["tcgen05_pair", "simt"])
def test_encaps_pv_extreme_accumulators(H, path):
    """|R| = 127 everywhere, A = q - 1, m = 65536: both signed byte-plane accumulators at +/- 255*127*65536 (just
    inside s32) and the signed recombination at its bounds, for both signs."""
    m = n = 65536
    n_small = 64
    for q in (12289, 65536):
        for sign in (1, -1):
            k, batch = 256, 1
            A = np.full((m, n_small), q - 1, np.uint16)
            t = np.full((batch, m), q - 1, np.uint16)
            R = np.full((batch, m, k), 127 * sign, np.int8)
            E1 = np.full((batch, n_small, k), -128 if sign < 0 else 127, np.int8)
            e2 = np.full((batch, k), 3 * sign, np.int8)
            mubits = np.full((batch, k // 8), 0xFF, np.uint8)
            with B().Context(n_small, m, k, q, 3, batch) as c:
                c.set_option(B().OPT_ENCAPS_PATH, path)
                U, v = H.dev_empty_u16(batch, n_small, k), H.dev_empty_u16(batch, k)
                c.encaps_pv(H.dev(A), H.dev(t), dev_s8(H, R), dev_s8(H, E1), dev_s8(H, e2), H.dev(mubits), U, v, batch)
                gU, gv = H.host_u16(U), H.host_u16(v)
            e1 = -128 if sign < 0 else 127
            assert np.all(gU == (m * (q - 1) * 127 * sign + e1) % q), (q, sign)
            assert np.all(gv == (m * (q - 1) * 127 * sign + 3 * sign + q // 2) % q), (q, sign)


@pytest.mark.parametrize("n,q,sigma,bound,batch", [(512, 3329, 2.3, 3, 2), (1024, 12289, 2.3, 3, 1), (2048, 12289, 2.3, 3, 1)])
def test_pv_full_path_from_seeds_matches_oracle_and_recovers_every_bit(H, n, q, sigma, bound, batch):
    """Table 1 rows 1-3 (row 4 at the size bench.py times it: tests/test_gpu_fullsize.py): every object drawn on the device from the seed, KeyGen (t = A s + e) ->
    Encrypt (U = A^T R + E1, v = t^T R + e2 + mu q/2) -> Decrypt, each output against the oracle's own draw."""
    import torch
    seed, k, inst0 = 41, 256, 3
    with B().Context(n, n, k, q, 3, batch) as c:
        dA = H.dev_empty_u16(n, n)
        c.sample_uniform(dA, 0, n * n, seed, W.TAG_A)
        s, e, t = H.dev_empty_u16(batch, n), H.dev_empty_u16(batch, n), H.dev_empty_u16(batch, n)
        R, E1, e2 = empty_s8(batch, n, k), empty_s8(batch, n, k), empty_s8(batch, k)
        mu, out = H.dev_empty_u8(batch, k // 8), H.dev_empty_u8(batch, k // 8)
        U, v = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k)
        c.sample_cbd(s, 0, n, seed, W.TAG_S, inst0, batch)                       # chi_3^n (the context's eta = 3)
        c.sample_gauss_u16(e, 0, n, seed, W.TAG_E, inst0, batch, sigma)
        c.sample_gauss_s8(R, 0, n * k, seed, W.TAG_RG, inst0, batch, sigma)
        c.sample_gauss_s8(E1, 0, n * k, seed, W.TAG_E1, inst0, batch, sigma)
        c.sample_cuniform_s8(e2, 0, k, seed, W.TAG_E2, inst0, batch, bound)
        c.sample_bits(mu, 0, k, seed, W.TAG_MU, inst0, batch)
        c.keygen(dA, 0, s, e, t, batch)
        c.encaps_pv(dA, t, R, E1, e2, mu, U, v, batch)
        c.decaps(U, v, s, out, batch)
        gA, gt, gU, gv, gout, gmu = H.host_u16(dA), H.host_u16(t), H.host_u16(U), H.host_u16(v), H.host_u8(out), H.host_u8(mu)
    A = O.sample_uniform(0, n * n, seed, O.TAG_A, 0, q).reshape(n, n)
    assert np.array_equal(gA, A)
    for b in range(batch):
        i = inst0 + b
        so = O.sample_cbd(0, n, seed, O.TAG_S, i, q, 3)
        eo = O.sample_gauss(0, n, seed, O.TAG_E, i, sigma, q)
        Ro = O.sample_gauss(0, n * k, seed, O.TAG_RG, i, sigma).reshape(n, k)
        E1o = O.sample_gauss(0, n * k, seed, O.TAG_E1, i, sigma).reshape(n, k)
        e2o = O.sample_cuniform(0, k, seed, O.TAG_E2, i, bound)
        muo = O.sample_bits(0, k, seed, O.TAG_MU, i)
        to = O.keygen(A, so, eo, q)
        Uo, vo = O.encaps_pv(A, to, Ro, E1o, e2o, muo, q)
        assert np.array_equal(gt[b], to) and np.array_equal(gmu[b], muo)
        assert np.array_equal(gU[b], Uo) and np.array_equal(gv[b], vo)
        assert np.array_equal(gout[b], O.decaps(Uo, vo, so, q))
        assert np.array_equal(gout[b], muo), "not every bit recovered"


@pytest.mark.parametrize("n,q,sigma,bound", [(4096, 12289, 1.7, 3), (8192, 65537, 1.2, 2)])
def test_sample_pke_at_the_sizes_bench_times_equals_the_six_sampler_calls(H, n, q, sigma, bound):
    """lwe_sample_pke in the launch configuration bench.py's N2 phases time (32 instances, Table 1 rows n = 4096 and
    n = 8192): byte for byte what the six single-object sampler calls write -- each of which is compared with the oracle
    in the tests above -- plus the oracle's own draw of one instance's s, e, e2, mu and of sampled blocks of R and E1."""
    import torch
    k, Bt, seed, eta = 256, 32, 9, 3
    wide = q > 65536
    with B().Context(n, n, k, q, eta, Bt) as c:
        def bufs():
            s = empty_s8(Bt, n) if wide else H.dev_empty_u16(Bt, n)
            e = empty_s8(Bt, n) if wide else H.dev_empty_u16(Bt, n)
            return s, e, empty_s8(Bt, n, k), empty_s8(Bt, n, k), empty_s8(Bt, k), H.dev_empty_u8(Bt, k // 8)
        one, six = bufs(), bufs()
        c.sample_pke(*one, seed, 0, Bt, sigma, bound)
        s, e, R, E1, e2, mu = six
        if wide:
            c.sample_cbd_s8(s, 0, n, seed, W.TAG_S, 0, Bt)
            c.sample_gauss_s8(e, 0, n, seed, W.TAG_E, 0, Bt, sigma)
        else:
            c.sample_cbd(s, 0, n, seed, W.TAG_S, 0, Bt)
            c.sample_gauss_u16(e, 0, n, seed, W.TAG_E, 0, Bt, sigma)
        c.sample_gauss_s8(R, 0, n * k, seed, W.TAG_RG, 0, Bt, sigma)
        c.sample_gauss_s8(E1, 0, n * k, seed, W.TAG_E1, 0, Bt, sigma)
        c.sample_cuniform_s8(e2, 0, k, seed, W.TAG_E2, 0, Bt, bound)
        c.sample_bits(mu, 0, k, seed, W.TAG_MU, 0, Bt)
        torch.cuda.synchronize()
        for name, a, b in zip("s e R E1 e2 mu".split(), one, six):
            assert torch.equal(a, b), name
        t = 17                                               # one instance against the oracle's own draws
        gR = one[2][t].cpu().numpy().view(np.int8).ravel()
        gE1 = one[3][t].cpu().numpy().view(np.int8).ravel()
        ge2 = one[4][t].cpu().numpy().view(np.int8)
        gmu = one[5][t].cpu().numpy()
    for first in (0, 8 * 1001, n * k - 4096):
        assert np.array_equal(gR[first:first + 4096], O.sample_gauss(first, 4096, seed, O.TAG_RG, t, sigma)), first
        assert np.array_equal(gE1[first:first + 4096], O.sample_gauss(first, 4096, seed, O.TAG_E1, t, sigma)), first
    assert np.array_equal(ge2, O.sample_cuniform(0, k, seed, O.TAG_E2, t, bound))
    assert np.array_equal(gmu, O.sample_bits(0, k, seed, O.TAG_MU, t))
