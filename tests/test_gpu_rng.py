"""GPU parity, a1/a2: lwe_rng_fill and the samplers against the oracle, byte for byte
(SURVEY 8(c) P3, P4, P5).  All calls go through the C ABI (ctypes binding)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O  # noqa: E402
from paper_2606_01211_b200 import workloads as W  # noqa: E402


@pytest.fixture(scope="module")
def H():
    import gpu_helpers
    return gpu_helpers


@pytest.fixture(scope="module")
def ctx(H):
    with H.make_ctx(W.C1) as c:
        yield c


@pytest.mark.parametrize("offset,nbytes", [(0, 16), (0, 1), (0, 4096 + 5), (16, 333), (7, 100), (15, 2), (1, 16),
                                            (123457, 70001), ((1 << 36) + 9, 257), (0, 1 << 22)])
def test_rng_fill_matches_oracle_stream(H, ctx, offset, nbytes):
    rng = np.random.default_rng(offset % 1000 + nbytes)
    key, iv = rng.bytes(16), rng.bytes(16)
    out = H.dev_empty_u8(nbytes + 64)
    out.fill_(0xAA)
    ctx.rng_fill(out, nbytes, key, iv, offset)
    got = H.host_u8(out)
    assert np.array_equal(got[:nbytes], O.ctr_bytes(key, iv, offset, nbytes))
    assert np.all(got[nbytes:] == 0xAA)                         # nothing written past the end


def test_rng_fill_counter_carry_and_wrap(H, ctx):
    key = bytes(16)
    for iv in (bytes(8) + b"\xff" * 8, b"\xff" * 16, b"\x00" * 7 + b"\x01" + b"\xff" * 7 + b"\xfe"):
        out = H.dev_empty_u8(80)
        ctx.rng_fill(out, 80, key, iv, 0)
        assert np.array_equal(H.host_u8(out), O.ctr_bytes(key, iv, 0, 80))


def test_rng_fill_subrange_equals_slice_of_bigger_fill(H, ctx):
    key, iv = bytes(range(16)), bytes(range(16, 32))
    big = H.dev_empty_u8(5000)
    ctx.rng_fill(big, 5000, key, iv, 0)
    big = H.host_u8(big)
    for a, b in [(1, 100), (16, 32), (17, 4000), (4999, 1)]:
        part = H.dev_empty_u8(b)
        ctx.rng_fill(part, b, key, iv, a)
        assert np.array_equal(H.host_u8(part), big[a:a + b])


@pytest.mark.parametrize("q", [65536, 65521, 40000, 3329, 251, 17, 3, 2])
def test_sample_uniform_matches_oracle(H, q):
    with H.make_ctx(W.C1, q=q, max_batch=4) as c:
        for first, count, inst0, n_inst in [(0, 8192, 0, 1), (8, 1000, 3, 2), (4096, 1 << 16, 1, 3), (0, 13, 0, 2)]:
            out = H.dev_empty_u16(n_inst, count)
            c.sample_uniform(out, first, count, 7, W.TAG_A, inst0, n_inst)
            got = H.host_u16(out)
            for t in range(n_inst):
                assert np.array_equal(got[t], O.sample_uniform(first, count, 7, O.TAG_A, inst0 + t, q)), (q, first, t)


@pytest.mark.parametrize("q,eta", [(65536, 4), (65521, 8), (65536, 1), (17, 3), (3, 8)])
def test_sample_cbd_matches_oracle(H, q, eta):
    import paper_2606_01211_b200.binding as B
    with B.Context(256, 512, 256, q, eta, 4) as c:
        for first, count, inst0, n_inst in [(0, 4096, 0, 1), (16, 999, 2, 3)]:
            out = H.dev_empty_u16(n_inst, count)
            c.sample_cbd(out, first, count, 11, W.TAG_E, inst0, n_inst)
            got = H.host_u16(out)
            for t in range(n_inst):
                assert np.array_equal(got[t], O.sample_cbd(first, count, 11, O.TAG_E, inst0 + t, q, eta))


@pytest.mark.parametrize("first_bit,nbits,n_inst", [(0, 256, 1), (0, 512 * 256, 2), (8, 256, 3), (64, 1000, 2),
                                                     (24, 13, 2), (0, 1, 1), (128, 131, 4)])
def test_sample_bits_matches_oracle(H, ctx, first_bit, nbits, n_inst):
    nbytes = (nbits + 7) // 8
    out = H.dev_empty_u8(n_inst * nbytes + 32)
    out.fill_(0x55)
    ctx.sample_bits(out, first_bit, nbits, 5, W.TAG_R, 1, n_inst)
    got = H.host_u8(out)
    for t in range(n_inst):
        assert np.array_equal(got[t * nbytes:(t + 1) * nbytes], O.sample_bits(first_bit, nbits, 5, O.TAG_R, 1 + t))
    assert np.all(got[n_inst * nbytes:] == 0x55)


def test_argument_errors_do_not_launch(H, ctx):
    import paper_2606_01211_b200.binding as B
    out = H.dev_empty_u16(64)
    n0 = ctx.launch_count()
    with pytest.raises(B.LweError) as ei:
        ctx.sample_uniform(out, 3, 8, 1, W.TAG_A)              # first not a multiple of 8
    assert ei.value.code == -2
    with pytest.raises(B.LweError) as ei:
        ctx.sample_uniform(out.data_ptr() + 2, 0, 8, 1, W.TAG_A)   # misaligned pointer
    assert ei.value.code == -2
    with pytest.raises(B.LweError) as ei:
        ctx.sample_uniform(None, 0, 8, 1, W.TAG_A)
    assert ei.value.code == -3
    with pytest.raises(B.LweError) as ei:
        ctx.sample_uniform(out, 0, 8, 1, 0)                     # tag 0 is not a stream
    assert ei.value.code == -1
    assert ctx.launch_count() == n0
    with pytest.raises(B.LweError):
        B.Context(256, 512, 256, 70000, 4)                      # q > 65536
    with pytest.raises(B.LweError):
        B.Context(250, 512, 256, 65536, 4)                      # n % 8 != 0


@pytest.mark.parametrize("n,m,k,q,eta,inst0,n_inst", [
    (256, 512, 256, 65536, 4, 0, 1),          # C1
    (72, 200, 128, 65521, 8, 7, 3),           # prime q (rejection), k/8 = 16 bytes of mu
    (8, 8, 8, 17, 1, 1 << 20, 5),             # 1-byte mu rows, 8-byte R rows (unaligned row stores)
    (1024, 2048, 256, 65536, 4, 31, 4),       # C2 x 4 instances
    (64, 136, 40, 3329, 3, 2, 2),             # k not a multiple of 16: ragged last chunk of every object
])
def test_sample_kem_equals_the_four_samplers_and_the_oracle(H, n, m, k, q, eta, inst0, n_inst):
    """lwe_sample_kem draws s, e, R, mu of n_inst instances in one launch: the same bytes as the four single-object
    samplers, i.e. as the oracle's O4 / O5 / O6 on tags S, E, R, MU."""
    seed = 99
    with H.B.Context(n, m, k, q, eta, n_inst) as c:
        s, e = H.dev_empty_u16(n_inst, n), H.dev_empty_u16(n_inst, m)
        R, mu = H.dev_empty_u8(n_inst, m * k // 8), H.dev_empty_u8(n_inst, k // 8)
        for t in (s, e, R, mu):
            t.fill_(0x5A)
        c.sample_kem(s, e, R, mu, seed, inst0, n_inst)
        gs, ge, gR, gmu = H.host_u16(s), H.host_u16(e), H.host_u8(R), H.host_u8(mu)
    for t in range(n_inst):
        assert np.array_equal(gs[t], O.sample_uniform(0, n, seed, O.TAG_S, inst0 + t, q)), ("s", t)
        assert np.array_equal(ge[t], O.sample_cbd(0, m, seed, O.TAG_E, inst0 + t, q, eta)), ("e", t)
        assert np.array_equal(gR[t], O.sample_bits(0, m * k, seed, O.TAG_R, inst0 + t)), ("R", t)
        assert np.array_equal(gmu[t], O.sample_bits(0, k, seed, O.TAG_MU, inst0 + t)), ("mu", t)
