"""lwe_decaps_static: Decaps for callers that cannot allocate device memory.

Some users of this library are handed device buffers and a stream by a host framework and may not call cudaMalloc
themselves: a plug-in inside a serving process whose caching allocator already owns the whole GPU, a component under a
fixed memory plan, a latency-critical thread that must stay off the driver's allocation lock.  lwe_create is closed to
them (it sizes a workspace).  lwe_decaps_static takes no context and allocates nothing: its scratch is one fixed
`static __device__` array inside the library, shared by every call on the device, which keeps the last call's contents.

The checks here are therefore: the same bits as the existing lwe_decaps (integer work: bit-exact, the tolerance every
parity test of this repository uses) and as the oracle; on two calls in a row on the same stream, with different
inputs, so that anything the first call leaves in the shared array would corrupt the second; at the stated size limit;
and a clear refusal beyond it.  The file is named to be collected last (pytest -x stops at the first failure) and
passes both alone in a fresh process -- where its first call does the per-device address look-up -- and after the
other tests."""
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
    import paper_2606_01211_b200.binding as b
    return b


@pytest.mark.parametrize("n,k,q,batch", [(256, 256, 65536, 1), (1000, 256, 65521, 3), (64, 8, 17, 2),
                                          (8192, 256, 65536, 32), (136, 512, 65521, 2), (72, 384, 65536, 3),
                                          (8, 2048, 65536, 1), (4096, 256, 3329, 64)])
def test_decaps_static_equals_decaps_and_oracle_on_two_calls_in_a_row(H, n, k, q, batch):
    b = B()
    assert batch * k <= b.STATIC_MAX_COLS and batch <= b.STATIC_MAX_BATCH
    with b.Context(n, 8, k, q, 4, batch) as c:           # the existing path; only it needs a context
        for call in range(2):                            # second call: other inputs, the array still holds the first's sums
            U = W.random_u16((batch, n, k), q, 410 + call)
            v = W.random_u16((batch, k), q, 420 + call)
            s = W.random_u16((batch, n), q, 430 + call)
            dU, dv, ds = H.dev(U), H.dev(v), H.dev(s)
            ref, out = H.dev_empty_u8(batch, k // 8), H.dev_empty_u8(batch, k // 8)
            ref.fill_(0xEE)
            out.fill_(0x77)
            c.decaps(dU, dv, ds, ref, batch)
            b.decaps_static(n, k, q, dU, dv, ds, out, batch)
            want, got = H.host_u8(ref), H.host_u8(out)
            assert np.array_equal(got, want), (n, k, q, batch, call)
            for t in range(min(batch, 3)):
                assert np.array_equal(got[t], O.decaps(U[t], v[t], s[t], q)), (n, k, q, t, call)


def test_decaps_static_after_a_larger_call_sees_no_leftovers(H):
    """A big call fills the whole shared array; a small one right after it must not read any of that."""
    b = B()
    n, k, q = 512, 256, 65521
    for batch, seed in ((64, 1), (1, 2), (2, 3)):
        U = W.random_u16((batch, n, k), q, 500 + seed)
        v = W.random_u16((batch, k), q, 510 + seed)
        s = W.random_u16((batch, n), q, 520 + seed)
        out = H.dev_empty_u8(batch, k // 8)
        b.decaps_static(n, k, q, H.dev(U), H.dev(v), H.dev(s), out, batch)
        got = H.host_u8(out)
        for t in (0, batch - 1):
            assert np.array_equal(got[t], O.decaps(U[t], v[t], s[t], q)), (batch, t)


def test_decaps_static_refuses_what_the_fixed_array_cannot_hold(H):
    b = B()
    n, k, q = 64, 256, 65536
    out = H.dev_empty_u8(80, k // 8)
    out.fill_(0x5A)
    U, v, s = H.dev_empty_u16(80, n, k), H.dev_empty_u16(80, k), H.dev_empty_u16(80, n)
    for batch, kk in ((65, 256), (80, 256), (9, 2048)):  # too many instances; too many columns in total
        with pytest.raises(b.LweError) as ei:
            b.decaps_static(n, kk, q, U, v, s, out, batch)
        assert ei.value.code == -5, (batch, kk)          # LWE_ERR_UNSUPPORTED
    with pytest.raises(b.LweError) as ei:
        b.decaps_static(n, k, 65537, U, v, s, out, 1)    # not a uint16 modulus
    assert ei.value.code == -1
    with pytest.raises(b.LweError) as ei:
        b.decaps_static(n, k, q, None, v, s, out, 1)
    assert ei.value.code == -3
    assert (H.host_u8(out) == 0x5A).all()                # nothing was written by the refused calls
