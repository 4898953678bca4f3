"""Randomised-shape / perturbed-timing stress of the tensor-core kernels against the oracle (-m gpu).

compute-sanitizer is closed on this pool, so races in the warp-specialised kernels (TMA
producer, MMA issuer, bit expanders, epilogue; 4 barrier families across a CTA pair) can only show up as wrong
results or as the watchdog trap of mbar_wait.  This test goes looking for them: seeded random shapes (ragged K
tails, ragged M / N tiles, k in {128, 256, 384, 512}, three moduli), every GEMM path and operand mode, row panels of
random height for the regenerated-A path, each case run while a second stream keeps the SMs busy with an unrelated
kernel of the library (AES fill) so that CTA placement and barrier timing differ from run to run, and repeated
back to back on one context.  Every U and v is compared with the oracle element by element."""
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


def random_cases(seed, count):
    rng = np.random.default_rng(seed)
    cases = []
    for _ in range(count):
        k = int(rng.choice([128, 256, 256, 256, 384, 512]))
        q = int(rng.choice([65536, 65521, 12289]))
        batch = int(rng.integers(1, 6))
        n = 8 * int(rng.integers(1, 90))
        m = 8 * int(rng.integers(2, 260))
        # keep the oracle's share of the test to ~0.2 s per case
        while m * n * k * batch > 1.5e8:
            m = max(16, m // 2 // 8 * 8)
        path = int(rng.choice([3, 3, 13, 2]))
        panel = int(8 * rng.integers(1, max(2, m // 8)))            # rows per panel of the regenerated-A run
        cases.append((m, n, k, q, batch, path, panel, int(rng.integers(1, 1 << 30))))
    return cases


@pytest.mark.parametrize("chunk", range(6))
def test_random_shapes_all_paths_under_a_competing_stream(H, chunk):
    import torch
    Bd = B()
    side = torch.cuda.Stream()
    noise = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    with Bd.Context(64, 64, 256, 65536, 4, 1) as filler:
        for (m, n, k, q, batch, path, panel, seed) in random_cases(1000 + chunk, 8):
            A = O.sample_uniform(0, m * n, seed, O.TAG_A, 0, q).reshape(m, n)
            b = W.random_u16((batch, m), q, seed + 1)
            Rbits = W.random_bytes(batch * m * k // 8, seed + 2).reshape(batch, -1)
            mubits = W.random_bytes(batch * k // 8, seed + 3).reshape(batch, -1)
            want = [O.encaps(A, b[t], Rbits[t], mubits[t], k, q) for t in range(batch)]
            with Bd.Context(n, m, k, q, 4, batch) as c:
                c.set_option(Bd.OPT_ENCAPS_PATH, path % 10)
                c.set_option(Bd.OPT_R_OPERAND, path // 10)
                c.set_option(Bd.OPT_REGEN_PATH, 1)
                c.set_option(Bd.OPT_PANEL_ROWS, panel)
                dA, db, dR, dmu = H.dev(A), H.dev(b), H.dev(Rbits), H.dev(mubits)
                runs = []
                for rep in range(3):
                    U, v = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k)
                    U.fill_(-1)
                    with torch.cuda.stream(side):                  # unrelated work beside the GEMM, different each rep
                        filler.rng_fill(noise, (8 + 24 * rep) << 20, bytes(16), bytes(16), 0)
                    if rep == 2:
                        c.encaps(None, seed, db, dR, dmu, U, v, batch)     # regenerated A, random panel height
                    else:
                        c.encaps(dA, 0, db, dR, dmu, U, v, batch)
                    runs.append((U, v))
                torch.cuda.synchronize()
                for rep, (U, v) in enumerate(runs):
                    gU, gv = H.host_u16(U), H.host_u16(v)
                    for t in range(batch):
                        assert np.array_equal(gv[t], want[t][1]), (m, n, k, q, batch, path, panel, rep, t, "v")
                        assert np.array_equal(gU[t], want[t][0]), (m, n, k, q, batch, path, panel, rep, t, "U")


@pytest.mark.parametrize("chunk", range(4))
def test_random_shapes_streaming_kernels_back_to_back(H, chunk):
    """The register-pipelined stream kernels (stored-A GEMV, batched tensor-core keygen, decaps: loads of the next batch in
    flight while the current one is consumed, rows that end inside a batch, u32 / u64 column sums) on seeded random
    shapes and moduli, launched back to back on reused buffers with programmatic dependent launch on and off, beside a
    competing stream; every b and every recovered bit string against the oracle."""
    import torch
    Bd = B()
    rng = np.random.default_rng(4000 + chunk)
    side = torch.cuda.Stream()
    noise = torch.empty(32 << 20, dtype=torch.uint8, device="cuda")
    with Bd.Context(64, 64, 256, 65536, 4, 1) as filler:
        for _ in range(6):
            k = int(rng.choice([64, 128, 256, 256, 384, 512]))
            q = int(rng.choice([65536, 65521, 4096, 3329]))
            batch = int(rng.integers(1, 5))
            n = 8 * int(rng.integers(1, 400))
            m = 8 * int(rng.integers(1, 300))
            seed = int(rng.integers(1, 1 << 30))
            A = W.random_u16((m, n), q, seed)
            s, e = W.random_u16((batch, n), q, seed + 1), W.random_u16((batch, m), q, seed + 2)
            U, v = W.random_u16((batch, n, k), q, seed + 3), W.random_u16((batch, k), q, seed + 4)
            want_b = [O.keygen(A, s[t], e[t], q) for t in range(batch)]
            want_o = [O.decaps(U[t], v[t], s[t], q) for t in range(batch)]
            with Bd.Context(n, m, k, q, 4, batch) as c:
                dA, ds, de, dU, dv = H.dev(A), H.dev(s), H.dev(e), H.dev(U), H.dev(v)
                b1, b2 = H.dev_empty_u16(batch, m), H.dev_empty_u16(batch, m)
                out = H.dev_empty_u8(batch, k // 8)
                for pdl in (1, 0):
                    c.set_option(Bd.OPT_PDL, pdl)
                    with torch.cuda.stream(side):
                        filler.rng_fill(noise, 32 << 20, bytes(16), bytes(16), 0)
                    for rep in range(3):                             # back to back, outputs overwritten each time
                        b1.fill_(-1); b2.fill_(-1); out.fill_(0xEE)
                        c.set_option(Bd.OPT_KEYGEN_PATH, 1)
                        c.keygen(dA, 0, ds, de, b1, batch)           # one GEMV per instance
                        c.set_option(Bd.OPT_KEYGEN_PATH, 0)
                        c.keygen(dA, 0, ds, de, b2, batch)           # auto: the skinny tensor-core GEMM for batch >= 2
                        c.decaps(dU, dv, ds, out, batch)
                    torch.cuda.synchronize()
                    g1, g2, go = H.host_u16(b1), H.host_u16(b2), H.host_u8(out)
                    for t in range(batch):
                        assert np.array_equal(g1[t], want_b[t]), (m, n, k, q, batch, pdl, t, "gemv")
                        assert np.array_equal(g2[t], want_b[t]), (m, n, k, q, batch, pdl, t, "keygen auto")
                        assert np.array_equal(go[t], want_o[t]), (m, n, k, q, batch, pdl, t, "decaps")
