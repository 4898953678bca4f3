"""GPU parity, a3-a6: keygen (stored and regenerated A), encaps (tcgen05 GEMM and
CUDA-core path), decaps -- bit-exact against the oracle on the same seeded inputs,
through the C ABI.  Sizes span several tiles and ragged tails; full configs are
checked on sampled rows plus invariants that hold at any size."""
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


# ---------------------------------------------------------------- keygen

KEYGEN_SHAPES = [  # (m, n, q, batch)
    (512, 256, 65536, 1), (2048, 1024, 65536, 1), (264, 4096, 65521, 1), (136, 4104, 65521, 2),
    (1000, 40, 65521, 3), (8, 8, 17, 1), (304, 8192, 65536, 2), (96, 16392, 65521, 1), (520, 2056, 3329, 1),
    (304, 2088, 65536, 1), (3000, 2600, 12289, 1),      # rows that end inside a lane batch; more rows than warps in flight
]


@pytest.mark.parametrize("m,n,q,batch", KEYGEN_SHAPES)
def test_keygen_stored_matches_oracle(H, m, n, q, batch):
    A = W.random_u16((m, n), q, 1)
    s = W.random_u16((batch, n), q, 2)
    e = W.random_u16((batch, m), q, 3)
    with B().Context(n, m, 256, q, 4, batch) as c:
        b = H.dev_empty_u16(batch, m)
        c.keygen(H.dev(A), 0, H.dev(s), H.dev(e), b, batch)
        got = H.host_u16(b)
    for t in range(batch):
        assert np.array_equal(got[t], O.keygen(A, s[t], e[t], q)), (m, n, q, t)


KEYGEN_TC_SHAPES = [  # (m, n, q, batch): forced tcgen05 skinny GEMM (reads A once for the whole batch)
    (512, 256, 65536, 1), (512, 256, 65536, 4), (264, 4096, 65521, 5), (136, 4104, 65521, 2), (1000, 40, 65521, 3),
    (256, 20000, 65521, 9), (256, 512, 32768, 40), (136, 264, 65536, 128),
    (8, 8, 17, 1), (2048, 1024, 65536, 32), (640, 520, 3329, 33), (384, 1024, 65521, 64), (16384, 8192, 65536, 32),
]


@pytest.mark.parametrize("m,n,q,batch", KEYGEN_TC_SHAPES)
def test_keygen_tensor_core_batched_matches_oracle_and_gemv(H, m, n, q, batch):
    A = W.random_u16((m, n), q, 11)
    s = W.random_u16((batch, n), q, 12)
    e = W.random_u16((batch, m), q, 13)
    with B().Context(n, m, 256, q, 4, batch) as c:
        dA, ds, de = H.dev(A), H.dev(s), H.dev(e)
        b_tc, b_gemv = H.dev_empty_u16(batch, m), H.dev_empty_u16(batch, m)
        b_tc.fill_(-1)
        c.set_option(B().OPT_KEYGEN_PATH, 2)
        c.keygen(dA, 0, ds, de, b_tc, batch)
        c.set_option(B().OPT_KEYGEN_PATH, 1)
        c.keygen(dA, 0, ds, de, b_gemv, batch)
        g_tc, g_gemv = H.host_u16(b_tc), H.host_u16(b_gemv)
    assert np.array_equal(g_tc, g_gemv)
    check = range(batch) if m * n <= (1 << 22) else (0, batch // 2, batch - 1)   # the oracle is slow: sample instances
    for t in check:
        assert np.array_equal(g_tc[t], O.keygen(A, s[t], e[t], q)), (m, n, q, t)


def test_keygen_tensor_core_extreme_values(H):
    # every byte product and every plane accumulator at its maximum: q = 65536 runs 2 operand columns per
    # instance and lets the s32 accumulators wrap (exact mod 2^16) at n = 32768, the path's limit; q = 65521 runs
    # 3 columns up to n = 16384 (the merged 2^8 accumulator just below 2^31) and 4 columns above
    for q, n in ((65536, 32768), (65521, 32768), (65521, 16384), (65536, 16384)):
        m, batch = 128, 2
        A = np.full((m, n), 0xFFFF if q == 65536 else q - 1, np.uint16)
        s = np.full((batch, n), 0xFFFF if q == 65536 else q - 1, np.uint16)
        e = np.full((batch, m), q - 1, np.uint16)
        with B().Context(n, m, 256, q, 4, batch) as c:
            b = H.dev_empty_u16(batch, m)
            c.set_option(B().OPT_KEYGEN_PATH, 2)
            c.keygen(H.dev(A), 0, H.dev(s), H.dev(e), b, batch)
            a0 = int(A[0, 0])
            assert np.all(H.host_u16(b) == (n * a0 * a0 + (q - 1)) % q)


def test_keygen_extreme_values(H):
    # every product and every partial sum at its maximum (P9)
    for q in (65536, 65521):
        m, n = 64, 32768
        A = np.full((m, n), q - 1, np.uint16)
        s = np.full((1, n), q - 1, np.uint16)
        e = np.full((1, m), q - 1, np.uint16)
        with B().Context(n, m, 256, q, 4, 1) as c:
            b = H.dev_empty_u16(1, m)
            c.keygen(H.dev(A), 0, H.dev(s), H.dev(e), b, 1)
            assert np.all(H.host_u16(b) == (n * (q - 1) * (q - 1) + (q - 1)) % q)


@pytest.mark.parametrize("m,n,q,seed", [(512, 256, 65536, 1), (264, 4096, 65521, 3), (72, 1032, 40000, 9),
                                         (2048, 1024, 65536, 2)])
def test_keygen_regenerated_A_equals_stored_and_oracle(H, m, n, q, seed):
    # P11: A never stored; must equal the oracle's A drawn from the same seed
    A = O.sample_uniform(0, m * n, seed, O.TAG_A, 0, q).reshape(m, n)
    s = W.random_u16((2, n), q, 5)
    e = W.random_u16((2, m), q, 6)
    with B().Context(n, m, 256, q, 4, 2) as c:
        b1, b2 = H.dev_empty_u16(2, m), H.dev_empty_u16(2, m)
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, seed, W.TAG_A)
        assert np.array_equal(H.host_u16(dA), A)
        c.keygen(dA, 0, H.dev(s), H.dev(e), b1, 2)
        c.keygen(None, seed, H.dev(s), H.dev(e), b2, 2)
        g1, g2 = H.host_u16(b1), H.host_u16(b2)
    assert np.array_equal(g1, g2)
    for t in range(2):
        assert np.array_equal(g2[t], O.keygen(A, s[t], e[t], q))


# ---------------------------------------------------------------- encaps

ENCAPS_SHAPES = [  # (m, n, k, q, batch)
    (512, 256, 256, 65536, 1),        # C1
    (640, 192, 256, 65521, 2),        # several K blocks, 3 M tiles, prime q
    (200, 72, 256, 65521, 3),         # ragged K tail (200 = 128 + 72), ragged M tile (144 bytes)
    (136, 64, 128, 65536, 3),         # k = 128: N tile straddles instances, ragged N tail (384 cols)
    (128, 64, 16, 17, 2),             # 32 columns in total
    (2048, 1024, 256, 65536, 1),      # C2
    (1160, 456, 256, 65521, 5),       # 10 K blocks (> ring depth) with a tail, 4 pair tiles (last ragged), 5 N tiles
    (384, 1280, 256, 65536, 2),       # 10 pair tiles x 2: more tiles than a wave of small grids, both accumulators reused
    (264, 136, 512, 65521, 2),        # k = 512: two N tiles per instance
    (136, 72, 384, 65536, 3),         # k = 384: N tiles straddle instances (half tiles do not); 12 words of bits per row
    (520, 64, 64, 3329, 5),           # k = 64: no bit operand (k % 128 != 0), 320 columns
    (128, 8, 2048, 65536, 1),         # the largest k the ABI takes; a single, mostly empty M tile
]


def run_encaps(H, path, m, n, k, q, batch, A, b, Rbits, mubits):
    with B().Context(n, m, k, q, 4, batch) as c:
        set_encaps_path(c, path)
        U, v = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k)
        U.fill_(-1)
        c.encaps(H.dev(A), 0, H.dev(b), H.dev(Rbits), H.dev(mubits), U, v, batch)
        return H.host_u16(U), H.host_u16(v)


# 3 = CTA-pair tcgen05 GEMM (B operand expanded from R's packed bits inside the kernel where k % 128 == 0, v computed by
# spare warps of the same kernel where k = 32 * 2^j), 103 = the same with v from the separate pass over R,
# 13 = the pair kernel reading the u8 operand expanded into the workspace, 2 = single-CTA tcgen05, 1 = CUDA cores
ENCAPS_PATHS = dict(argvalues=[3, 103, 13, 2, 1],
                    ids=["tcgen05_pair", "tcgen05_pair_separate_v", "tcgen05_pair_expandedR", "tcgen05", "simt"])


def set_encaps_path(c, path):
    c.set_option(B().OPT_ENCAPS_PATH, path % 10)
    c.set_option(B().OPT_R_OPERAND, (path // 10) % 10)
    c.set_option(B().OPT_V_PATH, path // 100)


@pytest.mark.parametrize("path", **ENCAPS_PATHS)
@pytest.mark.parametrize("m,n,k,q,batch", ENCAPS_SHAPES)
def test_encaps_matches_oracle(H, path, m, n, k, q, batch):
    A = W.random_u16((m, n), q, 21)
    b = W.random_u16((batch, m), q, 22)
    Rbits = W.random_bytes(batch * m * k // 8, 23).reshape(batch, -1)
    mubits = W.random_bytes(batch * k // 8, 24).reshape(batch, -1)
    U, v = run_encaps(H, path, m, n, k, q, batch, A, b, Rbits, mubits)
    for t in range(batch):
        Uo, vo = O.encaps(A, b[t], Rbits[t], mubits[t], k, q)
        assert np.array_equal(v[t], vo), ("v", t)
        bad = np.argwhere(U[t] != Uo)
        assert bad.size == 0, (f"U mismatch inst {t}: {len(bad)} entries, first {bad[:5].tolist()}, "
                               f"got {U[t][tuple(bad[0])]} want {Uo[tuple(bad[0])]}")


@pytest.mark.parametrize("path", **ENCAPS_PATHS)
def test_encaps_extreme_accumulators(H, path):
    # P9: A = q-1 (or 65535), R = all ones, m = 65536 -> both byte-plane accumulators and the
    # recombined 32-bit value hit their bounds exactly
    for q in (65536, 65521):
        m, n, k = 65536, 64, 256
        A = np.full((m, n), q - 1, np.uint16)
        b = np.full((1, m), q - 1, np.uint16)
        Rbits = np.full((1, m * k // 8), 0xFF, np.uint8)
        mubits = np.full((1, k // 8), 0xFF, np.uint8)
        U, v = run_encaps(H, path, m, n, k, q, 1, A, b, Rbits, mubits)
        assert np.all(U == (m * (q - 1)) % q)
        assert np.all(v == (m * (q - 1) + q // 2) % q)


@pytest.mark.parametrize("path", **ENCAPS_PATHS)
def test_encaps_more_than_65536_rows_worst_case(H, path):
    """m = 131072 > 65536: the contraction runs in passes of 65536 rows whose residues are added mod q; with
    A = q-1 and R = all ones every 32-bit partial sum (byte planes, recombined value, the column sums of v) sits at
    its bound in both passes.  A wrap anywhere changes the result."""
    for q in (65536, 65521):
        m, n, k = 131072, 64, 256
        A = np.full((m, n), q - 1, np.uint16)
        b = np.full((2, m), q - 1, np.uint16)
        Rbits = np.full((2, m * k // 8), 0xFF, np.uint8)
        Rbits[1, : (m // 2) * k // 8 : 2] = 0x55           # second instance: a mixed pattern in the first pass
        mubits = np.full((2, k // 8), 0xFF, np.uint8)
        U, v = run_encaps(H, path, m, n, k, q, 2, A, b, Rbits, mubits)
        assert np.all(U[0] == (m * (q - 1)) % q)
        assert np.all(v[0] == (m * (q - 1) + q // 2) % q)
        ones = np.unpackbits(Rbits[1], bitorder="little").reshape(m, k).sum(axis=0).astype(np.int64)
        assert np.array_equal(U[1], np.broadcast_to((ones * (q - 1)) % q, (n, k)))
        assert np.array_equal(v[1], (ones * (q - 1) + q // 2) % q)


@pytest.mark.parametrize("path", **ENCAPS_PATHS)
def test_encaps_regenerated_A_more_than_65536_rows(H, path):
    """d_A = NULL with m = 131072 and a small n: the row panel the context could hold (256 MiB / 2n) is far more than
    65536 rows, but one tensor-core pass may not be (a byte-plane sum over more rows, recombined as lo + (hi << 8),
    leaves 32 bits for a prime modulus).  R = all ones, so every U[j][c] is the column sum of the regenerated A: with a
    uniform A the recombined value of a 131072-row pass is ~2^32 and wraps in about half the columns.  Expected values
    from the ORACLE's own draw of A."""
    m, n, k, q, seed = 131072, 64, 256, 65521, 77
    A = O.sample_uniform(0, m * n, seed, O.TAG_A, 0, q).reshape(m, n)
    b = W.random_u16((1, m), q, 22)
    Rbits = np.full((1, m * k // 8), 0xFF, np.uint8)
    mubits = np.zeros((1, k // 8), np.uint8)
    with B().Context(n, m, k, q, 4, 1) as c:
        set_encaps_path(c, path)
        c.set_option(B().OPT_REGEN_PATH, 1)              # row panels through the GEMM (the fused kernel is bounded by m <= 65536 itself)
        U, v = H.dev_empty_u16(1, n, k), H.dev_empty_u16(1, k)
        U.fill_(-1)
        c.encaps(None, seed, H.dev(b), H.dev(Rbits), H.dev(mubits), U, v, 1)
        U, v = H.host_u16(U), H.host_u16(v)
    colsum = (A.astype(np.uint64).sum(axis=0) % q).astype(np.uint16)
    assert np.array_equal(U[0], np.broadcast_to(colsum[:, None], (n, k)))
    assert np.all(v[0] == int(b[0].astype(np.uint64).sum() % q))


@pytest.mark.parametrize("path", [3, 2], ids=["tcgen05_pair", "tcgen05"])
def test_encaps_one_hot_R_picks_a_row_of_A(H, path):
    m, n, k, q = 256, 128, 256, 65521
    A = W.random_u16((m, n), q, 31)
    b = W.random_u16((1, m), q, 32)
    R = np.zeros((m, k), np.uint8)
    R[77, 200] = 1
    R[5, 0] = 1
    Rbits = np.packbits(R.ravel(), bitorder="little")[None, :]
    mubits = np.zeros((1, k // 8), np.uint8)
    U, v = run_encaps(H, path, m, n, k, q, 1, A, b, Rbits, mubits)
    assert np.array_equal(U[0][:, 200], A[77]) and np.array_equal(U[0][:, 0], A[5])
    assert int(v[0][200]) == int(b[0][77]) and int(v[0][0]) == int(b[0][5])
    U[0][:, 200] = 0
    U[0][:, 0] = 0
    assert not U.any()


@pytest.mark.parametrize("path", **ENCAPS_PATHS)
@pytest.mark.parametrize("m,n,k,q,batch,seed,panel", [
    (512, 256, 256, 65536, 1, 1, 0),        # C1: a single panel (default panel >= m)
    (512, 256, 256, 65536, 2, 1, 128),      # 4 full panels, accumulate across them
    (1160, 456, 256, 65521, 3, 3, 384),     # prime q (rejection sampling inside the panels), ragged last panel (8 rows)
    (200, 72, 128, 40000, 3, 9, 72),        # panels that are not a multiple of the K block, ragged tail (56 rows)
    (2048, 1024, 256, 65536, 1, 2, 1024),   # C2 in two panels
])
def test_encaps_regenerated_A_equals_stored_and_oracle(H, path, m, n, k, q, batch, seed, panel):
    """BJ configs[4] / S8(c) P11: lwe_encaps(d_A = NULL) regenerates A from its seed one row panel at a time and
    accumulates U over the panels; the result equals the stored-A path and the oracle (whose A is its own draw
    from the same seed) bit for bit, whatever the panel height."""
    A = O.sample_uniform(0, m * n, seed, O.TAG_A, 0, q).reshape(m, n)
    b = W.random_u16((batch, m), q, 22)
    Rbits = W.random_bytes(batch * m * k // 8, 23).reshape(batch, -1)
    mubits = W.random_bytes(batch * k // 8, 24).reshape(batch, -1)
    with B().Context(n, m, k, q, 4, batch) as c:
        set_encaps_path(c, path)
        c.set_option(B().OPT_REGEN_PATH, 1)                    # row panels (the fused kernel has its own test)
        c.set_option(B().OPT_PANEL_ROWS, panel)
        U, v = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k)
        U.fill_(-1)
        c.encaps(None, seed, H.dev(b), H.dev(Rbits), H.dev(mubits), U, v, batch)
        Ug, vg = H.host_u16(U), H.host_u16(v)
    Us, vs = run_encaps(H, path, m, n, k, q, batch, A, b, Rbits, mubits)
    assert np.array_equal(Ug, Us) and np.array_equal(vg, vs)
    for t in range(batch):
        Uo, vo = O.encaps(A, b[t], Rbits[t], mubits[t], k, q)
        assert np.array_equal(vg[t], vo), ("v", t)
        assert np.array_equal(Ug[t], Uo), ("U", t)


@pytest.mark.parametrize("m,n,k,q,seed", [
    (512, 256, 256, 65536, 1),           # C1: 4 tiles, one K range each
    (2048, 1024, 256, 65536, 2),         # C2: 16 tiles x several K ranges combined under the tile locks
    (1160, 456, 256, 65521, 3),          # prime q (rejection inside the generator), n % 64 != 0, ragged K tail
    (200, 72, 128, 40000, 9),            # k < 256 (second R box out of range)
    (4104, 8, 16, 12289, 5),             # one tile, mostly empty; many K ranges
    (12288, 9472, 256, 65536, 4),        # 148 tiles = exactly one wave of CTAs; two K ranges per tile
])
def test_encaps_fused_regenerated_A_matches_oracle(H, m, n, k, q, seed):
    """S8(f) N4: lwe_encaps(d_A = NULL) for one instance generates the A tiles inside the GEMM's producer (A never in
    HBM).  Equals the oracle, whose A is its own draw from the same seed, bit for bit; run twice on one context (the
    per-tile locks and counters reset themselves) and against the row-panel path."""
    b = W.random_u16((1, m), q, 22)
    Rbits = W.random_bytes(m * k // 8, 23).reshape(1, -1)
    mubits = W.random_bytes(k // 8, 24).reshape(1, -1)
    with B().Context(n, m, k, q, 4, 1) as c:
        c.set_option(B().OPT_REGEN_PATH, 2)
        U, v = H.dev_empty_u16(1, n, k), H.dev_empty_u16(1, k)
        got = []
        for _ in range(2):
            U.fill_(-1)
            c.profile_reset()
            c.set_option(B().OPT_PROFILE, 1)
            c.encaps(None, seed, H.dev(b), H.dev(Rbits), H.dev(mubits), U, v, 1)
            got.append((H.host_u16(U).copy(), H.host_u16(v).copy()))
            assert c.profile_read()["encaps_regen_tc"][1] == 1, "the fused kernel did not run"
        c.set_option(B().OPT_PROFILE, 0)
        c.set_option(B().OPT_REGEN_PATH, 1)
        U.fill_(-1)
        c.encaps(None, seed, H.dev(b), H.dev(Rbits), H.dev(mubits), U, v, 1)
        Up = H.host_u16(U).copy()
    if m * n <= 1 << 22:
        A = O.sample_uniform(0, m * n, seed, O.TAG_A, 0, q).reshape(m, n)
        Uo, vo = O.encaps(A, b[0], Rbits[0], mubits[0], k, q)
    else:                                                       # sampled rows of U (columns of A by counter index)
        rows = np.unique(np.concatenate([np.arange(0, 70), np.arange(n - 70, n), np.arange(63, n, 997)])).astype(np.uint32)
        cols = np.stack([O.sample_uniform_strided(int(j), n, m, seed, O.TAG_A, 0, q) for j in rows], axis=1)
        Usub, vo = O.encaps(cols, b[0], Rbits[0], mubits[0], k, q)
        Uo = None
    for Ug, vg in got:
        assert np.array_equal(vg[0], vo)
        if Uo is not None:
            assert np.array_equal(Ug[0], Uo)
        else:
            assert np.array_equal(Ug[0][rows], Usub)
    assert np.array_equal(got[0][0], Up), "fused vs row-panel path"


# ---------------------------------------------------------------- decaps

@pytest.mark.parametrize("n,k,q,batch", [(256, 256, 65536, 1), (1000, 256, 65521, 3), (64, 8, 17, 2),
                                          (4096, 128, 65521, 2), (8192, 256, 65536, 4), (136, 512, 65521, 2),
                                          (72, 384, 65536, 3), (8, 2048, 65536, 1),
                                          (520, 64, 4096, 3), (8192, 256, 2, 2),      # small powers of two: the u32 wrap-around sums
                                          (16384, 256, 65521, 2)])                    # u64 sums, many rows per thread
def test_decaps_matches_oracle(H, n, k, q, batch):
    U = W.random_u16((batch, n, k), q, 41)
    v = W.random_u16((batch, k), q, 42)
    s = W.random_u16((batch, n), q, 43)
    with B().Context(n, 8, k, q, 4, batch) as c:
        out = H.dev_empty_u8(batch, k // 8)
        for _ in range(2):                               # second call: workspace was left clean
            out.fill_(0xEE)
            c.decaps(H.dev(U), H.dev(v), H.dev(s), out, batch)
            got = H.host_u8(out)
            for t in range(batch):
                assert np.array_equal(got[t], O.decaps(U[t], v[t], s[t], q)), (n, k, q, t)


def test_decaps_rounding_boundaries(H):
    # U = 0 so d = v: sweep v over the decision boundaries (P10)
    for q in (65536, 65521):
        k, n = 256, 8
        edges = [0, 1, q // 4 - 1, q // 4, q // 4 + 1, q // 2, 3 * q // 4 - 1, 3 * q // 4, 3 * q // 4 + 1, q - 1]
        v = np.array([(edges * 26)[:k]], np.uint16)
        U = np.zeros((1, n, k), np.uint16)
        s = W.random_u16((1, n), q, 1)
        with B().Context(n, 8, k, q, 4, 1) as c:
            out = H.dev_empty_u8(1, k // 8)
            c.decaps(H.dev(U), H.dev(v), H.dev(s), out, 1)
            got = H.unpack_bits(H.host_u8(out)[0], k)
        want = np.array([1 if (4 * int(d) >= q and 4 * int(d) < 3 * q) else 0 for d in v[0]])
        assert np.array_equal(got, want)


@pytest.mark.parametrize("q", [65521, 40000, 12289, 3329])
def test_decaps_u64_sum_reduction_at_its_edges(H, q):
    """The 64-bit column sum sum_j U[j][c] s[j] is reduced mod q without a 64-bit remainder ((hi mod q)(2^32 mod q) +
    lo, Barrett steps).  Columns are built so that the exact sum S = hi 2^32 + lo hits the edges of every
    step (hi, lo in {0, 1, q-1, q, q+1, 2q-1, ..., 2^32-1}); each S is used by TWO columns whose v puts d exactly on
    the two sides of the decision boundary q/4, so an error of even 1 in S mod q flips one of the two bits."""
    k, nmax = 256, 200000
    top = (q - 1) * (q - 1)
    his = [h for h in (0, 1, 2, q - 2, q - 1, q, q + 1, 2 * q - 1, 2 * q, 3 * q - 1, 3 * q + 1)
           if (h + 1) << 32 <= (nmax - 8) * top]
    los = [0, 1, q - 1, q, q + 1, (1 << 32) - 1, (1 << 32) - q, (1 << 32) - q - 1, 1 << 31, 123456789]
    sums = [(h << 32) + lo for h in his for lo in los][: k // 2]
    n_top = max(S // top for S in sums)
    n = ((n_top + 2 + 7) // 8) * 8                         # rows [0, n_top): s = q-1; row n_top: s = q-1; row n_top+1: s = 1
    s = np.zeros((1, n), np.uint16)
    s[0, : n_top + 1] = q - 1
    s[0, n_top + 1] = 1
    U = np.zeros((1, n, k), np.uint16)
    v = np.zeros((1, k), np.uint16)
    lo_edge = -(-q // 4)                                   # smallest d with 4d >= q
    want = np.zeros(k, np.uint8)
    for x, S in enumerate(sums):
        a, rem = divmod(S, top)
        b_, rem2 = divmod(rem, q - 1)
        for c, d in ((2 * x, lo_edge), (2 * x + 1, lo_edge - 1)):
            U[0, :a, c] = q - 1
            U[0, n_top, c] = b_
            U[0, n_top + 1, c] = rem2
            v[0, c] = (S + d) % q                          # d = v - S mod q
            want[c] = 1 if 4 * d >= q and 4 * d < 3 * q else 0
        assert a * top + b_ * (q - 1) + rem2 == S and b_ < q and rem2 < q
    with B().Context(n, 8, k, q, 4, 1) as c:
        out = H.dev_empty_u8(1, k // 8)
        c.decaps(H.dev(U), H.dev(v), H.dev(s), out, 1)
        got = H.unpack_bits(H.host_u8(out)[0], k)
    assert np.array_equal(got[: 2 * len(sums)], want[: 2 * len(sums)])
    assert np.array_equal(got, H.unpack_bits(O.decaps(U[0], v[0], s[0], q), k))


# ---------------------------------------------------------------- whole path from seeds

def gpu_kem_from_seed(H, c, w, n, m, batch, dA):
    k = w.k
    s, e, b = H.dev_empty_u16(batch, n), H.dev_empty_u16(batch, m), H.dev_empty_u16(batch, m)
    Rbits, mubits = H.dev_empty_u8(batch, m * k // 8), H.dev_empty_u8(batch, k // 8)
    U, v, out = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k), H.dev_empty_u8(batch, k // 8)
    c.sample_uniform(s, 0, n, w.seed, W.TAG_S, 0, batch)
    c.sample_cbd(e, 0, m, w.seed, W.TAG_E, 0, batch)
    c.sample_bits(Rbits, 0, m * k, w.seed, W.TAG_R, 0, batch)
    c.sample_bits(mubits, 0, k, w.seed, W.TAG_MU, 0, batch)
    c.keygen(dA, 0, s, e, b, batch)
    c.encaps(dA, 0, b, Rbits, mubits, U, v, batch)
    c.decaps(U, v, s, out, batch)
    return dict(s=H.host_u16(s), e=H.host_u16(e), b=H.host_u16(b), Rbits=H.host_u8(Rbits),
                mubits=H.host_u8(mubits), U=H.host_u16(U), v=H.host_u16(v), out=H.host_u8(out))


@pytest.mark.parametrize("w,n,m,batch", [(W.C1, None, None, 1), (W.C2, None, None, 1), (W.C3, 512, 1024, 1),
                                          (W.C4, 256, 512, 4)])
def test_full_path_small_matches_oracle_everywhere(H, w, n, m, batch):
    n, m = n or w.n, m or w.m
    with H.make_ctx(w, n=n, m=m, max_batch=batch) as c:
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
        g = gpu_kem_from_seed(H, c, w, n, m, batch, dA)
        A = H.host_u16(dA)
    for t in range(batch):
        oi = H.OracleInstance(w, t, n, m)
        assert np.array_equal(A, oi.A)
        assert np.array_equal(g["s"][t], oi.s) and np.array_equal(g["e"][t], oi.e)
        assert np.array_equal(g["Rbits"][t], oi.Rbits) and np.array_equal(g["mubits"][t], oi.mubits)
        b = O.keygen(oi.A, oi.s, oi.e, w.q)
        assert np.array_equal(g["b"][t], b)
        U, v = O.encaps(oi.A, b, oi.Rbits, oi.mubits, w.k, w.q)
        assert np.array_equal(g["U"][t], U) and np.array_equal(g["v"][t], v)
        assert np.array_equal(g["out"][t], O.decaps(U, v, oi.s, w.q))
        assert np.array_equal(g["out"][t], oi.mubits)                # every bit recovered


@pytest.mark.parametrize("pdl", [0, 1], ids=["stream_order", "programmatic_dependent_launch"])
def test_full_path_back_to_back_batches_with_and_without_pdl(H, pdl):
    """LWE_OPT_PDL: with programmatic dependent launch a kernel's prologue overlaps its predecessor's tail and it waits on
    the device before touching data.  Six batches enqueued back to back on one stream REUSING the same buffers (so
    that every kernel overwrites what its predecessor still reads or wrote: write-after-read and read-after-write
    across every kernel boundary); the last batch and a checksum of all equal the oracle."""
    import torch
    w, n, m, batch = W.C3, 512, 1024, 3
    k, q = w.k, w.q
    with H.make_ctx(w, n=n, m=m, max_batch=batch) as c:
        c.set_option(B().OPT_PDL, pdl)
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
        s, e, b = H.dev_empty_u16(batch, n), H.dev_empty_u16(batch, m), H.dev_empty_u16(batch, m)
        Rb, mu = H.dev_empty_u8(batch, m * k // 8), H.dev_empty_u8(batch, k // 8)
        U, v, o = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k), H.dev_empty_u8(batch, k // 8)
        acc_v = torch.zeros(batch, k, dtype=torch.int64, device="cuda")
        bad = torch.zeros((), dtype=torch.int64, device="cuda")
        for i in range(6):
            c.sample_kem(s, e, Rb, mu, w.seed, 10 * i, batch)
            c.keygen(dA, 0, s, e, b, batch)
            c.encaps(dA, 0, b, Rb, mu, U, v, batch)
            c.decaps(U, v, s, o, batch)
            acc_v += v.to(torch.int64) & 0xFFFF
            bad += (o != mu).sum()
        torch.cuda.synchronize()
        assert int(bad.item()) == 0
        A, gb, gU, gv = H.host_u16(dA), H.host_u16(b), H.host_u16(U), H.host_u16(v)
        g_acc = acc_v.cpu().numpy()
    want_acc = np.zeros((batch, k), np.int64)
    for i in range(6):
        for t in range(batch):
            oi = H.OracleInstance(w, 10 * i + t, n, m, with_A=False)
            ob = O.keygen(A, oi.s, oi.e, q)
            ov = O.encaps_v(ob, oi.Rbits, oi.mubits, k, q)
            want_acc[t] += ov
            if i == 5:
                oU, ov2 = O.encaps(A, ob, oi.Rbits, oi.mubits, k, q)
                assert np.array_equal(gb[t], ob) and np.array_equal(gU[t], oU) and np.array_equal(gv[t], ov2)
    assert np.array_equal(g_acc, want_acc)


def test_two_contexts_of_different_shape_interleaved_on_two_streams(H):
    """Two contexts (different n, m, q, eta) driven alternately on two streams, several rounds: the per-kernel launch
    state the library caches (shared-memory attributes, occupancy, grids) must not leak between shapes, and the two
    streams' work may overlap on the device.  Every object of every round equals the oracle."""
    import torch
    cfgs = [(W.C1, 256, 512, 2), (W.C3, 512, 1024, 3)]
    st = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs, As, outs = [], [], [[], []]
    for w, n, m, batch in cfgs:
        c = H.make_ctx(w, n=n, m=m, max_batch=batch)
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
        ctxs.append(c); As.append(dA)
    torch.cuda.synchronize()
    try:
        for rnd in range(3):
            for x, (w, n, m, batch) in enumerate(cfgs):
                c, k = ctxs[x], w.k
                with torch.cuda.stream(st[x]):
                    s, e, b = H.dev_empty_u16(batch, n), H.dev_empty_u16(batch, m), H.dev_empty_u16(batch, m)
                    b2 = H.dev_empty_u16(1, m)
                    Rb, mu = H.dev_empty_u8(batch, m * k // 8), H.dev_empty_u8(batch, k // 8)
                    U, v, o = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k), H.dev_empty_u8(batch, k // 8)
                    c.sample_kem(s, e, Rb, mu, w.seed, 10 * rnd, batch)
                    c.keygen(As[x], 0, s, e, b, batch)
                    c.keygen(None, w.seed, s[:1], e[:1], b2, 1)             # A regenerated inside the GEMV
                    c.encaps(As[x], 0, b, Rb, mu, U, v, batch)
                    c.decaps(U, v, s, o, batch)
                    outs[x].append((rnd, s, e, b, b2, Rb, mu, U, v, o))
        torch.cuda.synchronize()
        for x, (w, n, m, batch) in enumerate(cfgs):
            A = H.host_u16(As[x])
            for rnd, s, e, b, b2, Rb, mu, U, v, o in outs[x]:
                gs, ge, gb, gb2 = H.host_u16(s), H.host_u16(e), H.host_u16(b), H.host_u16(b2)
                gR, gmu, gU, gv, go = H.host_u8(Rb), H.host_u8(mu), H.host_u16(U), H.host_u16(v), H.host_u8(o)
                for t in range(batch):
                    oi = H.OracleInstance(w, 10 * rnd + t, n, m, with_A=False)
                    assert np.array_equal(gs[t], oi.s) and np.array_equal(ge[t], oi.e)
                    assert np.array_equal(gR[t], oi.Rbits) and np.array_equal(gmu[t], oi.mubits)
                    ob = O.keygen(A, oi.s, oi.e, w.q)
                    assert np.array_equal(gb[t], ob)
                    if t == 0:
                        assert np.array_equal(gb2[0], ob)
                    oU, ov = O.encaps(A, ob, oi.Rbits, oi.mubits, w.k, w.q)
                    assert np.array_equal(gU[t], oU) and np.array_equal(gv[t], ov)
                    assert np.array_equal(go[t], oi.mubits)
    finally:
        for c in ctxs:
            c.close()


def test_pipelined_batches_on_two_contexts_and_streams_with_fo_decaps(H):
    """The two-context / two-stream pipeline bench.py reports as `pipelined_B32` (S8(f) N3): five consecutive
    batches alternate between two contexts on two streams (same shape, shared A), each batch = sample_kem -> keygen ->
    encaps -> decaps with the FO re-encryption check; kernels of neighbouring batches may overlap on the device.
    Every object of every batch equals the oracle, every honest ciphertext is accepted."""
    import torch
    w, n, m, batch, nb = W.C2, 384, 776, 3, 5
    k, q = w.k, w.q
    st = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs = [H.make_ctx(w, n=n, m=m, max_batch=batch) for _ in range(2)]
    dA = H.dev_empty_u16(m, n)
    ctxs[0].sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
    torch.cuda.synchronize()
    outs = []
    try:
        for i in range(nb):
            c = ctxs[i & 1]
            with torch.cuda.stream(st[i & 1]):
                s, e, b = H.dev_empty_u16(batch, n), H.dev_empty_u16(batch, m), H.dev_empty_u16(batch, m)
                Rb, mu = H.dev_empty_u8(batch, m * k // 8), H.dev_empty_u8(batch, k // 8)
                U, v = H.dev_empty_u16(batch, n, k), H.dev_empty_u16(batch, k)
                o, ok = H.dev_empty_u8(batch, k // 8), H.dev_empty_u8(batch)
                c.sample_kem(s, e, Rb, mu, w.seed, 100 * i, batch)
                c.keygen(dA, 0, s, e, b, batch)
                c.encaps(dA, 0, b, Rb, mu, U, v, batch)
                c.decaps_fo(dA, b, U, v, s, Rb, o, ok, batch)
                outs.append((i, s, e, b, Rb, mu, U, v, o, ok))
        torch.cuda.synchronize()
        A = H.host_u16(dA)
        assert np.array_equal(A, O.sample_uniform(0, m * n, w.seed, O.TAG_A, 0, q).reshape(m, n))
        for i, s, e, b, Rb, mu, U, v, o, ok in outs:
            gb, gU, gv, go, gok = H.host_u16(b), H.host_u16(U), H.host_u16(v), H.host_u8(o), H.host_u8(ok)
            for t in range(batch):
                oi = H.OracleInstance(w, 100 * i + t, n, m, with_A=False)
                ob = O.keygen(A, oi.s, oi.e, q)
                oU, ov = O.encaps(A, ob, oi.Rbits, oi.mubits, k, q)
                assert np.array_equal(gb[t], ob) and np.array_equal(gU[t], oU) and np.array_equal(gv[t], ov), (i, t)
                o_out, o_ok = O.decaps_fo(A, ob, oU, ov, oi.s, oi.Rbits, q)
                assert np.array_equal(go[t], o_out) and np.array_equal(go[t], oi.mubits) and int(gok[t]) == o_ok == 1, (i, t)
    finally:
        for c in ctxs:
            c.close()


def test_contexts_on_two_devices_in_one_process(H):
    """Launch state (shared-memory opt-ins, occupancy) is per context, i.e. per device: after a full pass on device
    0 the same calls on a context of device 1 must work and agree with the oracle.  Needs two GPUs."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("one GPU")
    w, n, m, batch = W.C3, 512, 1024, 2
    res = []
    for device in (0, 1, 0):
        with torch.cuda.device(device):
            c = B().Context(n, m, w.k, w.q, w.eta, batch, device)
            dA = torch.empty(m, n, dtype=torch.int16, device=f"cuda:{device}")
            c.sample_uniform(dA, 0, m * n, w.seed, W.TAG_A)
            dev_tensors = {}
            k = w.k
            mk = lambda *shape, dt=torch.int16: torch.empty(*shape, dtype=dt, device=f"cuda:{device}")  # noqa: E731
            s, e, b, b2 = mk(batch, n), mk(batch, m), mk(batch, m), mk(1, m)
            Rb, mu, o = mk(batch, m * k // 8, dt=torch.uint8), mk(batch, k // 8, dt=torch.uint8), mk(batch, k // 8, dt=torch.uint8)
            U, v, U2, v2 = mk(batch, n, k), mk(batch, k), mk(1, n, k), mk(1, k)
            c.sample_kem(s, e, Rb, mu, w.seed, 0, batch)
            c.keygen(dA, 0, s, e, b, batch)                       # tensor-core skinny GEMM
            c.keygen(None, w.seed, s[:1], e[:1], b2, 1)           # AES inside the GEMV (64 KB table: needs the opt-in)
            c.encaps(dA, 0, b, Rb, mu, U, v, batch)
            c.encaps(None, w.seed, b[:1], Rb[:1], mu[:1], U2, v2, 1)   # fused regenerated-A GEMM
            c.decaps(U, v, s, o, batch)
            torch.cuda.synchronize(device)
            res.append(dict(A=dA.cpu().numpy().view(np.uint16), b=b.cpu().numpy().view(np.uint16),
                            b2=b2.cpu().numpy().view(np.uint16), U=U.cpu().numpy().view(np.uint16),
                            U2=U2.cpu().numpy().view(np.uint16), v=v.cpu().numpy().view(np.uint16), o=o.cpu().numpy(),
                            mu=mu.cpu().numpy()))
            c.close()
            del dev_tensors
    oA = O.sample_uniform(0, m * n, w.seed, O.TAG_A, 0, w.q).reshape(m, n)
    for r in res:
        assert np.array_equal(r["A"], oA)
        for t in range(batch):
            oi = H.OracleInstance(w, t, n, m, with_A=False)
            ob = O.keygen(oA, oi.s, oi.e, w.q)
            oU, ov = O.encaps(oA, ob, oi.Rbits, oi.mubits, w.k, w.q)
            assert np.array_equal(r["b"][t], ob) and np.array_equal(r["U"][t], oU) and np.array_equal(r["v"][t], ov)
            assert np.array_equal(r["o"][t], oi.mubits)
            if t == 0:
                assert np.array_equal(r["b2"][0], ob) and np.array_equal(r["U2"][0], oU)


# ---------------------------------------------------------------- end to end with host buffers

@pytest.mark.parametrize("n,m,k,q,batch,regen", [
    (256, 512, 256, 65536, 1, False),      # one chunk
    (192, 384, 256, 65521, 9, False),      # chunks of 1, 1, 2, 4, 1 instances, prime q
    (128, 264, 256, 65536, 32, False),     # chunks of 1, 1, 2, 4, 8, 16 (the shape of bench.py's e2e leg), ragged K tail
    (64, 128, 256, 65536, 200, False),     # more instances than the chunk plan has doubling steps: the last chunk takes the rest
    (64, 128, 8, 17, 9, False),            # packed-bit rows narrower than 16 bytes: falls back to one chunk
    (192, 384, 256, 65536, 9, True),       # A regenerated from its seed for keygen and encaps (one chunk)
    (64, 128, 256, 65536, 20, True),       # regenerated A, two equal chunks
])
def test_kem_host_pipeline_matches_oracle(H, n, m, k, q, batch, regen):
    """lwe_kem_host (the e2e call bench.py times): pinned host buffers in, KeyGen once for the batch, then a chunked
    copy / Encrypt + Decrypt / copy-out pipeline inside, every output compared with the oracle per instance."""
    import torch
    seed = 11
    A = O.sample_uniform(0, m * n, seed, O.TAG_A, 0, q).reshape(m, n)
    s, e = W.random_u16((batch, n), q, 51), W.random_u16((batch, m), 5, 52)
    Rbits = W.random_bytes(batch * m * k // 8, 53).reshape(batch, -1)
    mubits = W.random_bytes(batch * k // 8, 54).reshape(batch, -1)

    def pinned(a):
        t = torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a).pin_memory()
        return t

    h_s, h_e, h_R, h_mu = pinned(s), pinned(e), pinned(Rbits), pinned(mubits)
    h_b = torch.zeros(batch, m, dtype=torch.int16).pin_memory()
    h_U = torch.zeros(batch, n, k, dtype=torch.int16).pin_memory()
    h_v = torch.zeros(batch, k, dtype=torch.int16).pin_memory()
    h_out = torch.zeros(batch, k // 8, dtype=torch.uint8).pin_memory()
    with B().Context(n, m, k, q, 4, batch) as c:
        dA = None if regen else H.dev(A)
        for _ in range(2):                                     # twice: the staging buffers are reused safely
            c.kem_host(dA, seed, h_s, h_e, h_R, h_mu, h_b, h_U, h_v, h_out, batch)
    gb, gU, gv, gout = (h_b.numpy().view(np.uint16), h_U.numpy().view(np.uint16), h_v.numpy().view(np.uint16),
                        h_out.numpy())
    for t in range(batch):
        b = O.keygen(A, s[t], e[t], q)
        U, v = O.encaps(A, b, Rbits[t], mubits[t], k, q)
        assert np.array_equal(gb[t], b), ("b", t)
        assert np.array_equal(gU[t], U) and np.array_equal(gv[t], v), ("U/v", t)
        assert np.array_equal(gout[t], O.decaps(U, v, s[t], q)), ("mu'", t)


def test_kem_host_rejects_misaligned_host_pointers(H):
    """include/lwe.h: every h_* pointer must be 16-byte aligned -> LWE_ERR_ALIGN before anything is enqueued"""
    import torch
    n, m, k, q = 64, 128, 256, 65536
    with B().Context(n, m, k, q, 4, 1) as c:
        dA = H.dev_empty_u16(m, n)
        c.sample_uniform(dA, 0, m * n, 1, W.TAG_A)
        pin = lambda *shape, dt=torch.int16: torch.zeros(*shape, dtype=dt).pin_memory()  # noqa: E731
        good = dict(h_s=pin(1, n), h_e=pin(1, m), h_R=pin(1, m * k // 8, dt=torch.uint8), h_mu=pin(1, k // 8, dt=torch.uint8),
                    h_b=pin(1, m), h_U=pin(1, n, k), h_v=pin(1, k), h_out=pin(1, k // 8, dt=torch.uint8))
        order = ["h_s", "h_e", "h_R", "h_mu", "h_b", "h_U", "h_v", "h_out"]
        c.kem_host(dA, 0, *[good[x] for x in order], 1)
        before = good["h_b"].clone()
        for bad in order:
            args = [good[x].data_ptr() + (2 if x == bad else 0) for x in order]
            with pytest.raises(B().LweError) as ei:
                c.kem_host(dA, 0, *args, 1)
            assert ei.value.code == -2, bad
        assert torch.equal(good["h_b"], before)


# ---------------------------------------------------------------- N3: decaps with the FO re-encryption check

@pytest.mark.parametrize("path", **ENCAPS_PATHS)
@pytest.mark.parametrize("n,m,k,q,batch", [(256, 512, 256, 65536, 1), (192, 392, 256, 65521, 6), (64, 136, 128, 65536, 5),
                                            (1280, 384, 256, 65521, 3)])
def test_decaps_fo_matches_oracle_honest_and_tampered(H, path, n, m, k, q, batch):
    """lwe_decaps_fo against the oracle's Alg. 5 (O11) instance by instance: honest ciphertexts, a tampered element of
    U in the first / last / a middle tile, a tampered v (small: m' unchanged; large: a bit of m' flips), wrong coins.
    U is compared inside the GEMM epilogue and is never written (checked)."""
    import torch
    A = W.random_u16((m, n), q, 61)
    s = W.random_u16((batch, n), q, 62)
    e = W.random_u16((batch, m), 5, 63)
    Rbits = W.random_bytes(batch * m * k // 8, 64).reshape(batch, -1)
    mubits = W.random_bytes(batch * k // 8, 65).reshape(batch, -1)
    b = np.stack([O.keygen(A, s[t], e[t], q) for t in range(batch)])
    U = np.empty((batch, n, k), np.uint16); v = np.empty((batch, k), np.uint16)
    for t in range(batch):
        U[t], v[t] = O.encaps(A, b[t], Rbits[t], mubits[t], k, q)
    R_in = Rbits.copy()
    # instance t gets tamper number t (0 = honest)
    tampers = ["honest", "U_first", "U_last", "v_small", "v_big", "coins"]
    for t in range(batch):
        kind = tampers[t % len(tampers)]
        if kind == "U_first": U[t, 0, 0] = (int(U[t, 0, 0]) + 1) % q
        if kind == "U_last": U[t, n - 1, k - 1] = (int(U[t, n - 1, k - 1]) + q - 1) % q
        if kind == "v_small": v[t, 3] = (int(v[t, 3]) + 1) % q
        if kind == "v_big": v[t, k - 1] = (int(v[t, k - 1]) + q // 2 + 3) % q
        if kind == "coins": R_in[t, 9] ^= 0x40
    with B().Context(n, m, k, q, 4, batch) as c:
        set_encaps_path(c, path)
        dU = H.dev(U)
        out, ok = H.dev_empty_u8(batch, k // 8), H.dev_empty_u8(batch)
        ok.fill_(7)
        c.decaps_fo(H.dev(A), H.dev(b), dU, H.dev(v), H.dev(s), H.dev(R_in), out, ok, batch)
        g_out, g_ok = H.host_u8(out), H.host_u8(ok)
        assert np.array_equal(H.host_u16(dU), U), "the received ciphertext must not be modified"
    for t in range(batch):
        o_out, o_ok = O.decaps_fo(A, b[t], U[t], v[t], s[t], R_in[t], q)
        assert int(g_ok[t]) == o_ok, (t, tampers[t % len(tampers)])
        assert np.array_equal(g_out[t], o_out), t
        assert o_ok == (1 if tampers[t % len(tampers)] == "honest" else 0)


def test_kem_host_chunk_plan_over_many_batch_sizes(H):
    """lwe_kem_host's chunk plan (1, 1, 2, 4, ... instances, the last chunk taking the rest) at every batch size from 1 to
    40 on one context: every output of every instance against the oracle (tiny shape, so that the sweep stays cheap)."""
    import torch
    n, m, k, q, seed, Bmax = 64, 128, 256, 65536, 5, 40
    A = O.sample_uniform(0, m * n, seed, O.TAG_A, 0, q).reshape(m, n)
    s, e = W.random_u16((Bmax, n), q, 61), W.random_u16((Bmax, m), 5, 62)
    Rbits = W.random_bytes(Bmax * m * k // 8, 63).reshape(Bmax, -1)
    mubits = W.random_bytes(Bmax * k // 8, 64).reshape(Bmax, -1)
    want = []
    for t in range(Bmax):
        b = O.keygen(A, s[t], e[t], q)
        U, v = O.encaps(A, b, Rbits[t], mubits[t], k, q)
        want.append((b, U, v, O.decaps(U, v, s[t], q)))

    def pinned(a):
        return torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a).pin_memory()

    h_s, h_e, h_R, h_mu = pinned(s), pinned(e), pinned(Rbits), pinned(mubits)
    with B().Context(n, m, k, q, 4, Bmax) as c:
        dA = H.dev(A)
        for batch in range(1, Bmax + 1):
            h_b = torch.zeros(batch, m, dtype=torch.int16).pin_memory()
            h_U = torch.zeros(batch, n, k, dtype=torch.int16).pin_memory()
            h_v = torch.zeros(batch, k, dtype=torch.int16).pin_memory()
            h_out = torch.zeros(batch, k // 8, dtype=torch.uint8).pin_memory()
            c.kem_host(dA, seed, h_s, h_e, h_R, h_mu, h_b, h_U, h_v, h_out, batch)
            gb, gU, gv, go = h_b.numpy().view(np.uint16), h_U.numpy().view(np.uint16), h_v.numpy().view(np.uint16), h_out.numpy()
            for t in range(batch):
                b, U, v, out = want[t]
                assert np.array_equal(gb[t], b) and np.array_equal(gU[t], U) and np.array_equal(gv[t], v), (batch, t)
                assert np.array_equal(go[t], out), (batch, t)
