"""ctypes wrapper around liblwe_oracle.so (ORACLE -- test infrastructure).

Argument marshalling only: numpy arrays in, numpy arrays out.  All arithmetic
is in lwe_oracle.c.  Names follow SURVEY.md 8(c) (O1..O9).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

TAG_A, TAG_S, TAG_E, TAG_R, TAG_MU = 1, 2, 3, 4, 5
TAG_RG, TAG_E1, TAG_E2 = 6, 7, 8          # N2: Gaussian r, e1 and centred-uniform e2 of the paper's PKE
GAUSS_TAU = 12

__all__ = [
    "TAG_A", "TAG_S", "TAG_E", "TAG_R", "TAG_MU", "TAG_RG", "TAG_E1", "TAG_E2", "GAUSS_TAU",
    "aes128_encrypt_block", "ctr_bytes", "seed_key", "object_iv",
    "sample_uniform", "sample_uniform_strided", "sample_cbd", "sample_bits",
    "keygen", "encaps", "encaps_rows", "encaps_v", "decaps", "decaps_fo", "num_threads",
    "gauss_cdt", "gauss_from_word", "sample_gauss", "sample_cuniform", "encaps_pv",
    "cbd_from_word", "round_bit",
    "set_num_threads", "sample_uniform32", "sample_uniform32_strided", "sample_cbd_s8", "keygen_w", "encaps_pv_w", "decaps_w",
]

_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(str(_build.build()))
        u8p, u16p, u32p = C.POINTER(C.c_uint8), C.POINTER(C.c_uint16), C.POINTER(C.c_uint32)
        u32, u64, sz = C.c_uint32, C.c_uint64, C.c_size_t
        lib.orc_aes128_encrypt_block.argtypes = [u8p, u8p, u8p]
        lib.orc_ctr_bytes.argtypes = [u8p, u8p, u64, sz, u8p]
        lib.orc_seed_key.argtypes = [u64, u8p]
        lib.orc_object_iv.argtypes = [u32, u32, u32, u8p]
        lib.orc_sample_uniform.argtypes = [u16p, u64, u64, u64, u32, u32, u32]
        lib.orc_sample_uniform_strided.argtypes = [u16p, u64, u64, u64, u64, u32, u32, u32]
        lib.orc_sample_cbd.argtypes = [u16p, u64, u64, u64, u32, u32, u32, u32]
        lib.orc_sample_bits.argtypes = [u8p, u64, u64, u64, u32, u32]
        lib.orc_keygen.argtypes = [u16p, u16p, u16p, u16p, u32, u32, u32]
        lib.orc_encaps.argtypes = [u16p, u16p, u8p, u8p, u16p, u16p, u32, u32, u32, u32]
        lib.orc_encaps_rows.argtypes = [u16p, u8p, u32p, u32, u16p, u32, u32, u32, u32]
        lib.orc_encaps_v.argtypes = [u16p, u8p, u8p, u16p, u32, u32, u32]
        lib.orc_decaps.argtypes = [u16p, u16p, u16p, u8p, u16p, u32, u32, u32]
        lib.orc_decaps_fo.argtypes = [u16p, u16p, u16p, u16p, u16p, u8p, u8p, u32, u32, u32, u32]
        lib.orc_decaps_fo.restype = C.c_int
        s8p, dbl = C.POINTER(C.c_int8), C.c_double
        lib.orc_gauss_cdt.argtypes = [dbl, u32p]
        lib.orc_gauss_cdt.restype = None
        lib.orc_gauss_from_word.argtypes = [u32, u32p]
        lib.orc_gauss_from_word.restype = C.c_int
        lib.orc_sample_gauss.argtypes = [s8p, u16p, u64, u64, u64, u32, u32, dbl, u32]
        lib.orc_sample_gauss.restype = None
        lib.orc_sample_cuniform.argtypes = [s8p, u64, u64, u64, u32, u32, u32]
        lib.orc_sample_cuniform.restype = None
        lib.orc_encaps_pv.argtypes = [u16p, u16p, s8p, s8p, s8p, u8p, u16p, u16p, u32, u32, u32, u32]
        lib.orc_encaps_pv.restype = None
        lib.orc_num_threads.restype = C.c_int
        lib.orc_set_num_threads.argtypes = [C.c_int]
        lib.orc_set_num_threads.restype = C.c_int
        lib.orc_cbd_from_word.argtypes = [u32, u32, u32]
        lib.orc_cbd_from_word.restype = C.c_uint16
        lib.orc_round_bit.argtypes = [u32, u32]
        lib.orc_round_bit.restype = C.c_uint32
        for f in ("orc_aes128_encrypt_block", "orc_ctr_bytes", "orc_seed_key", "orc_object_iv",
                  "orc_sample_uniform", "orc_sample_uniform_strided", "orc_sample_cbd", "orc_sample_bits", "orc_keygen",
                  "orc_encaps", "orc_encaps_rows", "orc_encaps_v", "orc_decaps"):
            getattr(lib, f).restype = None
        lib.orc_sample_uniform32.argtypes = [u32p, u64, u64, u64, u32, u32, u32]
        lib.orc_sample_uniform32_strided.argtypes = [u32p, u64, u64, u64, u64, u32, u32, u32]
        lib.orc_sample_cbd_s8.argtypes = [s8p, u64, u64, u64, u32, u32, u32]
        lib.orc_keygen_w.argtypes = [u32p, s8p, s8p, u32p, u32, u32, u32]
        lib.orc_encaps_pv_w.argtypes = [u32p, u32p, s8p, s8p, s8p, u8p, u32p, u32p, u32, u32, u32, u32]
        lib.orc_decaps_w.argtypes = [u32p, u32p, s8p, u8p, u32p, u32, u32, u32]
        for f in ("orc_sample_uniform32", "orc_sample_uniform32_strided", "orc_sample_cbd_s8", "orc_keygen_w",
                  "orc_encaps_pv_w", "orc_decaps_w"):
            getattr(lib, f).restype = None
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _u8(x, n=None):
    a = np.ascontiguousarray(np.frombuffer(bytes(x), dtype=np.uint8) if isinstance(x, (bytes, bytearray)) else x,
                             dtype=np.uint8)
    if n is not None and a.size != n:
        raise ValueError(f"expected {n} bytes, got {a.size}")
    return a


def _u16(x):
    return np.ascontiguousarray(x, dtype=np.uint16)


def aes128_encrypt_block(key, block) -> bytes:
    k, b = _u8(key, 16), _u8(block, 16)
    out = np.zeros(16, np.uint8)
    _L().orc_aes128_encrypt_block(_p(k, C.c_uint8), _p(b, C.c_uint8), _p(out, C.c_uint8))
    return out.tobytes()


def ctr_bytes(key, iv, byte_offset: int, nbytes: int) -> np.ndarray:
    k, v = _u8(key, 16), _u8(iv, 16)
    out = np.zeros(nbytes, np.uint8)
    _L().orc_ctr_bytes(_p(k, C.c_uint8), _p(v, C.c_uint8), byte_offset, nbytes, _p(out, C.c_uint8))
    return out


def seed_key(seed: int) -> bytes:
    out = np.zeros(16, np.uint8)
    _L().orc_seed_key(seed, _p(out, C.c_uint8))
    return out.tobytes()


def object_iv(tag: int, attempt: int, inst: int) -> bytes:
    out = np.zeros(16, np.uint8)
    _L().orc_object_iv(tag, attempt, inst, _p(out, C.c_uint8))
    return out.tobytes()


def sample_uniform(first: int, count: int, seed: int, tag: int, inst: int, q: int) -> np.ndarray:
    out = np.zeros(count, np.uint16)
    _L().orc_sample_uniform(_p(out, C.c_uint16), first, count, seed, tag, inst, q)
    return out


def sample_uniform_strided(first: int, stride: int, count: int, seed: int, tag: int, inst: int, q: int) -> np.ndarray:
    out = np.zeros(count, np.uint16)
    _L().orc_sample_uniform_strided(_p(out, C.c_uint16), first, stride, count, seed, tag, inst, q)
    return out


def sample_cbd(first: int, count: int, seed: int, tag: int, inst: int, q: int, eta: int) -> np.ndarray:
    out = np.zeros(count, np.uint16)
    _L().orc_sample_cbd(_p(out, C.c_uint16), first, count, seed, tag, inst, q, eta)
    return out


def sample_bits(first_bit: int, nbits: int, seed: int, tag: int, inst: int) -> np.ndarray:
    out = np.zeros((nbits + 7) // 8, np.uint8)
    _L().orc_sample_bits(_p(out, C.c_uint8), first_bit, nbits, seed, tag, inst)
    return out


def keygen(A, s, e, q: int) -> np.ndarray:
    A, s, e = _u16(A), _u16(s), _u16(e)
    m, n = A.shape
    assert s.shape == (n,) and e.shape == (m,)
    b = np.zeros(m, np.uint16)
    _L().orc_keygen(_p(A, C.c_uint16), _p(s, C.c_uint16), _p(e, C.c_uint16), _p(b, C.c_uint16), m, n, q)
    return b


def encaps(A, b, Rbits, mubits, k: int, q: int):
    A, b, Rbits, mubits = _u16(A), _u16(b), _u8(Rbits), _u8(mubits)
    m, n = A.shape
    assert b.shape == (m,) and Rbits.size == m * k // 8 and mubits.size == k // 8
    U = np.zeros((n, k), np.uint16)
    v = np.zeros(k, np.uint16)
    _L().orc_encaps(_p(A, C.c_uint16), _p(b, C.c_uint16), _p(Rbits, C.c_uint8), _p(mubits, C.c_uint8),
                    _p(U, C.c_uint16), _p(v, C.c_uint16), m, n, k, q)
    return U, v


def encaps_rows(A, Rbits, rows, k: int, q: int) -> np.ndarray:
    A, Rbits = _u16(A), _u8(Rbits)
    rows = np.ascontiguousarray(rows, dtype=np.uint32)
    m, n = A.shape
    out = np.zeros((rows.size, k), np.uint16)
    _L().orc_encaps_rows(_p(A, C.c_uint16), _p(Rbits, C.c_uint8), _p(rows, C.c_uint32), rows.size,
                         _p(out, C.c_uint16), m, n, k, q)
    return out


def encaps_v(b, Rbits, mubits, k: int, q: int) -> np.ndarray:
    b, Rbits, mubits = _u16(b), _u8(Rbits), _u8(mubits)
    v = np.zeros(k, np.uint16)
    _L().orc_encaps_v(_p(b, C.c_uint16), _p(Rbits, C.c_uint8), _p(mubits, C.c_uint8), _p(v, C.c_uint16),
                      b.size, k, q)
    return v


def decaps(U, v, s, q: int, return_d: bool = False):
    U, v, s = _u16(U), _u16(v), _u16(s)
    n, k = U.shape
    assert v.shape == (k,) and s.shape == (n,)
    out = np.zeros(k // 8, np.uint8)
    d = np.zeros(k, np.uint16)
    _L().orc_decaps(_p(U, C.c_uint16), _p(v, C.c_uint16), _p(s, C.c_uint16), _p(out, C.c_uint8),
                    _p(d, C.c_uint16), n, k, q)
    return (out, d) if return_d else out


def decaps_fo(A, b, U, v, s, Rbits, q: int):
    """O11: (m' packed bits, verdict c' == c) of Alg. 5 lines 1, 2, 4"""
    A, b, U, v, s = _u16(A), _u16(b), _u16(U), _u16(v), _u16(s)
    m, n = A.shape
    n2, k = U.shape
    assert n2 == n and b.shape == (m,) and v.shape == (k,) and s.shape == (n,)
    Rbits = _u8(Rbits, m * k // 8)
    out = np.zeros(k // 8, np.uint8)
    ok = _L().orc_decaps_fo(_p(A, C.c_uint16), _p(b, C.c_uint16), _p(U, C.c_uint16), _p(v, C.c_uint16),
                            _p(s, C.c_uint16), _p(Rbits, C.c_uint8), _p(out, C.c_uint8), m, n, k, q)
    return out, int(ok)


def gauss_cdt(sigma: float) -> np.ndarray:
    """O12: the 24-entry 16-bit cumulative table of the rounded Gaussian"""
    cdt = np.zeros(2 * GAUSS_TAU, np.uint32)
    _L().orc_gauss_cdt(float(sigma), _p(cdt, C.c_uint32))
    return cdt


def gauss_from_word(w: int, cdt) -> int:
    cdt = np.ascontiguousarray(cdt, dtype=np.uint32)
    return int(_L().orc_gauss_from_word(int(w), _p(cdt, C.c_uint32)))


def sample_gauss(first: int, count: int, seed: int, tag: int, inst: int, sigma: float, q: int | None = None) -> np.ndarray:
    """O12: int8 samples (q is None) or their residues mod q as uint16"""
    if q is None:
        out = np.zeros(count, np.int8)
        _L().orc_sample_gauss(_p(out, C.c_int8), None, first, count, seed, tag, inst, float(sigma), 2)
    else:
        out = np.zeros(count, np.uint16)
        _L().orc_sample_gauss(None, _p(out, C.c_uint16), first, count, seed, tag, inst, float(sigma), q)
    return out


def sample_cuniform(first: int, count: int, seed: int, tag: int, inst: int, bound: int) -> np.ndarray:
    out = np.zeros(count, np.int8)
    _L().orc_sample_cuniform(_p(out, C.c_int8), first, count, seed, tag, inst, bound)
    return out


def encaps_pv(A, t, R, E1, e2, mubits, q: int):
    """O14: (U, v) of the paper's Encrypt for all k bits; R [m][k], E1 [n][k], e2 [k] int8"""
    A, t = _u16(A), _u16(t)
    m, n = A.shape
    R, E1, e2 = (np.ascontiguousarray(x, dtype=np.int8) for x in (R, E1, e2))
    k = e2.shape[0]
    assert R.shape == (m, k) and E1.shape == (n, k) and t.shape == (m,)
    mubits = _u8(mubits, k // 8)
    U, v = np.zeros((n, k), np.uint16), np.zeros(k, np.uint16)
    _L().orc_encaps_pv(_p(A, C.c_uint16), _p(t, C.c_uint16), _p(R, C.c_int8), _p(E1, C.c_int8), _p(e2, C.c_int8),
                       _p(mubits, C.c_uint8), _p(U, C.c_uint16), _p(v, C.c_uint16), m, n, k, q)
    return U, v


# ---- q > 65536 (Table 1 rows n >= 8192): uint32 residues, int8 small objects (readings S23-S25)

def _u32(x):
    return np.ascontiguousarray(x, dtype=np.uint32)


def _s8(x):
    return np.ascontiguousarray(x, dtype=np.int8)


def sample_uniform32(first: int, count: int, seed: int, tag: int, inst: int, q: int) -> np.ndarray:
    out = np.zeros(count, np.uint32)
    _L().orc_sample_uniform32(_p(out, C.c_uint32), first, count, seed, tag, inst, q)
    return out


def sample_uniform32_strided(first: int, stride: int, count: int, seed: int, tag: int, inst: int, q: int) -> np.ndarray:
    out = np.zeros(count, np.uint32)
    _L().orc_sample_uniform32_strided(_p(out, C.c_uint32), first, stride, count, seed, tag, inst, q)
    return out


def sample_cbd_s8(first: int, count: int, seed: int, tag: int, inst: int, eta: int) -> np.ndarray:
    out = np.zeros(count, np.int8)
    _L().orc_sample_cbd_s8(_p(out, C.c_int8), first, count, seed, tag, inst, eta)
    return out


def keygen_w(A, s, e, q: int) -> np.ndarray:
    """O7w: t = A s + e mod q; A uint32 [m][n], s int8 [n], e int8 [m]"""
    A, s, e = _u32(A), _s8(s), _s8(e)
    m, n = A.shape
    assert s.shape == (n,) and e.shape == (m,)
    t = np.zeros(m, np.uint32)
    _L().orc_keygen_w(_p(A, C.c_uint32), _p(s, C.c_int8), _p(e, C.c_int8), _p(t, C.c_uint32), m, n, q)
    return t


def encaps_pv_w(A, t, R, E1, e2, mubits, q: int):
    """O14w: (U, v) uint32; A uint32 [m][n], t uint32 [m], R [m][k], E1 [n][k], e2 [k] int8"""
    A, t = _u32(A), _u32(t)
    m, n = A.shape
    R, E1, e2 = _s8(R), _s8(E1), _s8(e2)
    k = e2.shape[0]
    assert R.shape == (m, k) and E1.shape == (n, k) and t.shape == (m,)
    mubits = _u8(mubits, k // 8)
    U, v = np.zeros((n, k), np.uint32), np.zeros(k, np.uint32)
    _L().orc_encaps_pv_w(_p(A, C.c_uint32), _p(t, C.c_uint32), _p(R, C.c_int8), _p(E1, C.c_int8), _p(e2, C.c_int8),
                         _p(mubits, C.c_uint8), _p(U, C.c_uint32), _p(v, C.c_uint32), m, n, k, q)
    return U, v


def decaps_w(U, v, s, q: int, return_d: bool = False):
    U, v, s = _u32(U), _u32(v), _s8(s)
    n, k = U.shape
    assert v.shape == (k,) and s.shape == (n,)
    out = np.zeros(k // 8, np.uint8)
    d = np.zeros(k, np.uint32)
    _L().orc_decaps_w(_p(U, C.c_uint32), _p(v, C.c_uint32), _p(s, C.c_int8), _p(out, C.c_uint8), _p(d, C.c_uint32), n, k, q)
    return (out, d) if return_d else out


def cbd_from_word(w: int, q: int, eta: int) -> int:
    return int(_L().orc_cbd_from_word(w, q, eta))


def round_bit(d: int, q: int) -> int:
    return int(_L().orc_round_bit(d, q))


def num_threads() -> int:
    return int(_L().orc_num_threads())


def set_num_threads(threads: int) -> int:
    """OpenMP threads of the loops from now on; returns the previous setting"""
    return int(_L().orc_set_num_threads(int(threads)))
