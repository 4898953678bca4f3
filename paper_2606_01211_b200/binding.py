"""Thin ctypes face of liblwe_b200.so -- argument marshalling only.

Same names as include/lwe.h.  Every step of the path runs in the library's CUDA
kernels; PyTorch appears only as the owner of device memory and streams.  There is
no fallback: if the library is missing or the device is not sm_100, calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import torch

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "lib" / "liblwe_b200.so"

LWE_OK = 0
ERRORS = {-1: "LWE_ERR_PARAM", -2: "LWE_ERR_ALIGN", -3: "LWE_ERR_NULLPTR", -4: "LWE_ERR_CUDA",
          -5: "LWE_ERR_UNSUPPORTED"}
TAG_A, TAG_S, TAG_E, TAG_R, TAG_MU = 1, 2, 3, 4, 5
TAG_RG, TAG_E1, TAG_E2 = 6, 7, 8
OPT_ENCAPS_PATH = 1
OPT_PROFILE = 2
OPT_KEYGEN_PATH = 4
OPT_PANEL_ROWS = 6
OPT_REGEN_PATH = 7
OPT_R_OPERAND = 8
OPT_V_PATH = 9
OPT_PDL = 10
KERNELS = ["rng_fill", "sample_uniform", "sample_cbd", "sample_bits", "keygen_stored", "keygen_regen",
           "expand_R_v", "encaps_tc", "encaps_simt", "decaps", "keygen_prep", "keygen_tc", "fo_verdict",
           "sample_gauss", "sample_cuniform", "prep_R_pv", "encaps_regen_tc", "sample_kem", "wide_pack", "wide_keygen", "sample_pke"]

EXPORTS = [
    "lwe_create", "lwe_destroy", "lwe_strerror", "lwe_last_cuda_error", "lwe_launch_count",
    "lwe_rng_fill", "lwe_sample_uniform", "lwe_sample_cbd", "lwe_sample_bits", "lwe_sample_kem",
    "lwe_keygen", "lwe_encaps", "lwe_decaps", "lwe_decaps_fo", "lwe_kem_host",
    "lwe_sample_gauss_s8", "lwe_sample_gauss_u16", "lwe_sample_cuniform_s8", "lwe_sample_pke", "lwe_encaps_pv", "lwe_set_option",
    "lwe_profile_read", "lwe_profile_reset",
    "lwe_sample_uniform_u32", "lwe_sample_cbd_s8", "lwe_wide_load_matrix", "lwe_wide_load_matrix_seeded", "lwe_wide_keygen",
    "lwe_wide_encaps", "lwe_wide_decaps",
    "lwe_decaps_static", "lwe_probe_int8_pipe",
]
STATIC_MAX_COLS, STATIC_MAX_BATCH = 16384, 64                # LWE_STATIC_MAX_COLS / _BATCH of include/lwe.h


class LweError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where}: {ERRORS.get(code, code)} {detail}".strip())


class lwe_params(C.Structure):
    _fields_ = [(x, C.c_uint32) for x in ("n", "m", "k", "q", "eta", "max_batch")]


_lib = None


def load_library() -> C.CDLL:
    """dlopen the in-tree library (no compute); raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_01211_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(str(LIB_PATH))
    vp, u64, u32, sz = C.c_void_p, C.c_uint64, C.c_uint32, C.c_size_t
    lib.lwe_create.argtypes = [C.POINTER(vp), C.POINTER(lwe_params), C.c_int]
    lib.lwe_destroy.argtypes = [vp]
    lib.lwe_destroy.restype = None
    lib.lwe_strerror.argtypes = [C.c_int]
    lib.lwe_strerror.restype = C.c_char_p
    lib.lwe_last_cuda_error.argtypes = [vp]
    lib.lwe_launch_count.argtypes = [vp]
    lib.lwe_launch_count.restype = u64
    lib.lwe_set_option.argtypes = [vp, C.c_int, C.c_int64]
    lib.lwe_profile_read.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(u64)]
    lib.lwe_profile_reset.argtypes = [vp]
    lib.lwe_rng_fill.argtypes = [vp, vp, sz, C.c_char_p, C.c_char_p, u64, vp]
    for f in (lib.lwe_sample_uniform, lib.lwe_sample_cbd, lib.lwe_sample_bits):
        f.argtypes = [vp, vp, u64, u64, u64, u32, u32, u32, vp]
    lib.lwe_sample_kem.argtypes = [vp, vp, vp, vp, vp, u64, u32, u32, vp]
    lib.lwe_keygen.argtypes = [vp, vp, u64, vp, vp, vp, u32, vp]
    lib.lwe_encaps.argtypes = [vp, vp, u64, vp, vp, vp, vp, vp, u32, vp]
    lib.lwe_decaps.argtypes = [vp, vp, vp, vp, vp, u32, vp]
    lib.lwe_decaps_fo.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, u32, vp]
    for f in (lib.lwe_sample_gauss_s8, lib.lwe_sample_gauss_u16):
        f.argtypes = [vp, vp, u64, u64, u64, u32, u32, u32, C.c_double, vp]
    lib.lwe_sample_cuniform_s8.argtypes = [vp, vp, u64, u64, u64, u32, u32, u32, u32, vp]
    lib.lwe_sample_pke.argtypes = [vp, vp, vp, vp, vp, vp, vp, u64, u32, u32, C.c_double, u32, vp]
    lib.lwe_encaps_pv.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, u32, vp]
    lib.lwe_kem_host.argtypes = [vp, vp, u64, vp, vp, vp, vp, vp, vp, vp, vp, u32, vp]
    for f in (lib.lwe_sample_uniform_u32, lib.lwe_sample_cbd_s8):
        f.argtypes = [vp, vp, u64, u64, u64, u32, u32, u32, vp]
    lib.lwe_wide_load_matrix.argtypes = [vp, vp, vp]
    lib.lwe_wide_load_matrix_seeded.argtypes = [vp, u64, vp]
    lib.lwe_wide_keygen.argtypes = [vp, vp, vp, vp, u32, vp]
    lib.lwe_wide_encaps.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, u32, vp]
    lib.lwe_wide_decaps.argtypes = [vp, vp, vp, vp, vp, u32, vp]
    lib.lwe_probe_int8_pipe.argtypes = [vp, u32, C.c_int, C.POINTER(u64), vp]
    lib.lwe_decaps_static.argtypes = [u32, u32, u32, vp, vp, vp, vp, u32, vp]
    _lib = lib
    return lib


def _ptr(t) -> int | None:
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def decaps_static(n: int, k: int, q: int, d_U, d_v, d_s, d_mubits_out, batch: int = 1, stream=None):
    """lwe_decaps_static: Decaps without a context, for callers that may not allocate device memory (they are handed
    buffers and a stream by a host framework whose allocator owns the device).  Nothing is allocated here or in the
    library: the scratch is a fixed array inside liblwe_b200.so, shared by every call on the device, so calls must not
    overlap on the GPU, and batch * k <= STATIC_MAX_COLS, batch <= STATIC_MAX_BATCH.  The tensors' device must be the
    current device.  Make the first call on a device outside stream capture."""
    rc = load_library().lwe_decaps_static(n, k, q, _ptr(d_U), _ptr(d_v), _ptr(d_s), _ptr(d_mubits_out), batch, _stream(stream))
    if rc != LWE_OK:
        raise LweError(rc, "lwe_decaps_static")


class Context:
    """RAII wrapper of lwe_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, n: int, m: int, k: int, q: int, eta: int, max_batch: int = 1, device: int = 0):
        self._h = C.c_void_p()
        self._lib = load_library()
        self.params = lwe_params(n, m, k, q, eta, max_batch)
        self.device = device
        rc = self._lib.lwe_create(C.byref(self._h), C.byref(self.params), device)
        if rc != LWE_OK:
            self._h = C.c_void_p()
            raise LweError(rc, "lwe_create")

    # -- plumbing
    def close(self):
        h = getattr(self, "_h", None)
        if h is not None and h.value:
            self._h = None                      # first: at interpreter shutdown module globals may already be gone
            self._lib.lwe_destroy(h)

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, rc: int, where: str):
        if rc != LWE_OK:
            detail = ""
            if rc == -4:
                detail = f"(cudaError {self._lib.lwe_last_cuda_error(self._h)})"
            raise LweError(rc, where, detail)

    def launch_count(self) -> int:
        return int(self._lib.lwe_launch_count(self._h))

    def set_option(self, option: int, value: int):
        self._check(self._lib.lwe_set_option(self._h, option, value), "lwe_set_option")

    def probe_int8_pipe(self, iters: int, signed_dense_b: bool = False, stream=None) -> int:
        """one launch of the tensor-pipe probe; returns the int8 operations it performs (time it with events)"""
        ops = C.c_uint64(0)
        self._check(self._lib.lwe_probe_int8_pipe(self._h, iters, int(signed_dense_b), C.byref(ops), _stream(stream)),
                    "lwe_probe_int8_pipe")
        return ops.value

    def profile_reset(self):
        self._check(self._lib.lwe_profile_reset(self._h), "lwe_profile_reset")

    def profile_read(self) -> dict:
        """{kernel name: (total device ms, timed launches)} since the last reset (synchronises)"""
        out = {}
        for kid, name in enumerate(KERNELS):
            ms, cnt = C.c_double(0), C.c_uint64(0)
            self._check(self._lib.lwe_profile_read(self._h, kid, C.byref(ms), C.byref(cnt)), "lwe_profile_read")
            if cnt.value:
                out[name] = (ms.value, int(cnt.value))
        return out

    # -- a1 / a2
    def rng_fill(self, d_out, nbytes: int, key: bytes, iv: bytes, byte_offset: int = 0, stream=None):
        assert len(key) == 16 and len(iv) == 16
        self._check(self._lib.lwe_rng_fill(self._h, _ptr(d_out), nbytes, key, iv, byte_offset, _stream(stream)),
                    "lwe_rng_fill")

    def sample_uniform(self, d_out, first: int, count: int, seed: int, tag: int, inst0: int = 0, n_inst: int = 1,
                       stream=None):
        self._check(self._lib.lwe_sample_uniform(self._h, _ptr(d_out), first, count, seed, tag, inst0, n_inst,
                                                 _stream(stream)), "lwe_sample_uniform")

    def sample_cbd(self, d_out, first: int, count: int, seed: int, tag: int, inst0: int = 0, n_inst: int = 1,
                   stream=None):
        self._check(self._lib.lwe_sample_cbd(self._h, _ptr(d_out), first, count, seed, tag, inst0, n_inst,
                                             _stream(stream)), "lwe_sample_cbd")

    def sample_bits(self, d_out, first_bit: int, nbits: int, seed: int, tag: int, inst0: int = 0, n_inst: int = 1,
                    stream=None):
        self._check(self._lib.lwe_sample_bits(self._h, _ptr(d_out), first_bit, nbits, seed, tag, inst0, n_inst,
                                              _stream(stream)), "lwe_sample_bits")

    def sample_kem(self, d_s, d_e, d_Rbits, d_mubits, seed: int, inst0: int = 0, n_inst: int = 1, stream=None):
        self._check(self._lib.lwe_sample_kem(self._h, _ptr(d_s), _ptr(d_e), _ptr(d_Rbits), _ptr(d_mubits), seed, inst0,
                                             n_inst, _stream(stream)), "lwe_sample_kem")

    # -- a3..a6
    def keygen(self, d_A, seed_A: int, d_s, d_e, d_b, batch: int = 1, stream=None):
        self._check(self._lib.lwe_keygen(self._h, _ptr(d_A), seed_A, _ptr(d_s), _ptr(d_e), _ptr(d_b), batch,
                                         _stream(stream)), "lwe_keygen")

    def encaps(self, d_A, seed_A: int, d_b, d_Rbits, d_mubits, d_U, d_v, batch: int = 1, stream=None):
        self._check(self._lib.lwe_encaps(self._h, _ptr(d_A), seed_A, _ptr(d_b), _ptr(d_Rbits), _ptr(d_mubits),
                                         _ptr(d_U), _ptr(d_v), batch, _stream(stream)), "lwe_encaps")

    def decaps(self, d_U, d_v, d_s, d_mubits_out, batch: int = 1, stream=None):
        self._check(self._lib.lwe_decaps(self._h, _ptr(d_U), _ptr(d_v), _ptr(d_s), _ptr(d_mubits_out), batch,
                                         _stream(stream)), "lwe_decaps")

    def decaps_fo(self, d_A, d_b, d_U, d_v, d_s, d_Rbits, d_mubits_out, d_ok, batch: int = 1, stream=None):
        self._check(self._lib.lwe_decaps_fo(self._h, _ptr(d_A), _ptr(d_b), _ptr(d_U), _ptr(d_v), _ptr(d_s),
                                            _ptr(d_Rbits), _ptr(d_mubits_out), _ptr(d_ok), batch, _stream(stream)),
                    "lwe_decaps_fo")

    # -- N2: the paper's own PKE variant
    def sample_gauss_s8(self, d_out, first: int, count: int, seed: int, tag: int, inst0: int, n_inst: int, sigma: float,
                        stream=None):
        self._check(self._lib.lwe_sample_gauss_s8(self._h, _ptr(d_out), first, count, seed, tag, inst0, n_inst,
                                                  float(sigma), _stream(stream)), "lwe_sample_gauss_s8")

    def sample_gauss_u16(self, d_out, first: int, count: int, seed: int, tag: int, inst0: int, n_inst: int, sigma: float,
                         stream=None):
        self._check(self._lib.lwe_sample_gauss_u16(self._h, _ptr(d_out), first, count, seed, tag, inst0, n_inst,
                                                   float(sigma), _stream(stream)), "lwe_sample_gauss_u16")

    def sample_cuniform_s8(self, d_out, first: int, count: int, seed: int, tag: int, inst0: int, n_inst: int, bound: int,
                           stream=None):
        self._check(self._lib.lwe_sample_cuniform_s8(self._h, _ptr(d_out), first, count, seed, tag, inst0, n_inst,
                                                     bound, _stream(stream)), "lwe_sample_cuniform_s8")

    def sample_pke(self, d_s, d_e, d_R, d_E1, d_e2, d_mubits, seed: int, inst0: int, n_inst: int, sigma: float, e2_bound: int,
                   stream=None):
        self._check(self._lib.lwe_sample_pke(self._h, _ptr(d_s), _ptr(d_e), _ptr(d_R), _ptr(d_E1), _ptr(d_e2), _ptr(d_mubits),
                                             seed, inst0, n_inst, float(sigma), e2_bound, _stream(stream)), "lwe_sample_pke")

    def encaps_pv(self, d_A, d_t, d_R, d_E1, d_e2, d_mubits, d_U, d_v, batch: int = 1, stream=None):
        self._check(self._lib.lwe_encaps_pv(self._h, _ptr(d_A), _ptr(d_t), _ptr(d_R), _ptr(d_E1), _ptr(d_e2),
                                            _ptr(d_mubits), _ptr(d_U), _ptr(d_v), batch, _stream(stream)),
                    "lwe_encaps_pv")

    # -- wide contexts (q > 65536: uint32 residues, int8 small objects)
    def sample_uniform_u32(self, d_out, first: int, count: int, seed: int, tag: int, inst0: int = 0, n_inst: int = 1,
                           stream=None):
        self._check(self._lib.lwe_sample_uniform_u32(self._h, _ptr(d_out), first, count, seed, tag, inst0, n_inst,
                                                     _stream(stream)), "lwe_sample_uniform_u32")

    def sample_cbd_s8(self, d_out, first: int, count: int, seed: int, tag: int, inst0: int = 0, n_inst: int = 1,
                      stream=None):
        self._check(self._lib.lwe_sample_cbd_s8(self._h, _ptr(d_out), first, count, seed, tag, inst0, n_inst,
                                                _stream(stream)), "lwe_sample_cbd_s8")

    def wide_load_matrix(self, d_A, stream=None):
        self._check(self._lib.lwe_wide_load_matrix(self._h, _ptr(d_A), _stream(stream)), "lwe_wide_load_matrix")

    def wide_load_matrix_seeded(self, seed_A: int, stream=None):
        self._check(self._lib.lwe_wide_load_matrix_seeded(self._h, seed_A, _stream(stream)), "lwe_wide_load_matrix_seeded")

    def wide_keygen(self, d_s, d_e, d_t, batch: int = 1, stream=None):
        self._check(self._lib.lwe_wide_keygen(self._h, _ptr(d_s), _ptr(d_e), _ptr(d_t), batch, _stream(stream)),
                    "lwe_wide_keygen")

    def wide_encaps(self, d_t, d_R, d_E1, d_e2, d_mubits, d_U, d_v, batch: int = 1, stream=None):
        self._check(self._lib.lwe_wide_encaps(self._h, _ptr(d_t), _ptr(d_R), _ptr(d_E1), _ptr(d_e2), _ptr(d_mubits),
                                              _ptr(d_U), _ptr(d_v), batch, _stream(stream)), "lwe_wide_encaps")

    def wide_decaps(self, d_U, d_v, d_s, d_mubits_out, batch: int = 1, stream=None):
        self._check(self._lib.lwe_wide_decaps(self._h, _ptr(d_U), _ptr(d_v), _ptr(d_s), _ptr(d_mubits_out), batch,
                                              _stream(stream)), "lwe_wide_decaps")

    def kem_host(self, d_A, seed_A: int, h_s, h_e, h_Rbits, h_mubits, h_b, h_U, h_v, h_mubits_out, batch: int = 1,
                 stream=None):
        self._check(self._lib.lwe_kem_host(self._h, _ptr(d_A), seed_A, _ptr(h_s), _ptr(h_e), _ptr(h_Rbits),
                                           _ptr(h_mubits), _ptr(h_b), _ptr(h_U), _ptr(h_v), _ptr(h_mubits_out),
                                           batch, _stream(stream)), "lwe_kem_host")
