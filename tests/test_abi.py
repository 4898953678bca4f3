"""The C-ABI library builds for sm_100a, loads without a GPU and exports every entry
point include/lwe.h declares; the binding mirrors them.  No compute calls here."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def declared_functions():
    text = (ROOT / "include" / "lwe.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lwe_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_01211_b200 import build
    path = build.build()
    return ctypes.CDLL(str(path))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for required in ("lwe_keygen", "lwe_encaps", "lwe_decaps", "lwe_rng_fill", "lwe_create", "lwe_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in include/lwe.h but not exported"


def test_binding_lists_the_same_entry_points():
    from paper_2606_01211_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()


def test_strerror_and_null_handling_without_a_gpu(lib):
    lib.lwe_strerror.restype = ctypes.c_char_p
    assert lib.lwe_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5):
        assert lib.lwe_strerror(code)
    assert lib.lwe_create(None, None, 0) == -3            # LWE_ERR_NULLPTR, nothing touched
    lib.lwe_destroy(None)                                 # no-op
    lib.lwe_launch_count.restype = ctypes.c_uint64
    assert lib.lwe_launch_count(None) == 0


def test_no_cuda_device_is_reported_not_faked(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2606_01211_b200 import binding
    with pytest.raises(binding.LweError) as ei:
        binding.Context(256, 512, 256, 65536, 4)
    assert ei.value.code in (-5, -4)                      # unsupported: there is no CPU fallback


def test_product_does_not_import_the_oracle():
    pkg = ROOT / "paper_2606_01211_b200"
    for p in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + [ROOT / "include" / "lwe.h"]:
        text = p.read_text()
        assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), p
        assert "lwe_oracle" not in text and "orc_" not in text, p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in (".py", ".c", ".h"):
            text = p.read_text()
            assert not re.search(r"^\s*(from|import)\s+paper_2606_01211_b200\b", text, flags=re.M), p
            assert "#include \"../paper" not in text and "lwe_internal" not in text and "lwe.h" not in text, p


def test_kernel_id_table_of_the_binding_matches_the_header():
    """binding.KERNELS[i] names kernel LWE_K_<NAME> = i of include/lwe.h (lwe_profile_read ids)"""
    import re
    from paper_2606_01211_b200 import binding as B
    header = (ROOT / "include" / "lwe.h").read_text()
    ids = {name: int(i) for name, i in re.findall(r"LWE_K_([A-Z0-9_]+) = (\d+)", header)}
    assert ids.pop("COUNT") == len(B.KERNELS) == len(ids)
    for name, i in ids.items():
        assert B.KERNELS[i].upper() == name, (i, name, B.KERNELS[i])


def test_decaps_static_checks_its_limits_before_touching_cuda(lib):
    """lwe_decaps_static (the entry point for callers that cannot allocate): argument and size-limit errors come back
    without any CUDA call, so they can be checked on a box with no GPU; the limits are those of include/lwe.h."""
    from paper_2606_01211_b200 import binding as B
    header = (ROOT / "include" / "lwe.h").read_text()
    assert int(re.search(r"#define LWE_STATIC_MAX_COLS (\d+)u", header).group(1)) == B.STATIC_MAX_COLS
    assert int(re.search(r"#define LWE_STATIC_MAX_BATCH (\d+)u", header).group(1)) == B.STATIC_MAX_BATCH
    f = B.load_library().lwe_decaps_static
    p = 4096                                               # any non-NULL 16-byte aligned value: never dereferenced here
    assert f(64, 256, 65536, p, p, p, p, B.STATIC_MAX_BATCH + 1, None) == -5
    assert f(64, 2048, 65536, p, p, p, p, B.STATIC_MAX_COLS // 2048 + 1, None) == -5
    assert f(64, 256, 65537, p, p, p, p, 1, None) == -1
    assert f(64, 12, 65536, p, p, p, p, 1, None) == -1
    assert f(64, 256, 65536, None, p, p, p, 1, None) == -3
    assert f(64, 256, 65536, p + 2, p, p, p, 1, None) == -2


def test_every_enqueueing_entry_point_opens_an_nvtx_range():
    """SURVEY section 5 row 1 (the paper profiles with Nsight Systems + NVTX): each lwe_* call that
    enqueues device work is bracketed by an NVTX range named after it."""
    src = (ROOT / "paper_2606_01211_b200" / "csrc" / "api.cu").read_text()
    bodies = re.findall(r"^(?:int|void) (lwe_[a-z0-9_]+)\([^{;]*\)\n\{\n(.*?)^\}", src, flags=re.M | re.S)
    assert len(bodies) >= 25
    quiet = {"lwe_last_cuda_error", "lwe_set_option", "lwe_profile_reset", "lwe_profile_read"}
    for name, body in bodies:
        if name not in quiet:
            assert f'NvtxScope nvtx_("{name}");' in body, name
