"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY section 5, row "sanitizers"): the checker every
parity claim rests on is itself checked for out-of-bounds accesses, signed overflow, bad shifts and misaligned loads.
A child process with libasan preloaded loads oracle/liblwe_oracle_san.so (gcc -fsanitize=address,undefined
-fno-sanitize-recover) through the ordinary oracle package and runs one case of every family of functions at sizes with
ragged edges; any finding aborts the child.  Its results must also equal the normal build's."""
import json
import os
import subprocess
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent

CHILD = r'''
import hashlib, json, sys
import numpy as np
sys.path.insert(0, sys.argv[1])
sys.path.insert(0, sys.argv[1] + "/tests")
import oracle as O
from oracle import build
import os
assert str(build.build()).endswith("_san.so") == (os.environ.get("LWE_ORACLE_SANITIZE") == "1"), "wrong library in the child"
from conftest import read_golden

out = {}
def put(name, *arrays):
    h = hashlib.sha256()
    for a in arrays:
        h.update(np.ascontiguousarray(a).tobytes())
    out[name] = h.hexdigest()

# the pencil-and-paper example (tests/golden/lwe_hand_example.txt)
g = read_golden("lwe_hand_example.txt")
mat = lambda s: np.array([[int(x) for x in row.split()] for row in s.split(";")])
q, k = int(g["q"]), int(g["k"])
A, s, e = mat(g["A"]).astype(np.uint16), mat(g["s"])[0].astype(np.uint16), mat(g["e"])[0].astype(np.uint16)
b = O.keygen(A, s, e, q)
assert b.tolist() == mat(g["b"])[0].tolist()
Rbits = np.packbits(mat(g["R"]).astype(np.uint8).ravel(), bitorder="little")
mubits = np.packbits(mat(g["mu"])[0].astype(np.uint8), bitorder="little")
U, v = O.encaps(A, b, Rbits, mubits, k, q)
assert U.tolist() == mat(g["U"]).tolist() and v.tolist() == mat(g["v"])[0].tolist()
put("hand", b, U, v, O.decaps(U, v, s, q))

# AES / CTR at unaligned offsets and across the 64-bit carry of the counter
put("ctr", O.ctr_bytes(bytes(range(16)), bytes([0] * 8 + [0xff] * 8), 5, 16 * 3 + 7), O.ctr_bytes(O.seed_key(9), O.object_iv(4, 3, 2), 0, 33))
# samplers: rejection (q = 65521 and a tiny modulus with many rejections), strided, CBD, bits at a ragged bit offset
put("uniform", O.sample_uniform(3, 4099, 11, O.TAG_A, 0, 65521), O.sample_uniform(0, 257, 11, O.TAG_S, 1, 3),
    O.sample_uniform_strided(5, 264, 77, 11, O.TAG_A, 0, 65521))
put("cbd_bits", O.sample_cbd(8, 1001, 12, O.TAG_E, 2, 3329, 8), O.sample_bits(13, 1003, 12, O.TAG_R, 0))
put("gauss", O.gauss_cdt(2.3), O.sample_gauss(8, 999, 13, O.TAG_RG, 1, 2.3), O.sample_gauss(0, 40, 13, O.TAG_E, 0, 1.0, 12289),
    O.sample_cuniform(3, 777, 13, O.TAG_E2, 0, 3))
# keygen / encaps / decaps / FO on a ragged prime-modulus instance, honest and tampered
rng = np.random.default_rng(5)
m, n, k, q = 72, 40, 24, 65521
A = rng.integers(0, q, (m, n)).astype(np.uint16); s = rng.integers(0, q, n).astype(np.uint16)
e = O.sample_cbd(0, m, 14, O.TAG_E, 0, q, 4)
b = O.keygen(A, s, e, q)
Rbits, mubits = O.sample_bits(0, m * k, 14, O.TAG_R, 0), O.sample_bits(0, k, 14, O.TAG_MU, 0)
U, v = O.encaps(A, b, Rbits, mubits, k, q)
rows = np.array([0, 7, 39], np.uint32)
assert np.array_equal(O.encaps_rows(A, Rbits, rows, k, q), U[rows]) and np.array_equal(O.encaps_v(b, Rbits, mubits, k, q), v)
mu1, ok1 = O.decaps_fo(A, b, U, v, s, Rbits, q)
U2 = U.copy(); U2[n - 1, k - 1] ^= 1
mu2, ok2 = O.decaps_fo(A, b, U2, v, s, Rbits, q)
assert ok1 and not ok2 and np.array_equal(mu1, mubits)
put("kem", b, U, v, mu1, mu2)
# the paper's PKE, uint16 and wide (q = 65537 with elements equal to 2^16 = -1)
q = 12289; n = 48
A = rng.integers(0, q, (n, n)).astype(np.uint16); t = rng.integers(0, q, n).astype(np.uint16)
R, E1 = O.sample_gauss(0, n * k, 15, O.TAG_RG, 0, 1.7).reshape(n, k), O.sample_gauss(0, n * k, 15, O.TAG_E1, 0, 1.7).reshape(n, k)
e2 = O.sample_cuniform(0, k, 15, O.TAG_E2, 0, 3)
put("pv", *O.encaps_pv(A, t, R, E1, e2, mubits, q))
q = 65537
Aw = O.sample_uniform32(0, n * n, 16, O.TAG_A, 0, q).reshape(n, n); Aw[3, 5] = 65536; Aw[n - 1, 0] = 65536
sw, ew = O.sample_cbd_s8(0, n, 16, O.TAG_S, 0, 3), O.sample_gauss(0, n, 16, O.TAG_E, 0, 1.2)
tw = O.keygen_w(Aw, sw, ew, q)
Uw, vw = O.encaps_pv_w(Aw, tw, R, E1, e2, mubits, q)
dw = O.decaps_w(Uw, vw, sw, q)
assert np.array_equal(dw, mubits)
put("wide", tw, Uw, vw, dw, O.sample_uniform32_strided(1, n, 9, 16, O.TAG_A, 0, q))
print("RESULT " + json.dumps(out))
'''


def run_child(sanitized: bool) -> dict:
    from oracle import build
    env = dict(os.environ)
    env.pop("LD_PRELOAD", None)
    env.pop("LWE_ORACLE_SANITIZE", None)
    if sanitized:
        build.build_sanitized()
        env.update({"LWE_ORACLE_SANITIZE": "1", "LD_PRELOAD": build.asan_runtime(),
                    "ASAN_OPTIONS": "detect_leaks=0:abort_on_error=1:halt_on_error=1", "UBSAN_OPTIONS": "print_stacktrace=1"})
    r = subprocess.run([sys.executable, "-c", CHILD, str(ROOT)], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, f"child failed (sanitized={sanitized}):\n{r.stdout[-2000:]}\n{r.stderr[-4000:]}"
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
    line = [x for x in r.stdout.splitlines() if x.startswith("RESULT ")][-1]
    return json.loads(line[len("RESULT "):])


def test_oracle_runs_clean_under_asan_and_ubsan_and_gives_the_same_results():
    san = run_child(True)
    plain = run_child(False)
    assert set(san) == {"hand", "ctr", "uniform", "cbd_bits", "gauss", "kem", "pv", "wide"}
    assert san == plain
