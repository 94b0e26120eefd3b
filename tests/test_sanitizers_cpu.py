"""AddressSanitizer + UndefinedBehaviorSanitizer builds of the two pieces of host code that index memory by hand:
the oracle (oracle/hxo.c) and the page allocator (csrc/hx_pool.cpp) ("Race detection /
sanitizers").  Each is compiled with -fsanitize=address,undefined -fno-sanitize-recover and driven in a child
python process with libasan preloaded: the oracle by its own pin tests, the allocator by a sequence that covers
every entry point and every error path.  Any bad access or undefined operation aborts the child."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]


def _libasan():
    out = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not out or not os.path.isabs(out) or not os.path.exists(out):
        pytest.skip("libasan.so not found next to gcc")
    return os.path.realpath(out)


def _child(code, args, timeout):
    env = dict(os.environ, LD_PRELOAD=_libasan(), ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="4", PYTHONPATH=ROOT)
    r = subprocess.run([sys.executable, "-c", code, *args], capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)
    assert r.returncode == 0, (r.stdout[-3000:], r.stderr[-3000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
    return r


def test_oracle_pins_under_asan_ubsan(tmp_path):
    so = str(tmp_path / "libhxo_san.so")
    subprocess.check_call(["gcc", "-std=c11", "-fopenmp", "-fPIC", "-shared", *SAN, "-o", so,
                           os.path.join(ROOT, "oracle", "hxo.c"), "-lm"])
    code = """
import sys
import oracle.hxo as H
H._SO = sys.argv[1]
H.build = lambda force=False: H._SO          # the pins below run against the sanitized build of the same source
import pytest
sys.exit(pytest.main(["-q", "-x", "-p", "no:cacheprovider", "-m", "not gpu", "-k", "not hypothesis and not fuzz",
                      "tests/test_oracle_pins.py", "tests/test_oracle_pins_next.py"]))
"""
    r = _child(code, [so], timeout=900)
    assert " passed" in r.stdout, r.stdout[-2000:]


def test_page_pool_under_asan_ubsan(tmp_path):
    stub = tmp_path / "stub.cpp"
    stub.write_text('#include <cstdarg>\nnamespace hx { void set_error(const char*, ...) {} }\n')
    so = str(tmp_path / "libpool_san.so")
    subprocess.check_call(["g++", "-std=c++17", "-fPIC", "-shared", *SAN, "-I", os.path.join(ROOT, "include"), "-o", so,
                           os.path.join(ROOT, "paper_2502_07903_b200", "csrc", "hx_pool.cpp"), str(stub)])
    code = """
import ctypes as C, sys
import numpy as np
L = C.CDLL(sys.argv[1])
L.hx_pool_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32]
L.hx_pool_shuffle.argtypes = [C.c_void_p, C.c_uint64]
L.hx_pool_alloc.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
L.hx_pool_free.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
L.hx_pool_num_free.argtypes = [C.c_void_p]
L.hx_pool_num_pages.argtypes = [C.c_void_p]
L.hx_pool_alloc_table.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32]
L.hx_pool_destroy.argtypes = [C.c_void_p]
OK, INVALID, NO_PAGES = 0, 1, 5
h = C.c_void_p()
assert L.hx_pool_create(C.byref(h), -1) == INVALID and L.hx_pool_create(None, 4) == INVALID
assert L.hx_pool_create(C.byref(h), 1000) == OK and L.hx_pool_shuffle(h, 42) == OK
rng = np.random.default_rng(0)
held = []
for it in range(300):                                        # random alloc / free traffic, page reuse all the time
    if held and rng.random() < 0.45:
        ids = held.pop(int(rng.integers(len(held))))
        assert L.hx_pool_free(h, ids.ctypes.data, ids.size) == OK
    else:
        n = int(rng.integers(0, 120))
        ids = np.empty(max(n, 1), dtype=np.int32)
        rc = L.hx_pool_alloc(h, n, ids.ctypes.data)
        if rc == OK:
            held.append(ids[:n].copy())
        else:
            assert rc == NO_PAGES and n > L.hx_pool_num_free(h)
flat = np.concatenate(held) if held else np.empty(0, dtype=np.int32)
assert len(set(flat.tolist())) == flat.size and L.hx_pool_num_free(h) == 1000 - flat.size
bad = np.array([1000, -1], dtype=np.int32)
assert L.hx_pool_free(h, bad.ctypes.data, 1) == INVALID and L.hx_pool_free(h, bad[1:].ctypes.data, 1) == INVALID
if flat.size:
    dup = np.array([flat[0], flat[0]], dtype=np.int32)
    nf = L.hx_pool_num_free(h)
    assert L.hx_pool_free(h, dup.ctypes.data, 2) == INVALID and L.hx_pool_num_free(h) == nf
for ids in held:
    assert L.hx_pool_free(h, ids.ctypes.data, ids.size) == OK
assert L.hx_pool_num_free(h) == 1000 == L.hx_pool_num_pages(h)
lens = np.array([17, 0, 1, 4096, 33], dtype=np.int32)
bt = np.empty((5, 256), dtype=np.int32)
assert L.hx_pool_alloc_table(h, lens.ctypes.data, 5, 16, bt.ctypes.data, 256) == OK
assert (bt >= 0).sum() == 2 + 0 + 1 + 256 + 3
assert L.hx_pool_alloc_table(h, lens.ctypes.data, 5, 16, bt.ctypes.data, 255) == INVALID       # row 3 does not fit
big = np.array([16 * 800], dtype=np.int32)
row = np.empty((1, 800), dtype=np.int32)
assert L.hx_pool_alloc_table(h, big.ctypes.data, 1, 16, row.ctypes.data, 800) == NO_PAGES
assert L.hx_pool_alloc_table(h, None, 1, 16, row.ctypes.data, 800) == INVALID
used = bt[bt >= 0].astype(np.int32)
assert L.hx_pool_free(h, used.ctypes.data, used.size) == OK and L.hx_pool_num_free(h) == 1000
L.hx_pool_destroy(h)
L.hx_pool_destroy(None)
z = C.c_void_p()
assert L.hx_pool_create(C.byref(z), 0) == OK and L.hx_pool_num_free(z) == 0
L.hx_pool_destroy(z)
print("pool ok")
"""
    r = _child(code, [so], timeout=300)
    assert "pool ok" in r.stdout
