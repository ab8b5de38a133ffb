"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md §5 "sanitizers").

compute-sanitizer is closed on the GPU pool, so the CPU oracle is the one piece that can run under
a sanitizer.  oracle/build.py builds oracle/liboracle_san.so (-fsanitize=address,undefined,
-fno-sanitize-recover=undefined); this test re-runs the oracle pins P1-P16 in a child process with
the ASan runtime preloaded and ORACLE_SANITIZE=1, so every out-of-bounds access, use after free,
signed overflow or misaligned access inside the oracle aborts the child.
"""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_pins_pass_under_asan_and_ubsan():
    from oracle import build as ob
    rt = ob.asan_runtime()
    assert os.path.exists(rt), f"ASan runtime not found: {rt}"
    lib = ob.build(sanitize=True)
    assert lib.endswith("liboracle_san.so") and os.path.exists(lib)
    env = dict(os.environ)
    env.update(ORACLE_SANITIZE="1", LD_PRELOAD=rt,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",     # CPython itself leaks by design
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    res = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                          os.path.join(ROOT, "tests", "test_oracle_pins.py")],
                         cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    tail = (res.stdout + res.stderr)[-3000:]
    assert res.returncode == 0, tail
    assert "passed" in res.stdout and "failed" not in res.stdout, tail
    assert "runtime error" not in tail and "AddressSanitizer" not in tail, tail


def test_sanitized_build_is_the_one_loaded():
    """ORACLE_SANITIZE=1 really switches the library (guards against the test above passing on the plain build)."""
    from oracle import build as ob
    env = dict(os.environ)
    env.update(ORACLE_SANITIZE="1", LD_PRELOAD=ob.asan_runtime(), ASAN_OPTIONS="detect_leaks=0")
    code = ("from oracle import scape_oracle as o; L = o._lib(); print(L._name); "
            "import ctypes; assert hasattr(L, '__asan_init') or 'san' in L._name")
    res = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    assert res.stdout.strip().endswith("liboracle_san.so"), res.stdout
