"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: oracle/avmo.cpp is rebuilt with
-fsanitize=address,undefined (every report fatal) and tests/sanitized_oracle_scenarios.py — a banded run with B, a
capacity overflow, a tetrahedral map (field evaluation incl. NaN and outside points, runs with a signal, ion drift), a
folded grid map with steps from beyond its edges, the NEXT-3 gas extensions — is run against that build in a subprocess
with the ASan runtime preloaded.  The oracle indexes band tables, bucket grids, element records, signal bins and ion
arrays; an out-of-range index or an overflow in any of them would make every parity claim built on it worthless."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _gcc_file(name):
    out = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


def test_oracle_scenarios_are_clean_under_asan_and_ubsan():
    sys.path.insert(0, ROOT)
    from oracle import avmo
    so = avmo.build(sanitize=True)
    syms = subprocess.run(["nm", "-D", "--undefined-only", so], capture_output=True, text=True).stdout
    assert "__asan_" in syms and "__ubsan_" in syms, "the sanitizer build is not instrumented"
    asan = _gcc_file("libasan.so")
    assert asan, "libasan.so (gcc's AddressSanitizer runtime) not found"
    env = dict(os.environ, AVMO_SANITIZED="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitized_oracle_scenarios.py")], cwd=ROOT, env=env,
                       capture_output=True, text=True, timeout=900)
    tail = r.stdout[-2000:] + r.stderr[-4000:]
    assert r.returncode == 0, tail
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, tail
    assert "sanitized oracle scenarios: ok" in r.stdout, tail
