"""The C oracle under AddressSanitizer + UndefinedBehaviorSanitizer.

oracle/wilson_clover.c is rebuilt with -fsanitize=address,undefined and every entry point is
driven on small lattices (2^4: both hops of an axis coincide; 4^3 x 6; both boundary conditions;
a singular clover site) in a subprocess with libasan preloaded.  Any out-of-bounds access,
use of uninitialised stack through UB, signed overflow or misaligned access aborts the child.
"""
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = textwrap.dedent("""
    import numpy as np, torch, sys
    sys.path.insert(0, %r)
    import gen, oracle
    for (L, T, bc, csw) in ((2, 2, 1, 1.0), (4, 6, 0, 1.5), (4, 4, 1, 1.0)):
        U = gen.gauge_field(L, T, 7, 0.4, True).numpy()
        ora = oracle.WilsonClover(L, T, csw, -0.1, bc, U)
        x = gen.spinor_field(L, T, 3).numpy()
        y = ora.apply_D(x)
        ys = ora.apply_schur(np.where(ora.even, x, 0.0))
        bh = ora.prepare_rhs(x)
        xo = ora.reconstruct_odd(x, np.where(ora.even, x, 0.0))
        assert all(np.isfinite(a).all() for a in (y, ys, bh, xo))
    try:
        oracle.WilsonClover(4, 4, 0.0, -4.0, 0, gen.unit_gauge_field(4, 4).numpy())   # A = 0: singular
    except Exception as e:
        print("singular reported:", type(e).__name__)
    print("SANITIZED-ORACLE-OK")
""")


def test_oracle_clean_under_asan_and_ubsan():
    from oracle.build import build_sanitized
    lib = build_sanitized()
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan.so not found next to gcc")
    env = dict(os.environ, ORACLE_LIB=lib, LD_PRELOAD=asan, OMP_NUM_THREADS="1",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:halt_on_error=1",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    r = subprocess.run([sys.executable, "-c", DRIVER % ROOT], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "SANITIZED-ORACLE-OK" in r.stdout
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-3000:]
