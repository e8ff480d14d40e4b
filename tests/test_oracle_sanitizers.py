"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: every entry point the pins and the
parity tests use runs once on small lattices (ragged shapes included) in a subprocess that loads the instrumented build;
any out-of-bounds access, use after free, signed overflow or misaligned access aborts it."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import sys
sys.path.insert(0, {root!r})
import numpy as np
from oracle import ulo
assert ulo.build().endswith("_san.so")
for Ns, Nt, d in ((4, 4, 2), (6, 4, 1), (2, 2, 2), (4, 8, 4)):
    o = ulo.Oracle(Ns, Nt, 0.97, 11)
    o.sweep(1, 2)
    o.set_update_algorithm(1, 1.1); o.sweep(1, 0); o.set_update_algorithm(0)
    for kind in (0, 1):
        for parity in (0, 1):
            for mu in range(4):
                o.substep(kind, parity, mu, d)
    links = o.get_links(); o.set_links(links); o.set_counter(o.get_counter() + 3)
    R = Ns // 2
    fps = [(0, 0, 0), (1, Ns - 1, 2), (-1, 0, 1)]
    o.multilevel(d, 2, R, fps); o.read_correlators(); o.read_slab_averages()
    o.set_multihit(1); o.multilevel(d, 1, R, fps); o.set_multihit(0)
    o.measure_begin(d, R); o.accumulate(); o.accumulate(); o.measure_end()
    if Nt % (2 * d) == 0:
        o.multilevel2(d, 2, 2 * d, 2, R, fps); o.read_correlators(); o.read_slab_field_averages()
        o.measure2_begin(d, 2 * d, R, fps); o.accumulate(); o.combine(); o.accumulate(); o.combine(); o.measure2_end()
    o.plaquette(); o.polyakov(0); o.polyakov(1); o.polyakov_naive(R); o.staple(2, Ns ** 3 * Nt - 1)
    o.close()
ulo.heatbath_phi(3.0, 5, 1, 2, 3, 7); ulo.philox4x32_10([1, 2, 3, 4], [5, 6]); ulo.paper_accumulator_bytes(24, 16, 2)
print("SANITIZED OK")
"""


@pytest.mark.timeout(600)
def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("no libasan next to gcc")
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, ULO_SANITIZE="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    out = subprocess.run([sys.executable, str(script)], env=env, capture_output=True, text=True, timeout=580)
    assert out.returncode == 0 and "SANITIZED OK" in out.stdout, (out.stdout[-2000:], out.stderr[-4000:])
