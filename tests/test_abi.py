"""The C-ABI library: builds, loads on a CPU-only box, exports every symbol include/ul.h
declares, fails loudly (no CPU fallback), and sizes its workspace like the paper says.  No GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libul():
    from paper_1309_3859_b200 import build, ul
    build.build()
    return ul


def test_exports_every_declared_symbol(libul):
    hdr = open(os.path.join(ROOT, "include", "ul.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ul_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(libul.SYMBOLS)
    L = libul.lib()
    for s in sorted(declared):
        assert hasattr(L, s), s


def test_no_cpu_fallback(libul):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    assert libul.lib().ul_create(C.byref(h), 4, 4, 1.0, 1) == libul.UL_ECUDA
    assert b"CUDA" in libul.lib().ul_last_error(None)
    with pytest.raises(libul.UlError):
        libul.Lattice(4, 4, 1.0, 1)


def test_argument_validation_without_device(libul):
    L = libul.lib()
    h = C.c_void_p()
    for Ns, Nt, beta in [(3, 4, 1.0), (4, 5, 1.0), (0, 4, 1.0), (4, 4, -1.0), (4, 4, float("nan"))]:
        assert L.ul_create(C.byref(h), Ns, Nt, beta, 1) == libul.UL_EINVAL
    assert L.ul_create(None, 4, 4, 1.0, 1) == libul.UL_EINVAL
    assert L.ul_sweep(None, 1, 1) == libul.UL_EINVAL
    assert L.ul_destroy(None) == libul.UL_OK


def test_workspace_sizing_follows_paper_formula(libul):
    # field accumulators = 2 x 8 B x (volume / step) x (points) per (mu, r, channel).
    # Here: Ns^3 (Nt/d) 3 r_max (1 + 12 n_fp) complex doubles plus O(volume) scratch: up to 8 batched
    # per-configuration tables of 64 B per (slab, site) (fp64 U, 12 fp32 plaquette sums).
    Ns, Nt, d, R, F = 24, 16, 2, 12, 5
    Vs, S = Ns ** 3, Nt // d
    acc = 16 * Vs * S * 3 * R * (1 + 12 * F)
    got = libul.workspace_bytes(Ns, Nt, d, 0, R, F)
    scratch = got - acc
    assert 0 < scratch < 8 * 64 * Vs * S + 2 * R * (1 + 12 * F) * 2 * 592 * 8 + 65536
    two = libul.workspace_bytes(Ns, Nt, 2, 4, R, F)
    assert abs((two - got) - acc // 2) < 4096
    assert libul.workspace_bytes(Ns, Nt, 3, 0, R, F) == 0          # 16 % 3 != 0
