"""ul_plaquette_noalloc: the plaquette average for callers that must not allocate (scratch in a fixed file-scope device array)
against ul_plaquette (scratch from cudaMalloc).  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ul():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1309_3859_b200 import build, ul as _ul
    build.build()
    return _ul


def test_plaquette_noalloc_equals_plaquette_on_two_calls_in_a_row(ul):
    import torch
    a = ul.Lattice(16, 4, 0.99, 3)                                 # gx = 1 block column
    b = ul.Lattice(24, 8, 1.0, 7)                                  # gx = 3: another grid shape through the same scratch array
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    for it in range(2):                                            # two calls in a row per lattice, the configuration moving on
        for L in (a, b):
            L.sweep(1, 2)
            n0 = L.launch_count()
            L.plaquette_noalloc(out)
            assert L.launch_count() - n0 == 3
            L.sync()
            got = out.cpu().numpy().copy()
            want = np.asarray(L.plaquette())
            # same kernels, same fixed order of additions: bit for bit (the tests' tolerance for reductions is 1e-12)
            assert np.array_equal(got, want), (it, got, want)
            assert abs(got[0] - 0.5 * (got[1] + got[2])) < 1e-15 and 0.0 < got[0] < 1.0
    # back to back without anything in between: the array keeps the last call's contents, the result does not depend on them
    a.plaquette_noalloc(out)
    b.plaquette_noalloc(out)
    a.plaquette_noalloc(out)
    a.sync()
    assert np.array_equal(out.cpu().numpy(), np.asarray(a.plaquette()))


def test_plaquette_noalloc_rejects_bad_arguments_and_sizes_beyond_the_scratch(ul):
    import torch
    a = ul.Lattice(8, 4, 1.0, 1)
    with pytest.raises(ValueError):
        a.plaquette_noalloc(torch.zeros(3, dtype=torch.float32, device="cuda"))
    rc = ul.lib().ul_plaquette_noalloc(a._h, None)
    assert rc == -1                                                # UL_EINVAL: null output
    # Ns = 392 needs ceil(392^2 / 256) = 601 > 592 block columns: beyond the fixed array (1.9 GB of links: fine on a B200)
    try:
        big = ul.Lattice(392, 2, 1.0, 1)
    except ul.UlError as e:                                        # no memory for the lattice itself: nothing to check
        pytest.skip(f"cannot create the 392^3 x 2 lattice: {e}")
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    with pytest.raises(ul.UlError) as ei:
        big.plaquette_noalloc(out)
    assert ei.value.code == -1 and "beyond the fixed scratch" in str(ei.value)
    big.close()
