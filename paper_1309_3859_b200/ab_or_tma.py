"""A/B of the two overrelaxation kernels on the 64^4 bench lattice: the direct gather (k_update<1, MU, 4>) against the
bulk-copy (TMA) staged gather (k_update_or_tma<MU>, selected with UL_OR_TMA=1).

    python -m paper_1309_3859_b200.ab_or_tma            # bit-identity + CUDA-event timings of both
    python -m paper_1309_3859_b200.ab_or_tma --profile  # a few launches of each, for ncu (profiles/r02_tma_ab.md)
"""
import os
import sys

import numpy as np


def main():
    import torch
    from . import ul
    os.environ.pop("UL_OR_TMA", None)
    a = ul.Lattice(64, 64, 0.98, 5)                       # direct
    os.environ["UL_OR_TMA"] = "1"
    b = ul.Lattice(64, 64, 0.98, 5)                       # staged
    os.environ.pop("UL_OR_TMA", None)

    def masked(L):
        for parity in (0, 1):
            for mu in range(4):
                L.substep(1, parity, mu, 2)

    for L in (a, b):
        L.sweep(1, 1)
    if "--profile" in sys.argv:
        for L in (a, b):
            L.substep(1, 0, 0, 0)
            L.substep(1, 0, 1, 2)
            L.sync()
        return
    for L in (a, b):
        L.sweep(0, 2)
        masked(L)
    print("bit-identical links after full and slab-masked overrelaxation sweeps:", np.array_equal(a.get_links_raw(), b.get_links_raw()))

    def ev(fn, n=20):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n * 1e3

    for name, L in (("direct", a), ("tma-staged", b)):
        print(f"{name:10s} OR sweep {ev(lambda: L.sweep(0, 1)):7.1f} us   slab-masked OR sweep (d=2) {ev(lambda: masked(L)):7.1f} us")


if __name__ == "__main__":
    main()
