"""GPU-vs-oracle parity (protocols P1-P3), through the C ABI.

P1  link level: per sub-step and per whole sweep, |theta_gpu - theta_cpu| mod 2pi <= 2e-5 rad
    except accept/reject flips (< 1e-5 of links) and the ill-conditioned class k < 0.05.
P2  frozen configuration: slab averages, correlators, fields, plaquette to relative 1e-5
    (DESIGN R17: abs <= 1e-5 * max(|cpu|, rms_term / sqrt(N))).
P3  ensemble: independent chains agree within 3 combined standard errors.
"""
import os

import numpy as np
import pytest

from tests import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

pytestmark = pytest.mark.gpu

TOL = 2e-5


@pytest.fixture(scope="module")
def ul():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1309_3859_b200 import build, ul as _ul
    build.build()
    return _ul


def wrapdiff(a, b):
    d = a.astype(np.float64) - b.astype(np.float64)
    return np.abs(d - 2 * np.pi * np.round(d / (2 * np.pi)))


def same_links(got, want):
    """Boundary round trip: the library keeps 32-bit binary angles (2 pi / 2^32 per
    unit).  fp32 radians come back bit for bit when 2^-6 <= |theta| < pi, to 1.2e-9 rad below that, and
    mod 2 pi at the fp32 neighbours of +-pi (fp32(pi) > pi wraps to the other end)."""
    a = np.abs(want)
    mid = (a >= 2.0 ** -6) & (a < 3.14159)
    d = wrapdiff(got, want)
    return np.array_equal(got[mid], want[mid]) and d[a < 3.14159].max(initial=0.0) <= 1.3e-9 and d.max(initial=0.0) <= 1e-7


def staple_k(o, mu, flat_sites):
    return np.array([o.staple(mu, int(s))[0] for s in flat_sites])


def check_links(got, want, before, o_before, label, allow_frac=1e-5):
    """P1 criterion.  o_before: oracle holding the configuration BEFORE the update (for k)."""
    diff = wrapdiff(got, want)
    untouched = (want == before)
    # frozen / other-parity links: boundary round trip only (an updated link whose new fp32 angle happens to equal its old one
    # also lands here: a few in 10^7, within the tolerance)
    assert (diff[untouched] > 1.3e-9).sum() <= 1e-6 * diff.size and diff[untouched].max(initial=0.0) <= TOL
    bad = np.argwhere(diff > TOL)
    n_links = got.size
    n_ill = 0
    n_other = 0
    for idx in bad:
        mu = int(idx[0])
        site = int(np.ravel_multi_index(tuple(idx[1:]), got.shape[1:]))
        k, _ = o_before.staple(mu, site)
        if k < 0.05:
            n_ill += 1
        else:
            n_other += 1          # accept/reject flip (heatbath) -- or a real bug
    assert n_other <= max(1, allow_frac * n_links), (label, n_other, n_ill, diff.max())
    assert n_ill <= max(2, 1e-4 * n_links), (label, n_ill)
    return n_other, n_ill, float(diff.max())


# ----------------------------------------------------------------------------- building blocks
def test_philox_known_answers_on_device(ul, ulo):
    import os
    rows = []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        rows.append([int(v, 16) for v in line.split() if v != "->"])
    rows = np.array(rows, dtype=np.uint64)
    out = ul.philox_selftest(rows[:, 0:4], rows[:, 4:6])
    assert np.array_equal(out, rows[:, 6:10].astype(np.uint32))
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2 ** 32, size=(1000, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(1000, 2), dtype=np.uint64).astype(np.uint32)
    out = ul.philox_selftest(ctr, key)
    for i in range(0, 1000, 37):
        assert np.array_equal(out[i], ulo.philox4x32_10(ctr[i], key[i]))


@pytest.mark.parametrize("Ns,Nt", [(2, 2), (4, 4), (6, 4), (8, 6), (16, 4)])
def test_hot_start_and_layout_roundtrip(ul, ulo, Ns, Nt):
    seed = (0x51 << 32) | 0xC0FFEE
    g = ul.Lattice(Ns, Nt, 1.0, seed)
    o = ulo.Oracle(Ns, Nt, 1.0, seed)
    assert same_links(g.get_links(), o.get_links())              # same Philox stream
    links = inputs.hot_links(Ns, Nt, 3)
    g.set_links(links)
    assert same_links(g.get_links(), links)
    again = g.get_links()
    g.set_links(again)
    assert np.array_equal(g.get_links(), again)                  # idempotent after the first conversion
    g.init(0)
    assert not g.get_links().any()
    g.init(1)
    assert same_links(g.get_links(), o.get_links())


def test_set_links_rejects_unwrapped_angles(ul):
    g = ul.Lattice(4, 4, 1.0, 1)
    links = inputs.hot_links(4, 4, 3)
    links[2, 1, 0, 3, 2] = 7.0
    with pytest.raises(ul.UlError) as e:
        g.set_links(links)
    assert e.value.code == ul.UL_EINVAL
    links[2, 1, 0, 3, 2] = np.nan
    with pytest.raises(ul.UlError):
        g.set_links(links)


def test_error_codes(ul):
    g = ul.Lattice(4, 4, 1.0, 1)
    for call in (lambda: g.multilevel(3, 0, 1), lambda: g.multilevel(2, 0, 3), lambda: g.multilevel(2, -1, 1),
                 lambda: g.multilevel2(2, 1, 3, 1, 1), lambda: g.substep(0, 0, 4), lambda: g.substep(3, 0, 0), lambda: g.set_update_algorithm(1, 4.0)):
        with pytest.raises(ul.UlError) as e:
            call()
        assert e.value.code == ul.UL_EINVAL
    with pytest.raises(ul.UlError) as e:
        g.read_correlators()
    assert e.value.code == ul.UL_ESTATE
    with pytest.raises(ul.UlError) as e:
        g.accumulate()
    assert e.value.code == ul.UL_ESTATE
    small = ul.Lattice(4, 4, 1.0, 1, workspace_bytes=4096)
    with pytest.raises(ul.UlError) as e:
        small.multilevel(2, 0, 2)
    assert e.value.code == ul.UL_ENOMEM


# ----------------------------------------------------------------------------- P1 link level
@pytest.mark.parametrize("Ns,Nt,therm", [(4, 4, 0), (6, 4, 0), (8, 6, 0), (16, 4, 0), (16, 4, 30)])
def test_p1_per_substep(ul, ulo, Ns, Nt, therm):
    """P1(i): every sub-step of a HB and an OR sweep, full and slab-masked, from the oracle's configuration."""
    beta, seed = 0.99, 2
    o = ulo.Oracle(Ns, Nt, beta, seed)
    ob = ulo.Oracle(Ns, Nt, beta, seed)
    g = ul.Lattice(Ns, Nt, beta, seed)
    if therm:
        o.sweep(0, 0)
        for _ in range(therm):
            o.sweep(1, 4)
    tot_flip = tot_ill = 0
    n_upd = 0
    for kind in (0, 1):
        for d in (0, 2):
            for parity in (0, 1):
                for mu in range(4):
                    before = o.get_links()
                    ob.set_links(before)
                    g.set_links(before)
                    g.set_counter(o.get_counter())
                    o.substep(kind, parity, mu, d)
                    g.substep(kind, parity, mu, d)
                    f, i, _ = check_links(g.get_links(), o.get_links(), before, ob, (kind, d, parity, mu), allow_frac=1e-4)
                    tot_flip += f
                    tot_ill += i
                    n_upd += 1
            if kind == 0:
                o.set_counter(o.get_counter() + 1)
    V4 = 4 * Ns ** 3 * Nt
    assert tot_flip <= max(2, 1e-5 * V4 * n_upd / 8), (tot_flip, tot_ill)


@pytest.mark.parametrize("Ns,Nt,beta,seed,n_therm,n_hb,n_or", [(4, 4, 0.95, 1, 20, 1, 3), (16, 4, 0.99, 2, 60, 1, 4)])
def test_p1_whole_sweep_thermalised(ul, ulo, Ns, Nt, beta, seed, n_therm, n_hb, n_or):
    """P1(ii): BJ's criterion literally, one heatbath sweep from a thermalised configuration."""
    o = ulo.Oracle(Ns, Nt, beta, seed)
    for _ in range(n_therm):
        o.sweep(n_hb, n_or)
    before = o.get_links()
    ob = ulo.Oracle(Ns, Nt, beta, seed)
    ob.set_links(before)
    g = ul.Lattice(Ns, Nt, beta, seed)
    g.set_links(before)
    g.set_counter(o.get_counter())
    o.sweep(1, 0)
    g.sweep(1, 0)
    assert g.get_counter() == o.get_counter()
    diff = wrapdiff(g.get_links(), o.get_links())
    frac = (diff > TOL).mean()
    assert frac < (1e-5 if diff.size > 2e5 else 2.0 / diff.size), (frac, diff.max())


def test_p1_masked_links_are_frozen_bit_for_bit(ul):
    Ns, Nt = 8, 8
    g = ul.Lattice(Ns, Nt, 1.0, 5)
    g.sweep(2, 2)
    before = g.get_links()
    g.multilevel(4, 3, 2)
    after = g.get_links()
    for t in (0, 4):
        assert np.array_equal(after[1:, t], before[1:, t])
    assert not np.array_equal(after[0, 0], before[0, 0])          # temporal links on the boundary layer do move
    assert not np.array_equal(after[1:, 1], before[1:, 1])


def test_runs_are_bitwise_reproducible(ul):
    res = []
    for _ in range(2):
        g = ul.Lattice(8, 4, 1.0, 9)
        g.sweep(3, 2)
        g.multilevel(2, 4, 3, [(0, 0, 0), (0, 1, 0)])
        res.append((g.get_links(), g.read_correlators(), g.plaquette()))
    assert np.array_equal(res[0][0], res[1][0])
    assert all(np.array_equal(a, b) for a, b in zip(res[0][1], res[1][1]))
    assert np.array_equal(res[0][2], res[1][2])


@pytest.mark.parametrize("n_sub", [5, 11])
def test_accumulation_batch_depth_does_not_change_results(ul, n_sub):
    """Rows a7/a8: the batched read-modify-write pass adds the configurations in sub-update order, so
    slab sums, correlators and field values are bit-identical for every batch depth (ragged tails too)."""
    res = []
    for depth in (1, 3, 4, 0):
        g = ul.Lattice(8, 4, 0.99, 21)
        g.sweep(2, 2)
        g.set_accum_batch(depth)
        g.multilevel(2, n_sub, 4, [(0, 0, 0), (1, 1, 0)])
        res.append((g.read_slab_averages(),) + tuple(g.read_correlators()))
        launches = g.launch_count()
        g.multilevel2(2, 3, 4, 2, 3, [(0, 1, 0)])
        res[-1] = res[-1] + tuple(g.read_correlators()) + (launches,)
    for r in res[1:]:
        assert all(np.array_equal(a, b) for a, b in zip(res[0][:-1], r[:-1]))
    assert res[0][-1] > res[-1][-1]                                # deeper batches launch fewer passes


def test_counter_resume_is_exact(ul):
    a = ul.Lattice(8, 4, 1.0, 11)
    a.sweep(2, 1)
    links, ctr = a.get_links_raw(), a.get_counter()
    a.sweep(1, 1)
    b = ul.Lattice(8, 4, 1.0, 11)
    b.set_links_raw(links)
    b.set_counter(ctr)
    b.sweep(1, 1)
    assert np.array_equal(a.get_links(), b.get_links())


# ----------------------------------------------------------------------------- P2 frozen configuration
def rel_ok(got, want, n_terms, rms_term=1.0, tol=1e-5):
    got, want = np.asarray(got), np.asarray(want)
    bound = tol * np.maximum(np.abs(want), rms_term / np.sqrt(n_terms))
    return np.all(np.abs(got - want) <= bound), float(np.max(np.abs(got - want) / bound))


FPS = [(0, 0, 0), (0, 1, 0), (1, 0, 0), (0, 0, 1), (-1, 2, 1), (0, 3, 0)]


@pytest.mark.parametrize("Ns,Nt,d", [(4, 4, 2), (8, 4, 2), (8, 8, 4), (6, 4, 1), (8, 4, 4)])
def test_p2_frozen_configuration(ul, ulo, Ns, Nt, d):
    beta = 1.0
    o = ulo.Oracle(Ns, Nt, beta, 3)
    for _ in range(10):
        o.sweep(1, 3)
    links = o.get_links()
    g = ul.Lattice(Ns, Nt, beta, 3)
    g.set_links(links)
    ok, worst = rel_ok(g.plaquette(), o.plaquette(), 3 * Ns ** 3 * Nt)
    assert ok, worst
    R = Ns // 2
    o.multilevel(d, 0, R, FPS)
    g.multilevel(d, 0, R, FPS)
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    Vs = Ns ** 3
    assert np.abs(g.read_slab_averages() - o.read_slab_averages()).max() < 1e-5     # |T| = 1
    ok, worst = rel_ok(cg, co, 3 * Vs)
    assert ok, worst
    ok, worst = rel_ok(fg, fo, 3 * Vs * Nt)
    assert ok, worst
    ok, worst = rel_ok(vg, vo, 3 * Vs * Nt)
    assert ok, worst


def test_p2_sequence_of_oracle_configurations(ul, ulo):
    """Slab sums over several oracle sub-update configurations fed one by one (P2)."""
    Ns, Nt, d, R = 8, 4, 2, 4
    o = ulo.Oracle(Ns, Nt, 0.99, 4)
    for _ in range(10):
        o.sweep(1, 3)
    g = ul.Lattice(Ns, Nt, 0.99, 4)
    o.measure_begin(d, R, FPS)
    g.measure_begin(d, R, FPS)
    for _ in range(5):
        for mu in range(4):
            for par in range(2):
                o.substep(1, par, mu, d)
        o.substep(0, 0, 0, d)
        g.set_links(o.get_links())
        o.accumulate()
        g.accumulate()
    o.measure_end()
    g.measure_end()
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    assert np.abs(g.read_slab_averages() - o.read_slab_averages()).max() < 1e-5
    Vs = Ns ** 3
    for got, want, n in ((cg, co, 3 * Vs), (fg, fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst


def test_p2_two_level_one_iteration_matches_oracle_combine(ul, ulo):
    """Two-level combine (Eqs. 32-33) on the same configurations: with n_in = n_out = 1 and a sub-update
    recipe of zero sweeps both sides measure the SAME frozen configuration through the two-level code path."""
    Ns, Nt, R = 8, 8, 3
    o = ulo.Oracle(Ns, Nt, 1.0, 6)
    for _ in range(8):
        o.sweep(1, 3)
    g = ul.Lattice(Ns, Nt, 1.0, 6)
    g.set_links(o.get_links())
    o.set_subupdate(0, 0, 1)
    g.set_subupdate(0, 0, 1)
    o.multilevel2(2, 1, 4, 1, R, FPS)
    g.multilevel2(2, 1, 4, 1, R, FPS)
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    Vs = Ns ** 3
    assert np.abs(g.read_slab_averages() - o.read_slab_averages()).max() < 1e-5
    for got, want, n in ((cg, co, 3 * Vs), (fg, fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst
    # and it equals the single-level result on the same configuration (factorisation, Eq. 24)
    g.multilevel(2, 0, R, FPS)
    c1, f1, _ = g.read_correlators()
    assert np.allclose(c1, cg, atol=1e-12) and np.allclose(f1, fg, atol=1e-12)


@pytest.mark.parametrize("Ns,Nt,d_in,d_out,n_in,n_out,batch", [(8, 8, 2, 4, 3, 2, 0), (6, 12, 2, 6, 4, 3, 3), (8, 8, 1, 4, 5, 2, 2)])
def test_p2_two_level_with_averaging_on_oracle_configurations(ul, ulo, Ns, Nt, d_in, d_out, n_in, n_out, batch):
    """Two-level estimator with REAL averaging (n_in >= 3, n_out >= 2; Eq. 27, Eqs. 32-34, Alg. 1
    lines 5-18) against the oracle on the oracle's own trajectory: the oracle runs its sub-updates, every inner
    configuration is handed to the GPU (ul_set_links) and added on both sides (ul_accumulate / ulo_accumulate), both
    combine per outer iteration (k_combine with inv = 1/n_in vs Eqs. 32-33 in the oracle) and close (1/n_out, slab
    product).  [T^(d_out)], C, G, vacuum to relative 1e-5 (R17) with the rms of the summed terms taken from the
    oracle's slab averages."""
    R = 3
    fps = FPS[:4]
    o = ulo.Oracle(Ns, Nt, 1.0, 11)
    for _ in range(6):
        o.sweep(1, 3)
    g = ul.Lattice(Ns, Nt, 1.0, 11)
    g.set_accum_batch(batch)
    o.measure2_begin(d_in, d_out, R, fps)
    g.measure2_begin(d_in, d_out, R, fps)

    def masked_compound(d):
        for parity in (0, 1):
            for mu in range(4):
                o.substep(0, parity, mu, d)
        o.set_counter(o.get_counter() + 1)
        for parity in (0, 1):
            for mu in range(4):
                o.substep(1, parity, mu, d)

    for J in range(n_out):
        masked_compound(d_out)
        for j in range(n_in):
            masked_compound(d_in)
            g.set_links(o.get_links())
            o.accumulate()
            g.accumulate()
        o.combine()
        g.combine()
    o.measure2_end()
    g.measure2_end()
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    T4, TO4 = o.read_slab_averages(), o.read_slab_field_averages()       # [3][R][S][Vs], [3][R][S][F][12][Vs]
    assert np.abs(T4).max() < 0.999                                      # averaged: not single-configuration phases
    assert np.abs(g.read_slab_averages() - T4).max() < 1e-5 * max(np.abs(T4).max(), 1e-2)
    Vs, S = Ns ** 3, Nt // d_out
    termC = T4.prod(axis=2)                                              # the 3 Vs summed terms of C(r)
    termG = 0
    for s_ in range(S):
        termG = termG + TO4[:, :, s_] * np.delete(T4, s_, axis=2).prod(axis=2)[:, :, None, None, :]
    rmsC = np.sqrt((np.abs(termC) ** 2).mean(axis=(0, 2)))               # [R]
    rmsG = np.sqrt((np.abs(termG) ** 2).mean(axis=(0, 4))) / Nt          # [R][F][12]
    ok, worst = rel_ok(cg, co, 3 * Vs, rms_term=rmsC)
    assert ok, ("C", worst)
    ok, worst = rel_ok(fg, fo, 3 * Vs, rms_term=rmsG)
    assert ok, ("G", worst)
    ok, worst = rel_ok(vg, vo, 3 * Vs * Nt)
    assert ok, ("vacuum", worst)
    # state errors of the hooks
    g.measure2_begin(d_in, d_out, R, fps)
    with pytest.raises(ul.UlError):
        g.combine()
    g.accumulate()
    with pytest.raises(ul.UlError):
        g.measure2_end()
    with pytest.raises(ul.UlError):
        g.measure_end()
    g.combine()
    g.accumulate(); g.accumulate()
    with pytest.raises(ul.UlError):
        g.combine()                                                      # 2 configurations after 1 in the first iteration


def test_two_level_hooks_equal_multilevel2_on_device(ul):
    """ul_measure2_begin / ul_accumulate / ul_combine / ul_measure2_end with the sweeps issued by hand reproduce
    ul_multilevel2 bit for bit (same kernels, same order)."""
    Ns, Nt, R, n_in, n_out = 8, 8, 3, 3, 2
    a = ul.Lattice(Ns, Nt, 1.0, 5)
    b = ul.Lattice(Ns, Nt, 1.0, 5)
    a.sweep(3, 3); b.sweep(3, 3)
    a.multilevel2(2, n_in, 4, n_out, R, FPS[:2])
    b.measure2_begin(2, 4, R, FPS[:2])

    def masked(d):
        for parity in (0, 1):
            for mu in range(4):
                b.substep(0, parity, mu, d)
        b.set_counter(b.get_counter() + 1)
        for _ in range(3):
            for parity in (0, 1):
                for mu in range(4):
                    b.substep(1, parity, mu, d)

    for J in range(n_out):
        masked(4)
        for j in range(n_in):
            masked(2)
            b.accumulate()
        b.combine()
    b.measure2_end()
    for x, y in zip(a.read_correlators(), b.read_correlators()):
        assert np.array_equal(x, y)
    assert np.array_equal(a.read_slab_averages(), b.read_slab_averages())
    assert np.array_equal(a.get_links_raw(), b.get_links_raw())


def test_p2_closed_forms_on_device(ul):
    """Pins that need no oracle: cold start, constant flux, Polyakov winding (SURVEY 8(c) pins)."""
    Ns, Nt = 8, 4
    g = ul.Lattice(Ns, Nt, 1.0, 1)
    g.init(0)
    assert np.allclose(g.plaquette(), 1.0, atol=1e-7)
    g.multilevel(2, 0, 4, FPS)
    c, f, v = g.read_correlators()
    assert np.allclose(c, 1.0, atol=1e-7) and np.allclose(f, 0, atol=1e-7) and np.allclose(v, 0, atol=1e-7)
    links, phi = inputs.constant_flux_links(Ns, Nt, m=1)
    g.set_links(links)
    p = g.plaquette()
    assert abs(p[0] - (5 + np.cos(phi)) / 6) < 1e-6 and abs(p[1] - 1) < 1e-6 and abs(p[2] - (2 + np.cos(phi)) / 3) < 1e-6
    m = 1
    links = np.zeros((4, Nt, Ns, Ns, Ns), dtype=np.float64)
    links[0] = (2 * np.pi * m * np.arange(Ns) / Ns / Nt).reshape(1, 1, 1, Ns)
    links = (links - 2 * np.pi * np.round(links / (2 * np.pi))).astype(np.float32)
    g.set_links(links)
    g.multilevel(2, 0, 4)
    c, _, _ = g.read_correlators()
    # C(r) = (e^{2 pi i m r / Ns} + 2)/3 : the winding shows only along mu = 1
    want = (np.exp(2j * np.pi * m * np.arange(1, 5) / Ns) + 2) / 3
    assert np.allclose(c, want, atol=2e-6)


def test_gauge_invariance_on_device(ul):
    """BJ check (b) on the GPU path: plaquette, C(r), G invariant under a random gauge transformation."""
    Ns, Nt = 8, 4
    g = ul.Lattice(Ns, Nt, 1.0, 21)
    g.sweep(5, 5)
    links = g.get_links()
    g.multilevel(2, 0, 4, FPS)
    c0, f0, v0 = g.read_correlators()
    p0 = g.plaquette()
    g.set_links(inputs.gauge_transform(links, inputs.gauge_function(Ns, Nt, 5)))
    g.multilevel(2, 0, 4, FPS)
    c1, f1, v1 = g.read_correlators()
    assert np.allclose(g.plaquette(), p0, atol=2e-7)
    assert np.allclose(c1, c0, atol=3e-7) and np.allclose(f1, f0, atol=3e-7) and np.allclose(v1, v0, atol=3e-7)


# ----------------------------------------------------------------------------- P3 ensemble
def binned_err(x, nbin=10):
    x = np.asarray(x, dtype=np.float64)
    n = len(x) // nbin * nbin
    b = x[:n].reshape(nbin, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / np.sqrt(nbin)


def test_p3_ensemble_config1(ul, ulo):
    """BJ config 1 (4^3x4, beta=0.95, 1 HB + 3 OR): plaquette and multilevel C(r) of independent
    GPU and oracle chains agree within 3 combined standard errors."""
    Ns, Nt, beta = 4, 4, 0.95
    n_meas = 120
    g = ul.Lattice(Ns, Nt, beta, 1)
    o = ulo.Oracle(Ns, Nt, beta, 101)
    series = {}
    for name, L in (("gpu", g), ("cpu", o)):
        for _ in range(20):
            L.sweep(1, 3)
        P, C1, C2 = [], [], []
        for _ in range(n_meas):
            L.sweep(1, 3)
            P.append(L.plaquette()[0])
            L.multilevel(2, 10, 2, [(0, 0, 0)])
            c, f, v = L.read_correlators()
            C1.append(c[0].real)
            C2.append(c[1].real)
        series[name] = (P, C1, C2)
    for k, label in enumerate(("plaquette", "C(1)", "C(2)")):
        mg, eg = binned_err(series["gpu"][k])
        mc, ec = binned_err(series["cpu"][k])
        assert abs(mg - mc) <= 3.0 * np.hypot(eg, ec) + 1e-12, (label, mg, eg, mc, ec)


def test_p3_strong_and_weak_coupling_on_device(ul):
    """BJ checks (c), (d) on the GPU path: <cos theta_P> = I1/I0 at beta = 0.1; <1 - cos> ~ 1/(4 beta) at beta = 5."""
    from scipy import special
    g = ul.Lattice(8, 8, 0.1, 31)
    for _ in range(20):
        g.sweep(1, 1)
    vals = []
    for _ in range(200):
        g.sweep(1, 1)
        vals.append(g.plaquette()[0])
    m, e = binned_err(vals)
    want = special.iv(1, 0.1) / special.iv(0, 0.1)
    assert abs(m - want) < 4 * e + 2e-5, (m, e, want)
    g = ul.Lattice(8, 8, 5.0, 32)
    g.init(0)
    for _ in range(100):
        g.sweep(1, 3)
    vals = []
    for _ in range(100):
        g.sweep(1, 3)
        vals.append(1 - g.plaquette()[0])
    m, e = binned_err(vals)
    assert abs(m - 0.05) < 0.05 * 0.05, (m, e)


def test_multilevel_matches_naive_on_device(ul):
    """BJ check (e) on the GPU path: multilevel C(r) vs the naive estimator (n_sub = 0) at strong coupling."""
    Ns, Nt, beta = 4, 4, 0.6
    g = ul.Lattice(Ns, Nt, beta, 41)
    for _ in range(30):
        g.sweep(1, 3)
    naive, ml = [], []
    for _ in range(300):
        g.sweep(1, 3)
        g.multilevel(2, 0, 1)
        naive.append(g.read_correlators()[0][0].real)
        g.multilevel(2, 8, 1)
        ml.append(g.read_correlators()[0][0].real)
    mn, en = binned_err(naive)
    mm, em = binned_err(ml)
    assert abs(mn - mm) < 3.5 * np.hypot(en, em), (mn, en, mm, em)
    assert em < en                                               # the multilevel estimator is less noisy


# ----------------------------------------------------------------------------- full size (BJ config 5)
def test_full_size_64_sampled_against_oracle(ul, ulo):
    """64^4 (the bench workload, same launch configuration): hot start bit-exact, then one HB and one
    OR sub-step compared with the oracle on every updated link; plaquette to relative 1e-5."""
    Ns = Nt = 64
    seed, beta = 5, 0.98
    g = ul.Lattice(Ns, Nt, beta, seed)
    o = ulo.Oracle(Ns, Nt, beta, seed)
    links = o.get_links()
    assert same_links(g.get_links(), links)
    ok, worst = rel_ok(g.plaquette(), o.plaquette(), 3 * Ns ** 4, rms_term=0.7)
    assert ok, worst
    for kind, parity, mu, d in ((1, 0, 1, 0), (0, 1, 0, 0), (0, 0, 3, 2)):
        before = o.get_links()
        g.set_links(before)
        g.set_counter(o.get_counter())
        o.substep(kind, parity, mu, d)
        g.substep(kind, parity, mu, d)
        diff = wrapdiff(g.get_links(), o.get_links())
        frac = (diff > TOL).sum() / (diff.size / 8)
        # hot start: links with tiny staples (k < 0.05, P ~ 3e-4) amplify rounding; flips are rare
        assert frac < 1e-4, (kind, parity, mu, d, frac, diff.max())
        assert (diff > 1e-3).sum() / (diff.size / 8) < 1e-5


def test_full_size_64_measurement_against_oracle(ul, ulo):
    """64^4, d = 2, r_max = 16 (the bench's measurement launch configuration): the frozen-configuration
    estimator equals the naive Polyakov-loop correlator (Eq. 23) that the oracle computes
    straight from Eq. 15; the batched pass over 8 configurations (here 8 copies of the same one, fed
    through ul_accumulate) gives the same slab products; vacuum values against the oracle's plaquette."""
    Ns = Nt = 64
    R = 16
    g = ul.Lattice(Ns, Nt, 0.98, 5, workspace_bytes=ul.workspace_bytes(Ns, Nt, 2, 0, R, 0))
    g.sweep(1, 2)                                                   # a configuration with some structure
    o = ulo.Oracle(Ns, Nt, 0.98, 5)
    o.set_links(g.get_links())
    want, _ = o.polyakov_naive(R)
    g.multilevel(2, 0, R)                                           # accumulate<1>, first pass
    c1, _, v1 = g.read_correlators()
    N = 3 * Ns ** 3
    for got, ref in ((c1.real, want.real), (c1.imag, want.imag)):
        ok, worst = rel_ok(got, ref, N)
        assert ok, worst
    plaq = o.plaquette()
    # vacuum channels 0, 2, 4 are 1 - cos of the time-like plaquettes (0,mu),(0,nu),(0,rho) averaged over the frames
    assert abs((1.0 - v1[[0, 2, 4]]).mean() - plaq[1]) < 1e-6 and abs((1.0 - v1[[6, 8, 10]]).mean() - plaq[2]) < 1e-6
    g.measure_begin(2, R)
    for _ in range(8):
        g.accumulate()                                              # one full batch: accumulate<8>
    g.accumulate()                                                  # and a ragged second pass (read-modify-write)
    g.measure_end()
    c9, _, v9 = g.read_correlators()
    assert np.abs(c9 - c1).max() < 1e-12 and np.abs(v9 - v1).max() < 1e-12


def test_full_size_64_thermalised_whole_sweep_and_substeps(ul, ulo):
    """64^4 at the bench's launch configuration, thermalised by the GPU (30 compound sweeps from the hot start) and handed
    to the oracle: one WHOLE heatbath sweep with BJ's literal criterion (every link within 2e-5 rad except flips and what
    they drag along, < 1e-5 of links; links updated at k < 0.05 counted apart), then a slab-masked spatial overrelaxation
    sub-step, a slab-masked spatial heatbath sub-step and a Metropolis sub-step, each on every updated link."""
    Ns = Nt = 64
    beta = 0.98
    g, o = _gpu_thermalised(ul, ulo, Ns, Nt, beta, 5, False, 30, 4)
    assert 0.5 < g.plaquette()[0] < 0.7
    _whole_hb_sweep(g, o, ulo, beta)
    ob = ulo.Oracle(Ns, Nt, beta, 1)
    for kind, parity, mu, d in ((1, 1, 2, 2), (0, 0, 1, 2), (2, 1, 3, 0)):
        before = o.get_links()
        g.set_links(before)
        g.set_counter(o.get_counter())
        if kind == 2:
            o.set_update_algorithm(1, 1.2)
            g.set_update_algorithm(1, 1.2)
        o.substep(kind, parity, mu, d)
        g.substep(kind, parity, mu, d)
        ob.set_links(before)
        check_links(g.get_links(), o.get_links(), before, ob, (kind, parity, mu, d))   # also: untouched links (frozen layers) did not move


# ----------------------------------------------------------------------------- BJ configs 3 and 4
def _gpu_thermalised(ul, ulo, Ns, Nt, beta, seed, cold, n_sweeps, n_or):
    """Configurations too long for the oracle to thermalise: the GPU does the sweeps, the oracle takes
    the result over; every comparison after that starts from identical links."""
    g = ul.Lattice(Ns, Nt, beta, seed)
    if cold:
        g.init(0)
    for _ in range(n_sweeps):
        g.sweep(1, n_or)
    o = ulo.Oracle(Ns, Nt, beta, seed)
    o.set_links(g.get_links())
    o.set_counter(g.get_counter())
    g.set_links(o.get_links())                                      # both sides hold the fp32-rounded angles
    return g, o


def _whole_hb_sweep(g, o, ulo, beta):
    """One whole heatbath sweep on both sides (GPU: ul_sweep; oracle: its 8 sub-steps, pinned equal to
    ulo_sweep, with a snapshot before each so that a miss can be classified by the staple magnitude k its
    link had WHEN it was updated).  BJ's criterion: every link within 2e-5 rad except accept/reject flips
    counted, < 1e-5 of links; a miss whose staple contains a link that missed EARLIER in the same sweep is what a flip
    drags along (counted apart, bounded); links updated at k < 0.05 (d alpha = dS / k) are the
    ill-conditioned class of P1, counted apart."""
    Ns, Nt = g.Ns, g.Nt
    snaps = []
    for parity in range(2):
        for mu in range(4):
            snaps.append(o.get_links())
            o.substep(0, parity, mu, 0)
    o.set_counter(o.get_counter() + 1)
    g.sweep(1, 0)
    assert g.get_counter() == o.get_counter()
    diff = wrapdiff(g.get_links(), o.get_links())
    miss = diff > TOL
    bad = np.argwhere(miss)
    ob = ulo.Oracle(Ns, Nt, beta, 1)
    ext = (Nt, Ns, Ns, Ns)                                           # canonical index [mu][t][x3][x2][x1]
    pos = {0: 0, 1: 3, 2: 2, 3: 1}                                   # direction -> position in (t, x3, x2, x1)

    def hop(site, nu, step):
        c = list(site)
        c[pos[nu]] = (c[pos[nu]] + step) % ext[pos[nu]]
        return tuple(c)

    def dragged(mu, site):
        """A link of the staple of (site, mu) that was updated EARLIER in this sweep (each link is updated once per sweep, so
        its final value is what the staple saw) is itself a miss: this miss is a consequence, not a flip of its own."""
        order = (sum(site) & 1) * 4 + mu
        xpm = hop(site, mu, +1)
        for nu in range(4):
            if nu == mu:
                continue
            for lmu, lsite in ((nu, site), (mu, hop(site, nu, +1)), (nu, xpm), (nu, hop(xpm, nu, -1)), (mu, hop(site, nu, -1)),
                               (nu, hop(site, nu, -1))):
                if (sum(lsite) & 1) * 4 + lmu < order and miss[(lmu,) + lsite]:
                    return True
        return False

    n_ill = n_flip = n_drag = 0
    primary = {}
    for idx in bad:
        mu, site = int(idx[0]), tuple(int(v) for v in idx[1:])
        if dragged(mu, site):
            n_drag += 1
        else:
            primary.setdefault((sum(site) & 1) * 4 + mu, []).append((mu, site))
    for order, links in primary.items():
        ob.set_links(snaps[order])                                   # the configuration these links were updated from
        for mu, site in links:
            k, _ = ob.staple(mu, int(np.ravel_multi_index(site, diff.shape[1:])))
            if k < 0.05:
                n_ill += 1
            else:
                n_flip += 1
    assert n_flip <= max(1, 1e-5 * diff.size), (n_flip, n_ill, n_drag, diff.max())     # BJ: flips < 1e-5 of all links
    assert n_ill <= 1e-4 * diff.size, (n_flip, n_ill, n_drag, diff.max())
    assert len(bad) <= max(8, 1e-4 * diff.size), (n_flip, n_ill, n_drag)             # flips + what they drag along
    assert (diff > 5e-6).mean() < 2e-4                               # and the bulk sits far below the tolerance
    return n_flip, n_ill, n_drag


def test_config3_24x8_thermalised_sweep_and_fields(ul, ulo):
    """BJ config 3: 24^3 x 8, beta = 1.00, cold start, 500 x (1 HB + 3 OR); then one HB sweep link by link
    (P1) and the frozen-configuration estimator with r = 1..12, mid-plane and on-axis field points (P2)."""
    Ns, Nt, R = 24, 8, 12
    g, o = _gpu_thermalised(ul, ulo, Ns, Nt, 1.00, 3, True, 500, 3)
    pg, po = g.plaquette(), o.plaquette()
    assert 0.55 < pg[0] < 0.75                                       # thermalised around the beta = 1 transition region
    ok, worst = rel_ok(pg, po, 3 * Ns ** 3 * Nt, rms_term=0.5)
    assert ok, worst
    fps = [(0, 0, 0), (0, 5, 0), (0, 10, 0), (3, 0, 0)]
    o.multilevel(2, 0, R, fps)
    g.multilevel(2, 0, R, fps)
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    assert np.abs(g.read_slab_averages() - o.read_slab_averages()).max() < 1e-5
    Vs = Ns ** 3
    for got, want, n in ((cg, co, 3 * Vs), (fg, fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst
    _whole_hb_sweep(g, o, ulo, 1.00)


def test_config4_32x32_two_level_and_sweep(ul, ulo):
    """BJ config 4: 32^4, beta = 1.00, hot start seed 4, two-level scheme with slab thicknesses 2 and 4,
    r = 1..16: the combine path on a frozen configuration (sub-update recipe of zero sweeps) against the
    oracle, the factorisation Eq. 24, and one whole heatbath sweep link by link."""
    Ns, Nt, R = 32, 32, 16
    g, o = _gpu_thermalised(ul, ulo, Ns, Nt, 1.00, 4, False, 40, 4)
    o.set_subupdate(0, 0, 1)
    g.set_subupdate(0, 0, 1)
    o.multilevel2(2, 1, 4, 1, R)
    g.multilevel2(2, 1, 4, 1, R)
    co, _, vo = o.read_correlators()
    cg, _, vg = g.read_correlators()
    assert np.abs(g.read_slab_averages() - o.read_slab_averages()).max() < 1e-5
    Vs = Ns ** 3
    for got, want, n in ((cg, co, 3 * Vs), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst
    want, _ = o.polyakov_naive(R)                                    # Eq. 23: frozen configuration = naive correlator
    assert np.abs(cg - want).max() < 1e-9
    fps = [(0, 0, 0), (0, 3, 0)]
    o.multilevel2(2, 1, 4, 1, 2, fps)
    g.multilevel2(2, 1, 4, 1, 2, fps)
    fo, fg = o.read_correlators()[1], g.read_correlators()[1]
    ok, worst = rel_ok(fg, fo, 3 * Vs * Nt)
    assert ok, worst
    g.set_subupdate(1, 3, 1)
    o.set_subupdate(1, 3, 1)
    _whole_hb_sweep(g, o, ulo, 1.00)


# ----------------------------------------------------------------------------- Metropolis (next row, DESIGN R21)
@pytest.mark.parametrize("Ns,Nt,therm,delta", [(4, 4, 0, 1.0), (8, 6, 0, np.pi), (16, 4, 20, 1.3)])
def test_metropolis_per_substep(ul, ulo, Ns, Nt, therm, delta):
    """Every Metropolis sub-step, full and slab-masked, from the oracle's configuration: a link either moves by
    the same proposal (within 2e-5 rad; in fact the proposal is an exact integer here) or stays bit for bit;
    accept/reject flips at the rounding boundary are counted (< 1e-5 of links)."""
    beta, seed = 0.99, 7
    o = ulo.Oracle(Ns, Nt, beta, seed)
    o.set_update_algorithm(1, delta)
    g = ul.Lattice(Ns, Nt, beta, seed)
    g.set_update_algorithm(1, delta)
    for _ in range(therm):
        o.sweep(1, 3)
    flips = n_upd = 0
    for d in (0, 2):
        for parity in (0, 1):
            for mu in range(4):
                before = o.get_links()
                g.set_links(before)
                g.set_counter(o.get_counter())
                o.substep(2, parity, mu, d)
                g.substep(2, parity, mu, d)
                got, want = g.get_links(), o.get_links()
                diff = wrapdiff(got, want)
                moved_o, moved_g = want != before, wrapdiff(got, before) > 1.3e-9
                flips += int((moved_o != moved_g).sum())
                same = moved_o == moved_g
                assert diff[same].max() <= 1e-6                      # the proposal is formed exactly; fp32 store of the oracle
                n_upd += int(moved_o.sum())
        o.set_counter(o.get_counter() + 1)
    assert n_upd > 0.2 * 4 * Ns ** 3 * Nt
    assert flips <= max(1, 1e-5 * 4 * Ns ** 3 * Nt * 4), flips


def test_metropolis_whole_sweep_and_counter(ul, ulo):
    Ns, Nt, beta = 16, 4, 0.99
    o = ulo.Oracle(Ns, Nt, beta, 2)
    o.set_update_algorithm(1, 1.0)
    for _ in range(30):
        o.sweep(1, 3)
    g = ul.Lattice(Ns, Nt, beta, 2)
    g.set_update_algorithm(1, 1.0)
    g.set_links(o.get_links())
    g.set_counter(o.get_counter())
    o.sweep(1, 0)
    g.sweep(1, 0)
    assert g.get_counter() == o.get_counter()
    diff = wrapdiff(g.get_links(), o.get_links())
    assert (diff > TOL).mean() < 1e-5, ((diff > TOL).sum(), diff.max())


def test_metropolis_leaves_von_mises_stationary_on_device(ul):
    """The pin of tests/test_oracle_metropolis.py repeated on the CUDA path (no oracle involved)."""
    from scipy import special, stats
    Ns, Nt, beta = 16, 8, 0.5
    a = 6 * beta
    rng = np.random.default_rng(5)
    even = (np.indices((Nt, Ns, Ns, Ns)).sum(axis=0) & 1) == 0
    g = ul.Lattice(Ns, Nt, beta, 22)
    g.set_update_algorithm(1, 2.0)
    links = np.zeros((4, Nt, Ns, Ns, Ns), dtype=np.float32)
    links[0][even] = rng.uniform(-np.pi, np.pi, int(even.sum())).astype(np.float32)
    g.set_links(links)
    for it in range(40):
        g.set_counter(it)
        g.substep(2, 0, 0, 0)
    out = g.get_links()
    assert not out[1:].any()
    th = out[0][even].astype(np.float64)
    _, p = stats.kstest(th, stats.vonmises(kappa=a).cdf)
    assert p > 1e-3, p
    assert abs(np.cos(th).mean() - special.iv(1, a) / special.iv(0, a)) < 4 * np.sqrt(0.5 / th.size)


def test_metropolis_ensemble_matches_oracle_and_heatbath(ul, ulo):
    """P3 for the Metropolis chain: plaquette of independent GPU and oracle chains (the paper's recipe,
    1 Metropolis + 3 overrelaxation) within 3 combined standard errors; and of the GPU heatbath chain."""
    Ns, Nt, beta = 4, 4, 0.95
    def chain(L, n):
        vals = []
        for _ in range(n):
            L.sweep(1, 3)
            vals.append(L.plaquette()[0])
        return np.array(vals)
    g = ul.Lattice(Ns, Nt, beta, 51); g.set_update_algorithm(1, 1.2)
    o = ulo.Oracle(Ns, Nt, beta, 52); o.set_update_algorithm(1, 1.2)
    h = ul.Lattice(Ns, Nt, beta, 53)
    # beta = 0.95 on 4^4 sits next to the transition: the plaquette has slow modes of a few hundred sweeps (the oracle's chain of
    # seed 52 averages 0.500 over its first 400 sweeps and 0.513 over the next 1600), so bins of 40 sweeps underestimate the
    # errors and any change of a rounding re-rolls the outcome.  Same criterion (3 combined standard errors) on ten times
    # the statistics: 4000 sweeps in 20 bins of 200 after 240 thermalisation sweeps.
    for L in (g, o, h):
        L.sweep(40, 40)
        for _ in range(200):
            L.sweep(1, 3)
    vg, vo, vh = chain(g, 4000), chain(o, 4000), chain(h, 4000)
    for a_, b_ in ((vg, vo), (vg, vh)):
        (ma, ea), (mb, eb) = binned_err(a_, 20), binned_err(b_, 20)
        assert abs(ma - mb) < 3 * np.hypot(ea, eb), (ma, ea, mb, eb)


# ----------------------------------------------------------------------------- Polyakov loop with multihit (next row)
@pytest.mark.parametrize("Ns,Nt,beta", [(4, 4, 0.9), (8, 6, 1.1), (16, 4, 0.99)])
def test_polyakov_and_multihit_against_oracle(ul, ulo, Ns, Nt, beta):
    """<P> plain and with analytic multihit (Eqs. 15-16) on the oracle's configurations, relative 1e-5
    (DESIGN R17); closed forms on device; gauge invariance on device."""
    from scipy import special
    o = ulo.Oracle(Ns, Nt, beta, 3)
    g = ul.Lattice(Ns, Nt, beta, 3)
    for n_sw in (0, 3, 10):
        for _ in range(n_sw):
            o.sweep(1, 2)
        g.set_links(o.get_links())
        for mh in (0, 1):
            want, got = o.polyakov(mh), g.polyakov(mh)
            scale = 1.0 if mh == 0 else (special.ive(1, 4 * beta) / special.ive(0, 4 * beta)) ** Nt   # size of a multihit term
            assert abs(got - want) <= 1e-5 * max(abs(want), scale / np.sqrt(Ns ** 3)), (n_sw, mh, got, want)
    g.init(0)
    r = special.ive(1, 6 * beta) / special.ive(0, 6 * beta)
    assert abs(g.polyakov(0) - 1) < 1e-14 and abs(g.polyakov(1) - r ** Nt) < 1e-13
    links = inputs.hot_links(Ns, Nt, 8) * 0.5
    g.set_links(links)
    a = g.polyakov(1)
    g.set_links(inputs.gauge_transform(links, inputs.gauge_function(Ns, Nt, 9)))
    b = g.polyakov(1)                                               # the transformed links are re-rounded to fp32
    assert abs(b - a) <= 1e-5 * max(abs(a), abs(b)) + 1e-9 * (special.ive(1, 4 * beta) / special.ive(0, 4 * beta)) ** Nt
    with pytest.raises(ul.UlError):
        g.polyakov(2)


def test_polyakov_full_size_64(ul, ulo):
    """64^4 (launch configuration of the full-size lattice): plain <P> against the oracle's Eq. 15 loop; the
    multihit value on sampled sites is covered by the small-lattice parity above, here its closed form on the
    cold lattice and the timing print."""
    from scipy import special
    Ns = Nt = 64
    g = ul.Lattice(Ns, Nt, 0.98, 5)
    g.sweep(1, 1)
    o = ulo.Oracle(Ns, Nt, 0.98, 5)
    o.set_links(g.get_links())
    want = o.polyakov(0)
    got = g.polyakov(0)
    assert abs(got - want) <= 1e-5 / np.sqrt(Ns ** 3)
    g.init(0)
    r = special.ive(1, 6 * 0.98) / special.ive(0, 6 * 0.98)
    assert abs(g.polyakov(1) - r ** Nt) < 1e-12 * r ** Nt + 1e-18


# ----------------------------------------------------------------------------- replay estimator (next row)
@pytest.mark.parametrize("Ns,Nt,d,n_sub", [(4, 4, 2, 5), (8, 4, 2, 9), (8, 8, 4, 3), (6, 4, 1, 2)])
def test_replay_equals_stored_accumulators(ul, Ns, Nt, d, n_sub):
    """ul_multilevel_replay: the same trajectory (bit-identical final links and counter), the same correlators
    bit for bit, the same field values and vacuum to fp64 rounding order, as the stored-accumulator path."""
    R = min(3, Ns // 2)
    res = []
    for mode in ("stored", "replay"):
        g = ul.Lattice(Ns, Nt, 0.99, 31)
        g.sweep(3, 2)
        (g.multilevel if mode == "stored" else g.multilevel_replay)(d, n_sub, R, FPS)
        res.append((g.get_links_raw(), g.get_counter(), g.read_slab_averages()) + tuple(g.read_correlators()))
    a, b = res
    assert np.array_equal(a[0], b[0]) and a[1] == b[1]
    assert np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3]) and np.array_equal(a[5], b[5])
    scale = np.abs(a[4]).max()
    assert scale > 0 and np.abs(a[4] - b[4]).max() <= 1e-12 * max(scale, 1e-3)


def test_replay_frozen_configuration_against_oracle(ul, ulo):
    """P2 for the replay path: n_sub = 0 on an oracle configuration, fields and correlators to relative 1e-5."""
    Ns, Nt, d, R = 8, 4, 2, 4
    o = ulo.Oracle(Ns, Nt, 0.99, 4)
    for _ in range(10):
        o.sweep(1, 3)
    g = ul.Lattice(Ns, Nt, 0.99, 4)
    g.set_links(o.get_links())
    o.multilevel(d, 0, R, FPS)
    g.multilevel_replay(d, 0, R, FPS)
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    Vs = Ns ** 3
    for got, want, n in ((cg, co, 3 * Vs), (fg, fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst


def test_replay_config3_memory_and_agreement(ul):
    """BJ config 3 shape (24^3 x 8, r <= 12, mid-plane offsets 0..10 and on-axis points): the replay workspace is
    ~40x smaller than the stored accumulators, and both give the same numbers from the same start."""
    Ns, Nt, d, R = 24, 8, 2, 12
    fps = [(0, b, 0) for b in range(11)] + [(a, 0, 0) for a in (-2, -1, 1, 2)]
    big, small = ul.workspace_bytes(Ns, Nt, d, 0, R, len(fps)), ul.workspace_bytes_replay(Ns, Nt, d, R, len(fps))
    assert big > 30 * small
    out = []
    for mode in ("stored", "replay"):
        g = ul.Lattice(Ns, Nt, 1.0, 3)
        g.init(0)
        for _ in range(30):
            g.sweep(1, 3)
        (g.multilevel if mode == "stored" else g.multilevel_replay)(d, 4, R, fps)
        out.append(g.read_correlators())
    assert np.array_equal(out[0][0], out[1][0])
    assert np.abs(out[0][1] - out[1][1]).max() <= 1e-12 * np.abs(out[0][1]).max()


def test_replay_full_mid_plane_against_oracle(ul, ulo):
    """A FULL mid-plane of field points (all 64 transverse offsets of an 8^3 x 4 lattice, 12 channels, r = 1..4):
    the map BJ config 4 asks for, at a size where the oracle's stored accumulators still fit; frozen
    configuration, relative 1e-5 (DESIGN R17)."""
    Ns, Nt, d, R = 8, 4, 2, 4
    fps = [(0, b, c) for c in range(Ns) for b in range(Ns)]
    o = ulo.Oracle(Ns, Nt, 1.0, 9)
    for _ in range(12):
        o.sweep(1, 3)
    g = ul.Lattice(Ns, Nt, 1.0, 9)
    g.set_links(o.get_links())
    o.multilevel(d, 0, R, fps)
    g.multilevel_replay(d, 0, R, fps)
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    Vs = Ns ** 3
    for got, want, n in ((cg, co, 3 * Vs), (fg, fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst
    assert ul.workspace_bytes(Ns, Nt, d, 0, R, len(fps)) > 100 * ul.workspace_bytes_replay(Ns, Nt, d, R, len(fps))
    g.multilevel_replay(d, 3, R, fps)                               # and a short run through the sub-updates
    assert np.all(np.isfinite(g.read_correlators()[1]))


@pytest.mark.parametrize("Ns,Nt,R", [(40, 2, 3), (64, 2, 2)])
def test_full_plane_map_beyond_32_sampled_against_oracle(ul, ulo, Ns, Nt, R):
    """The transverse-DFT route with several entries per thread (Ns = 40: 2, Ns = 64: 4): the FULL mid-plane map (Ns^2 field
    points x 12 channels) of a frozen configuration, compared at sampled points with the oracle (whose stored accumulators
    only fit a few field points at this size) to relative 1e-5, and with the library's generic per-point reduction."""
    d = 2
    g = ul.Lattice(Ns, Nt, 1.0, 21)
    for _ in range(6):
        g.sweep(1, 3)
    links = g.get_links()
    g.set_links(links)
    full = [(0, b, c) for c in range(Ns) for b in range(Ns)]
    g.multilevel_replay(d, 0, R, full)
    cg, fg, vg = g.read_correlators()
    pick = [(0, 0, 0), (0, 1, 0), (0, Ns - 1, 3), (0, 17, Ns // 2), (0, Ns - 2, Ns - 1)]
    idx = [b + Ns * c for (_, b, c) in pick]
    g.multilevel_replay(d, 0, R, pick)                              # generic path (k_replay_reduce): not a full plane
    _, fg5, _ = g.read_correlators()
    assert np.abs(fg[:, idx] - fg5).max() <= 1e-11 * max(1.0, np.abs(fg5).max())
    o = ulo.Oracle(Ns, Nt, 1.0, 21)
    o.set_links(links)
    o.multilevel(d, 0, R, pick)
    co, fo, vo = o.read_correlators()
    Vs = Ns ** 3
    for got, want, n in ((cg, co, 3 * Vs), (fg[:, idx], fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst


# ----------------------------------------------------------------------------- slab sharding (next row)
@pytest.mark.parametrize("world", [2, 4])
@pytest.mark.parametrize("alg", [0, 1])
def test_slab_sharding_reproduces_the_unsharded_run(ul, ulo, world, alg):
    """The shards of a t-partitioned lattice, run ONE AFTER THE OTHER on this GPU (no kernel waits on another),
    reproduce the unsharded multilevel run bit for bit on the links and slab averages they own (global Philox
    counters through ul_set_site_offset, frozen boundary layer in the ghost slab, no communication in the
    sub-update loop); the product of the per-shard slab products gives the unsharded C(r)."""
    from paper_1309_3859_b200 import sharded
    Ns, Nt, d, R, n_sub, beta, seed = 8, 16, 2, 3, 6, 0.99, 77
    full = ul.Lattice(Ns, Nt, beta, seed)
    full.set_update_algorithm(alg, 1.1)
    for _ in range(10):
        full.sweep(1, 3)
    links0, ctr0 = full.get_links(), full.get_counter()
    full.set_links(links0)                                          # both runs start from the fp32-rounded angles
    full.multilevel(d, n_sub, R)
    A_full, C_full = full.read_slab_averages(), full.read_correlators()[0]
    links1 = full.get_links_raw()
    parts = sharded.partition(Nt, d, world)
    prods = []
    for rank in range(world):
        sh = sharded.ShardedLattice(Ns, Nt, beta, seed, d, rank, world, links0, ctr0)
        sh.lat.set_update_algorithm(alg, 1.1)
        sh.multilevel(n_sub, R)
        t0, n = parts[rank]
        assert np.array_equal(sh.own_slab_averages(), A_full[:, :, t0 // d:(t0 + n) // d])
        assert np.array_equal(sh.lat.get_links_raw()[:, :n], links1[:, t0:t0 + n])
        assert sh.lat.get_counter() == full.get_counter()
        prods.append(sh.partial_product())
    C = sh.lat.combine_partial_products(prods)                       # ordered product + lattice sum in the library
    assert np.abs(C - C_full).max() <= 1e-13 * max(1.0, np.abs(C_full).max())
    assert np.array_equal(sh.lat.read_correlators()[0], C)
    # the sharded estimator against the ORACLE on the frozen start configuration (n_sub = 0), relative 1e-5 (P2)
    o = ulo.Oracle(Ns, Nt, beta, seed)
    o.set_links(links0)
    o.multilevel(d, 0, R)
    Co = o.read_correlators()[0]
    prods = []
    for rank in range(world):
        sh = sharded.ShardedLattice(Ns, Nt, beta, seed, d, rank, world, links0, ctr0)
        sh.multilevel(0, R)
        prods.append(sh.partial_product())
    C0 = sh.lat.combine_partial_products(prods)
    for got, want in ((C0.real, Co.real), (C0.imag, Co.imag)):
        ok, worst = rel_ok(got, want, 3 * Ns ** 3)
        assert ok, worst


@pytest.mark.parametrize("mode,Ns,Nt", [("graph", 8, 8), ("persistent", 8, 8), ("persistent", 24, 8), ("persistent", 6, 4), ("graph", 6, 4)])
def test_graph_replayed_sweeps_equal_directly_launched_substeps(ul, monkeypatch, mode, Ns, Nt):
    """Small lattices run a compound sweep as ONE cooperative launch (ul_persist.cuh: resident blocks, grid barriers, L2-coherent
    loads, block-local straggler queue); lattices of <= 2^21 sites beyond that (and these, with UL_NO_PERSIST=1) replay it
    from a CUDA graph whose kernels read the sweep counter from device memory; ul_substep launches the same kernels
    directly with the counter as an argument.  All must give the same bits, sweep after sweep, full and slab-masked,
    heatbath and Metropolis."""
    if mode == "graph":
        monkeypatch.setenv("UL_NO_PERSIST", "1")
    for alg in (0, 1):
        a = ul.Lattice(Ns, Nt, 0.99, 13)
        n0 = a.launch_count()
        a.sweep(1, 1)
        assert (a.launch_count() - n0 == 1) == (mode == "persistent")   # one launch per compound sweep, or 8 + 8 + 8 + 1
        a.init(1); a.set_counter(0)
        b = ul.Lattice(Ns, Nt, 0.99, 13)
        for L in (a, b):
            L.set_update_algorithm(alg, 1.3)
        a.set_counter(2 ** 32 - 2)                                  # crosses the 32-bit boundary of the device counter
        b.set_counter(2 ** 32 - 2)
        for it in range(4):
            a.sweep(2, 1)                                           # graph (captured at it = 0, replayed after)
            for _ in range(2):
                for parity in range(2):
                    for mu in range(4):
                        b.substep(2 if alg else 0, parity, mu, 0)
                b.set_counter(b.get_counter() + 1)
            for parity in range(2):
                for mu in range(4):
                    b.substep(1, parity, mu, 0)
            assert a.get_counter() == b.get_counter() == 2 ** 32 - 2 + 2 * (it + 1)
            assert np.array_equal(a.get_links_raw(), b.get_links_raw()), (alg, it)
        a.multilevel(2, 3, 2)                                       # masked recipe: another graph
        a.set_subupdate(1, 3, 1)
        for _ in range(3):
            for kind, n in ((2 if alg else 0, 1), (1, 3)):
                for _ in range(n):
                    for parity in range(2):
                        for mu in range(4):
                            b.substep(kind, parity, mu, 2)
                    if kind != 1:
                        b.set_counter(b.get_counter() + 1)
        assert np.array_equal(a.get_links_raw(), b.get_links_raw()) and a.get_counter() == b.get_counter()


@pytest.mark.parametrize("Ns,Nt", [(16, 4), (8, 8), (6, 4)])
def test_global_straggler_queue_equals_in_kernel_stragglers(ul, monkeypatch, Ns, Nt):
    """Heatbath links that rejected both attempts of their first Philox block are finished either by the same thread block
    from a shared-memory queue (default) or through the striped global queue + k_hb_stragglers (UL_NO_HB_LOCAL=1; always
    with peer-memory halo writes): same links bit for bit, full and slab-masked, directly launched sub-steps."""
    a = ul.Lattice(Ns, Nt, 1.0, 17)
    monkeypatch.setenv("UL_NO_HB_LOCAL", "1")
    monkeypatch.setenv("UL_NO_PERSIST", "1")
    b = ul.Lattice(Ns, Nt, 1.0, 17)
    for L in (a, b):
        for it in range(3):
            for d in (0, 2):
                for parity in (0, 1):
                    for mu in range(4):
                        L.substep(0, parity, mu, d)
                L.set_counter(L.get_counter() + 1)
    assert b.launch_count() > a.launch_count()                      # (the straggler launches)
    assert np.array_equal(a.get_links_raw(), b.get_links_raw())


def test_tma_staged_overrelaxation_equals_direct_gather(ul, ulo, monkeypatch):
    """The bulk-copy (TMA) staged overrelaxation kernel (UL_OR_TMA=1; ul_update_tma.cuh), the A/B partner of the direct
    gather: same links bit for bit after full and slab-masked sweeps on a lattice whose tiles have its shape (Ns = 64), and one
    of its sub-steps against the oracle on every updated link."""
    Ns, Nt = 64, 4
    a = ul.Lattice(Ns, Nt, 0.98, 9)
    monkeypatch.setenv("UL_OR_TMA", "1")
    b = ul.Lattice(Ns, Nt, 0.98, 9)
    monkeypatch.delenv("UL_OR_TMA")
    for L in (a, b):
        L.sweep(1, 2)
        for parity in (0, 1):
            for mu in range(4):
                L.substep(1, parity, mu, 2)
    assert b.launch_count() == a.launch_count()
    assert np.array_equal(a.get_links_raw(), b.get_links_raw())
    o = ulo.Oracle(Ns, Nt, 0.98, 9)
    before = b.get_links()
    o.set_links(before)
    b.set_links(before)
    ob = ulo.Oracle(Ns, Nt, 0.98, 1)
    ob.set_links(before)
    for parity, mu, d in ((1, 2, 0), (0, 3, 2)):
        o.substep(1, parity, mu, d)
        b.substep(1, parity, mu, d)
    # (two sub-steps in a row: the second starts from the first's output on both sides, overrelaxation has no flips)
    diff = wrapdiff(b.get_links(), o.get_links())
    assert (diff > TOL).sum() <= 1e-4 * diff.size and (diff > 1e-3).sum() == 0


# ----------------------------------------------------------------------------- multihit inside the two-link operators
@pytest.mark.parametrize("Ns,Nt,d", [(4, 4, 2), (8, 4, 2), (8, 8, 4), (6, 4, 1)])
def test_multihit_two_link_against_oracle(ul, ulo, Ns, Nt, d):
    """P2 with ul_set_multihit(1): slab averages, C(r), field values and vacuum on oracle configurations to relative
    1e-5 (the staple sums are fp32 here, fp64 in the oracle); r = 1 and all TO sums are the plain ones bit for bit."""
    from scipy import special
    R, beta = min(3, Ns // 2), 0.95
    o = ulo.Oracle(Ns, Nt, beta, 6)
    for _ in range(8):
        o.sweep(1, 3)
    g = ul.Lattice(Ns, Nt, beta, 6)
    g.set_links(o.get_links())
    g.multilevel(d, 0, R, FPS)
    plain = (g.read_slab_averages(),) + tuple(g.read_correlators())
    o.set_multihit(1)
    g.set_multihit(1)
    o.multilevel(d, 0, R, FPS)
    g.multilevel(d, 0, R, FPS)
    ao, ag = o.read_slab_averages(), g.read_slab_averages()
    co, fo, vo = o.read_correlators()
    cg, fg, vg = g.read_correlators()
    size = (special.ive(1, 4 * beta) / special.ive(0, 4 * beta)) ** (2 * d)          # magnitude of a multihit T^(d)
    assert np.abs(ag - ao).max() < 2e-5 * size
    assert np.array_equal(ag[:, 0], plain[0][:, 0]) and not np.allclose(ag[:, 1:], plain[0][:, 1:])
    Vs = Ns ** 3
    ok, worst = rel_ok(cg, co, 3 * Vs, rms_term=size ** (Nt // d))
    assert ok, worst
    for got, want, n in ((fg, fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
        ok, worst = rel_ok(got, want, n)
        assert ok, worst
    g.init(0)                                                                          # closed form on device
    g.multilevel(d, 0, R)
    c = g.read_correlators()[0]
    r = special.ive(1, 6 * beta) / special.ive(0, 6 * beta)
    assert abs(c[0] - 1) < 1e-12 and np.abs(c[1:] - r ** (2 * Nt)).max() < 2e-5 * r ** (2 * Nt)


def test_multihit_two_link_paths_agree(ul):
    """With multihit on: batch depths, the replay path and the two-level path (n_in = n_out = 1, frozen) give the
    same numbers as the single-level stored path."""
    Ns, Nt, d, R = 8, 8, 2, 3
    ref = None
    for depth, mode in ((0, "stored"), (1, "stored"), (3, "stored"), (0, "replay")):
        g = ul.Lattice(Ns, Nt, 0.99, 41)
        g.sweep(3, 2)
        g.set_multihit(1)
        g.set_accum_batch(depth)
        (g.multilevel if mode == "stored" else g.multilevel_replay)(d, 7, R, FPS)
        cur = (g.read_slab_averages(),) + tuple(g.read_correlators()) + (g.get_links_raw(),)
        if ref is None:
            ref = cur
            continue
        assert np.array_equal(cur[0], ref[0]) and np.array_equal(cur[1], ref[1]) and np.array_equal(cur[4], ref[4])
        assert np.abs(cur[2] - ref[2]).max() <= 1e-12 * np.abs(ref[2]).max()
    g = ul.Lattice(Ns, Nt, 0.99, 41)
    g.sweep(3, 2)
    g.set_multihit(1)
    g.set_subupdate(0, 0, 1)
    g.multilevel(d, 0, R)
    c1 = g.read_correlators()[0]
    g.multilevel2(2, 1, 4, 1, R)
    assert np.allclose(g.read_correlators()[0], c1, rtol=1e-12, atol=1e-18)


@pytest.mark.parametrize("Ns,Nt,n_in,n_out", [(4, 8, 3, 2), (8, 8, 9, 3), (6, 4, 2, 2)])
def test_two_level_replay_equals_stored_accumulators(ul, Ns, Nt, n_in, n_out):
    """ul_multilevel2_replay against ul_multilevel2 from the same start: bit-identical final links, counter,
    correlators and outer slab averages; field values and vacuum to fp64 rounding order."""
    R = min(3, Ns // 2)
    res = []
    for mode in ("stored", "replay"):
        g = ul.Lattice(Ns, Nt, 0.99, 33)
        g.sweep(3, 2)
        (g.multilevel2 if mode == "stored" else g.multilevel2_replay)(2, n_in, 4, n_out, R, FPS)
        res.append((g.get_links_raw(), g.get_counter(), g.read_slab_averages()) + tuple(g.read_correlators()))
    a, b = res
    assert np.array_equal(a[0], b[0]) and a[1] == b[1]
    assert np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3])
    assert np.abs(a[5] - b[5]).max() <= 1e-12
    scale = np.abs(a[4]).max()
    assert scale > 0 and np.abs(a[4] - b[4]).max() <= 1e-12 * max(scale, 1e-3)
    # BJ config 4 with a 64-point field map: 0.46 TB of stored accumulators against ~2 GB for the replay
    assert ul.workspace_bytes(32, 32, 2, 4, 16, 64) > 200 * ul.workspace_bytes_replay2(32, 32, 2, 4, 16, 64)


def test_config4_full_mid_plane_field_map_by_replay(ul):
    """BJ config 4 as stated: 32^4, two levels (d = 2 and 4), r = 1..16, the FULL mid-plane of field points
    (32 x 32 transverse offsets, 12 channels).  Stored accumulators would need ~7 TB; the replay needs 1.6 GB.
    Reduced n_in = n_out = 2 here.  The correlators equal those of ul_multilevel2 without fields bit for bit, and
    the map at sampled points equals the stored path run with just those points."""
    import time
    Ns = Nt = 32
    R = 16
    plane = [(0, b, c) for c in range(Ns) for b in range(Ns)]
    sample = [plane[0], plane[5 + 32 * 3], plane[17 + 32 * 30]]
    assert ul.workspace_bytes_replay2(Ns, Nt, 2, 4, R, len(plane)) < 2 * 2 ** 30 < 1000 * 2 ** 30 < ul.workspace_bytes(Ns, Nt, 2, 4, R, len(plane))
    out = {}
    for mode in ("map", "sampled", "nofields"):
        g = ul.Lattice(Ns, Nt, 1.0, 4)
        for _ in range(10):
            g.sweep(1, 3)
        t0 = time.perf_counter()
        if mode == "map":
            g.multilevel2_replay(2, 2, 4, 2, R, plane)
        elif mode == "sampled":
            g.multilevel2(2, 2, 4, 2, R, sample)
        else:
            g.multilevel2(2, 2, 4, 2, R)
        out[mode] = g.read_correlators() + (g.get_links_raw(), time.perf_counter() - t0)
    print("config 4 full mid-plane map by replay (n_in = n_out = 2): %.2f s" % out["map"][4])   # 0.04 s through the transverse DFT
    assert np.array_equal(out["map"][0], out["nofields"][0]) and np.array_equal(out["map"][3], out["nofields"][3])
    fmap = out["map"][1]                                            # [r][fp][12]
    idx = [plane.index(p) for p in sample]
    assert np.all(np.isfinite(fmap))
    ref = out["sampled"][1]
    assert np.abs(fmap[:, idx] - ref).max() <= 1e-11 * np.abs(ref).max()


def test_graph_cache_stays_bounded_over_a_beta_scan(ul):
    """Every new recipe (here: 40 values of beta) captures a new graph; the cache keeps the last 16.  The scan must
    give the same links as the same scan issued sub-step by sub-step."""
    a = ul.Lattice(8, 4, 0.5, 3)
    b = ul.Lattice(8, 4, 0.5, 3)
    for i in range(40):
        beta = 0.5 + 0.02 * i
        a.set_beta(beta)
        b.set_beta(beta)
        a.sweep(1, 1)
        for kind in (0, 1):
            for parity in range(2):
                for mu in range(4):
                    b.substep(kind, parity, mu, 0)
            if kind == 0:
                b.set_counter(b.get_counter() + 1)
    assert np.array_equal(a.get_links_raw(), b.get_links_raw()) and a.get_counter() == b.get_counter() == 40


@pytest.mark.parametrize("world", [2, 4])
@pytest.mark.parametrize("alg", [0, 1])
def test_sharded_full_sweeps_reproduce_the_unsharded_run(ul, world, alg):
    """Full (unmasked) sweeps of a t-sharded lattice with one halo exchange per sub-step, the shards run one after
    the other on this GPU and the exchange done as copies: bit-identical to ul_sweep on the whole lattice."""
    from paper_1309_3859_b200 import sharded
    Ns, Nt, beta, seed = 8, 16, 0.99, 91
    full = ul.Lattice(Ns, Nt, beta, seed)
    full.set_update_algorithm(alg, 1.2)
    full.sweep(2, 1)
    links0, ctr0 = full.get_links(), full.get_counter()
    full.set_links(links0)
    full.sweep(2, 2)
    want = full.get_links_raw()
    shards = [sharded.ShardedSweeper(Ns, Nt, beta, seed, r, world, links0, ctr0) for r in range(world)]
    for sh in shards:
        sh.alg = alg
        sh.lat.set_update_algorithm(alg, 1.2)
    sharded.sharded_sweep(shards, 2, 2)
    got = np.concatenate([sh.own_links_raw() for sh in shards], axis=1)
    assert np.array_equal(got, want)
    assert all(sh.lat.get_counter() == full.get_counter() for sh in shards)


@pytest.mark.parametrize("world,flags", [(2, False), (4, False), (2, True), (4, True), (1, True)])
@pytest.mark.parametrize("alg", [0, 1])
def test_peer_memory_halo_writes_reproduce_the_unsharded_run(ul, world, flags, alg):
    """Full sweeps of a t-sharded lattice with the halo exchange FUSED into the sub-step kernels (ul_set_halo_peers: the kernels
    store their boundary layers into the neighbours' ghost layers, here peer pointers on the same device) and, with flags,
    every shard on its own stream, ordered only by the stream-ordered flag words between neighbours
    (cuStreamWriteValue32 / cuStreamWaitValue32: no host synchronisation, no kernel waits on another): bit-identical
    to ul_sweep on the whole lattice."""
    import torch
    from paper_1309_3859_b200 import sharded
    Ns, Nt, beta, seed = 8, 16, 0.99, 91
    full = ul.Lattice(Ns, Nt, beta, seed)
    full.set_update_algorithm(alg, 1.2)
    full.sweep(2, 1)
    links0, ctr0 = full.get_links(), full.get_counter()
    full.set_links(links0)
    full.sweep(2, 3)
    want = full.get_links_raw()
    streams = [torch.cuda.Stream() if flags else None for _ in range(world)]
    shards = [sharded.ShardedSweeper(Ns, Nt, beta, seed, r, world, links0, ctr0, stream=streams[r]) for r in range(world)]
    for sh in shards:
        sh.alg = alg
        sh.lat.set_update_algorithm(alg, 1.2)
        sh.lat.sync()
    sharded.connect_peers(shards, flags=flags)
    n0 = [sh.lat.launch_count() for sh in shards]
    sharded.sharded_sweep(shards, 2, 3, peer=True)
    for sh in shards:
        sh.lat.sync()
    got = np.concatenate([sh.own_links_raw() for sh in shards], axis=1)
    assert np.array_equal(got, want)
    assert all(sh.lat.get_counter() == full.get_counter() for sh in shards)
    assert all(sh.lat.launch_count() - n for sh, n in zip(shards, n0))


TWO_PROCESS_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_1309_3859_b200 import sharded, ul
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2)
rank, world = dist.get_rank(), 2
Ns, Nt, d, R, n_sub, beta, seed = 8, 16, 2, 3, 5, 0.99, 77
bufs = [torch.zeros((4, Nt, Ns, Ns, Ns), dtype=torch.float32), torch.zeros((4, Nt, Ns, Ns, Ns), dtype=torch.int32),
        torch.zeros((4, Nt, Ns, Ns, Ns), dtype=torch.int32), torch.zeros(2 * R + 2, dtype=torch.float64)]
if rank == 0:                                        # the unsharded runs: one multilevel measurement, then full sweeps
    full = ul.Lattice(Ns, Nt, beta, seed)
    for _ in range(10):
        full.sweep(1, 3)
    links0, ctr0 = full.get_links(), full.get_counter()
    full.set_links(links0)
    full.multilevel(d, n_sub, R)
    C_full = full.read_correlators()[0]
    after_ml = full.get_links_raw()
    ctr1 = full.get_counter()
    full.set_links(links0); full.set_counter(ctr0)
    full.sweep(2, 2)
    after_sw = full.get_links_raw()
    bufs = [torch.from_numpy(links0.copy()), torch.from_numpy(after_ml.copy()), torch.from_numpy(after_sw.copy()),
            torch.from_numpy(np.concatenate([C_full.real, C_full.imag, [float(ctr0), float(ctr1)]]))]
    del full
for b in bufs:
    dist.broadcast(b, 0)
links0, after_ml, after_sw = (b.numpy() for b in bufs[:3])
C_full = bufs[3][:R].numpy() + 1j * bufs[3][R:2 * R].numpy()
ctr0, ctr1 = int(bufs[3][2 * R]), int(bufs[3][2 * R + 1])
# (1) slab-sharded multilevel: no communication in the sub-update loop, one all-gather, product in the library
sh = sharded.ShardedLattice(Ns, Nt, beta, seed, d, rank, world, links0, ctr0)
sh.multilevel(n_sub, R)
t0, n = sh.parts[rank]
ok_links = np.array_equal(sh.lat.get_links_raw()[:, :n], after_ml[:, t0:t0 + n]) and sh.lat.get_counter() == ctr1
C = sh.correlators(dist, stage_on_host=True)
ok_C = np.abs(C - C_full).max() <= 1e-13 * max(1.0, np.abs(C_full).max())
# (2) halo-exchanged full sweeps
sw = sharded.ShardedSweeper(Ns, Nt, beta, seed, rank, world, links0, ctr0, stage_on_host=True)
sharded.sharded_sweep([sw], 2, 2, dist)
ok_sweep = np.array_equal(sw.own_links_raw(), after_sw[:, sw.t0:sw.t0 + sw.nt_loc]) and sw.lat.get_counter() == ctr0 + 2
# (3) the same sweeps with peer-memory halo writes between the two PROCESSES: CUDA IPC handles of the link arrays and
# flag words, the kernels write the neighbour's ghost layers, the streams wait on the flag words (no communication call)
import signal
signal.alarm(240)                                    # a lost hand-shake must not outlive the test
pw = sharded.ShardedSweeper(Ns, Nt, beta, seed, rank, world, links0, ctr0)
sharded.connect_peers_ipc(pw, dist)
sharded.sharded_sweep([pw], 2, 2, peer=True)
pw.lat.sync()
ok_peer = np.array_equal(pw.own_links_raw(), after_sw[:, pw.t0:pw.t0 + pw.nt_loc]) and pw.lat.get_counter() == ctr0 + 2
dist.barrier()
signal.alarm(0)
print("RESULT", rank, bool(ok_links), bool(ok_C), bool(ok_sweep), bool(ok_peer))
dist.destroy_process_group()
"""


def test_two_processes_on_one_gpu_sharded_multilevel_and_sweeps(ul, tmp_path):
    """The real multi-process code path of paper_1309_3859_b200/sharded.py: two ranks (two processes, both on cuda:0,
    torch.distributed over gloo with host-staged tensors; no kernel of one rank waits on the other: the waits are the
    hosts') run ShardedLattice and ShardedSweeper and reproduce the unsharded run bit for bit / to 1e-13; then the same
    sweeps with peer-memory halo writes between the processes (CUDA IPC; stream-ordered flag words, no spinning kernel)."""
    import subprocess
    import sys
    script = tmp_path / "worker.py"
    script.write_text(TWO_PROCESS_WORKER.format(root=ROOT))
    port = 33500 + os.getpid() % 2000
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    try:
        outs = [p.communicate(timeout=600) for p in procs]
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    assert all(p.returncode == 0 for p in procs), outs
    for r in range(2):
        line = [l for l in outs[r][0].splitlines() if l.startswith("RESULT")][0]
        assert line == f"RESULT {r} True True True True", (line, outs[r][1][-2000:])


# ----------------------------------------------------------------------------- asynchronous read-back
def test_get_links_async_equals_get_links(ul):
    """ul_get_links_async / ul_get_links_wait return the same bytes as ul_get_links: one call, two calls before one wait (the
    second waits on the stream for the first copy), and a call overtaken by the next ul_set_links and sweeps (the copy reads its
    own buffer, not the link array that is being overwritten)."""
    import torch
    Ns, Nt = 16, 8
    g = ul.Lattice(Ns, Nt, 0.99, 17)
    g.sweep(1, 2)
    want = g.get_links()
    a = torch.empty(4 * g.V, dtype=torch.float32).pin_memory()
    b = torch.empty(4 * g.V, dtype=torch.float32).pin_memory()
    g.get_links_async(a)
    g.get_links_wait()
    assert np.array_equal(a.numpy().reshape(want.shape), want)
    g.get_links_wait()                                              # nothing pending: returns at once
    a.zero_()
    g.get_links_async(a)
    g.sweep(1, 1)
    want2 = g.get_links()
    g.get_links_async(b)                                            # second call before the wait
    g.set_links(want)                                               # overtakes the copies
    g.sweep(0, 3)
    g.get_links_wait()
    assert np.array_equal(a.numpy().reshape(want.shape), want)
    assert np.array_equal(b.numpy().reshape(want.shape), want2)
    # the upload in two parts: started while sweeps run, committed afterwards; equals ul_set_links
    src = torch.from_numpy(want.reshape(-1).copy()).pin_memory()
    g.set_links(want2)
    g.set_links_async(src)
    g.sweep(1, 1)                                                   # works on want2 while the upload is in flight
    g.set_links_commit()
    assert np.array_equal(g.get_links(), want)
    with pytest.raises(Exception):
        g.set_links_commit()                                        # nothing pending
    src[5] = float("nan")
    g.set_links_async(src)
    with pytest.raises(Exception):
        g.set_links_commit()                                        # validation as in ul_set_links
    c = np.empty(4 * g.V, dtype=np.float32)                         # pageable memory: still correct
    g.set_links(want2)
    g.get_links_async(torch.from_numpy(c))
    g.get_links_wait()
    assert np.array_equal(c.reshape(want.shape), want2)


# ----------------------------------------------------------------------------- degenerate and extreme shapes
@pytest.mark.parametrize("Ns,Nt,d", [(2, 2, 2), (2, 4, 1), (4, 2, 2), (6, 6, 6), (4, 8, 8), (10, 4, 2), (4, 12, 3), (4, 30, 5), (4, 24, 8),
                                     (2, 126, 7)])
def test_degenerate_shapes_against_oracle(ul, ulo, Ns, Nt, d):
    """Smallest lattice (2^4 sites wrap onto themselves), a single slab (d = Nt), thickness 1 (every spatial link
    frozen), several slabs of thickness 3, 5, 7, 8 (the masked spatial launches enumerate the d - 1 non-frozen layers of every
    slab), r_max = Ns/2 (the largest separation), rows that are not a multiple of the vector width (Ns = 6, 10):
    one heatbath and one overrelaxation sweep link by link, then the frozen-configuration estimator, stored and replay."""
    beta, R = 0.9, Ns // 2
    o = ulo.Oracle(Ns, Nt, beta, 8)
    ob = ulo.Oracle(Ns, Nt, beta, 8)
    g = ul.Lattice(Ns, Nt, beta, 8)
    assert same_links(g.get_links(), o.get_links())
    for kind in (0, 1):
        for slab in (0, d):
            for parity in range(2):
                for mu in range(4):
                    before = o.get_links()
                    ob.set_links(before)
                    g.set_links(before)
                    g.set_counter(o.get_counter())
                    o.substep(kind, parity, mu, slab)
                    g.substep(kind, parity, mu, slab)
                    check_links(g.get_links(), o.get_links(), before, ob, (kind, slab, parity, mu), allow_frac=1e-3)
    fps = [(0, 0, 0), (0, 1, 0), (-1, 0, 1)]
    g.set_links(o.get_links())
    o.multilevel(d, 0, R, fps)
    co, fo, vo = o.read_correlators()
    Vs = Ns ** 3
    for call in (g.multilevel, g.multilevel_replay):
        call(d, 0, R, fps)
        cg, fg, vg = g.read_correlators()
        assert np.abs(g.read_slab_averages() - o.read_slab_averages()).max() < 1e-5
        for got, want, n in ((cg, co, 3 * Vs), (fg, fo, 3 * Vs * Nt), (vg, vo, 3 * Vs * Nt)):
            ok, worst = rel_ok(got, want, n)
            assert ok, worst
    g.multilevel(d, 3, R, fps)                                      # and the sub-update loop runs (d = 1: nothing spatial moves)
    assert np.all(np.isfinite(g.read_correlators()[0]))


def test_beta_zero_heatbath_is_uniform_on_device(ul):
    from scipy import stats
    g = ul.Lattice(16, 4, 0.0, 5)
    g.init(0)
    g.sweep(1, 0)
    th = g.get_links().astype(np.float64).ravel()
    _, p = stats.kstest(th, lambda x: (x + np.pi) / (2 * np.pi))
    assert p > 1e-3 and abs(g.plaquette()[0]) < 0.01


# ----------------------------------------------------------------------------- slab-group-major order
@pytest.mark.parametrize("Ns,Nt,d,grp,streams,alg,n_fp,mh", [(8, 8, 2, 1, 1, 0, 0, 0), (8, 12, 2, 4, 1, 0, 3, 0), (6, 8, 4, 1, 1, 1, 2, 0), (16, 16, 2, 3, 1, 0, 0, 0),
                                                             (8, 16, 2, 2, 2, 0, 0, 0), (8, 12, 2, 1, 4, 1, 2, 0), (16, 16, 2, 3, 2, 0, 3, 0), (8, 8, 4, 1, 3, 0, 0, 0),
                                                             (8, 12, 2, 2, 2, 0, 2, 1), (8, 8, 2, 1, 4, 0, 0, 1)])
def test_slab_group_major_order_is_bit_identical(ul, Ns, Nt, d, grp, streams, alg, n_fp, mh):
    """ul_set_slab_group / ul_set_slab_group_streams: the n_sub loop run slab group by slab group (ragged last group, ragged
    last round, ragged last batch), one group after the other or several side by side on their own streams (a round's compound
    sub-update captured as one CUDA graph with a fork and a join), gives the same links, sweep counter, slab sums, C(r) and G
    bit for bit as the sub-update-major order; vacuum to 1e-13."""
    R, n_sub = 3, 5
    fps = FPS[:n_fp]
    res = []
    for mode in (0, grp):
        g = ul.Lattice(Ns, Nt, 1.0, 9)
        g.sweep(2, 2)
        if alg:
            g.set_update_algorithm(1, 1.3)
        g.set_accum_batch(2)
        g.set_multihit(mh)
        g.set_slab_group(mode)
        g.set_slab_group_streams(streams)
        g.multilevel(d, n_sub, R, fps)
        g.multilevel(d, n_sub, R, fps)                               # (the second call replays the captured rounds)
        res.append((g.get_links_raw(), g.get_counter(), g.read_slab_averages(), *g.read_correlators()))
    a, b = res
    assert np.array_equal(a[0], b[0]) and a[1] == b[1]
    assert np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3]) and np.array_equal(a[4], b[4])
    assert np.allclose(a[5], b[5], rtol=0, atol=1e-13)


def test_slab_group_rounds_follow_a_changed_measurement(ul):
    """The captured rounds are keyed by everything their launches were recorded with: a second measurement with another r_max
    (the library-owned workspace grows and moves), another n_sub, another beta and another sub-update recipe must not replay a
    stale graph: every call equals the one-launch form bit for bit."""
    Ns, Nt, d = 8, 16, 2
    res = {}
    for mode in (0, 2):
        g = ul.Lattice(Ns, Nt, 1.0, 23)
        g.sweep(2, 2)
        g.set_slab_group(mode)
        g.set_slab_group_streams(2)
        out = []
        for R, n_sub, beta, recipe in ((2, 5, 1.0, (1, 3)), (4, 5, 1.0, (1, 3)), (4, 3, 0.9, (1, 3)), (3, 9, 0.9, (2, 1)), (2, 5, 1.0, (1, 3))):
            g.set_beta(beta)
            g.set_subupdate(*recipe, 1)
            g.multilevel(d, n_sub, R)
            out.append((g.get_links_raw(), g.get_counter(), g.read_correlators()[0]))
        res[mode] = out
    for a, b in zip(res[0], res[2]):
        assert np.array_equal(a[0], b[0]) and a[1] == b[1] and np.array_equal(a[2], b[2])


def test_default_slab_groups_at_bench_size_are_bit_identical(ul):
    """64^4, the bench's multilevel call in its default form (rounds of 4 groups x 2 slabs side by side, graph-replayed, heatbath
    stragglers finished in the kernel) against the one-launch-over-all-slabs form: same links, counter and C(r) bit for bit."""
    Ns = Nt = 64
    R = 16
    g = ul.Lattice(Ns, Nt, 0.98, 5, workspace_bytes=ul.workspace_bytes(Ns, Nt, 2, 0, R, 0))
    g.sweep(1, 2)
    g.set_subupdate(1, 4, 1)
    raw, ctr = g.get_links_raw(), g.get_counter()
    res = []
    for mode in (-1, 0):
        g.set_slab_group(mode)
        g.set_links_raw(raw)
        g.set_counter(ctr)
        n0 = g.launch_count()
        g.multilevel(2, 9, R)                                      # a full batch and a ragged one
        res.append((g.get_links_raw(), g.get_counter(), g.read_correlators()[0], g.launch_count() - n0))
    assert np.array_equal(res[0][0], res[1][0]) and res[0][1] == res[1][1] and np.array_equal(res[0][2], res[1][2])
    assert res[0][3] > 4 * res[1][3] // 2                           # the grouped form really ran (many small launches)


def test_substep_slabs_covers_the_masked_substep(ul):
    """ul_substep_slabs over a partition of the slabs == ul_substep with the same mask (heatbath, every direction)."""
    Ns, Nt, d = 8, 12, 2
    a = ul.Lattice(Ns, Nt, 1.0, 4)
    b = ul.Lattice(Ns, Nt, 1.0, 4)
    for parity in (0, 1):
        for mu in range(4):
            a.substep(0, parity, mu, d)
            for s0, s1 in ((4, 6), (0, 1), (1, 4)):
                b.substep_slabs(0, parity, mu, d, s0, s1)
    assert np.array_equal(a.get_links_raw(), b.get_links_raw())
    with pytest.raises(ul.UlError):
        b.substep_slabs(0, 0, 0, d, 3, 7)


def test_vacuum_without_field_points_is_that_of_the_final_configuration(ul, ulo):
    """n_fp = 0: the plaquettes are not evaluated per sub-update (U-table fast path); the vacuum values returned are
    those of the final configuration (include/ul.h), checked against the oracle's frozen-configuration vacuum."""
    Ns, Nt = 8, 4
    g = ul.Lattice(Ns, Nt, 1.0, 2)
    g.sweep(3, 3)
    g.multilevel(2, 3, 3)
    _, _, vg = g.read_correlators()
    o = ulo.Oracle(Ns, Nt, 1.0, 2)
    o.set_links(g.get_links())
    o.multilevel(2, 0, 1)
    _, _, vo = o.read_correlators()
    ok, worst = rel_ok(vg, vo, 3 * Ns ** 3 * Nt)
    assert ok, worst
