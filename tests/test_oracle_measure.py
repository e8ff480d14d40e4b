"""Pins for the oracle's observables: plaquette, Polyakov-loop correlators, the single- and
two-level multilevel estimators and the plaquette-inserted field channels.  CPU only."""
import numpy as np
import pytest

from tests import inputs
from tests.inputs import shift


# ----------------------------------------------------------------------------- brute force in numpy
def frame(mu):
    return 1 + (mu % 3), 1 + ((mu + 1) % 3)


def comp_dirs(mu, comp):
    nu, rho = frame(mu)
    return [(0, mu), (0, nu), (0, rho), (nu, rho), (rho, mu), (mu, nu)][comp]


def plaq(th, a, b):
    """theta_P(a,b)(y) = theta_a(y) + theta_b(y+a) - theta_a(y+b) - theta_b(y)"""
    return th[a] + shift(th[b], a) - shift(th[a], b) - th[b]


def brute_force_single_config(links, d, r_max, fps):
    """C(r), G(r,fp,ch) for ONE configuration straight from Eqs. 22, 25, 31, 34 with np.roll:
    no slab averaging is involved, so [T] = T and the estimator is the plain product."""
    th = links.astype(np.float64)
    Nt, Ns = th.shape[1], th.shape[2]
    S = Nt // d
    C = np.zeros(r_max, dtype=complex)
    G = np.zeros((r_max, len(fps), 12), dtype=complex)
    for r in range(1, r_max + 1):
        for mu in (1, 2, 3):
            nu, rho = frame(mu)
            T = np.exp(1j * (shift(th[0], mu, r) - th[0]))                   # Eq. 22, per (t, x)
            T2 = T.reshape(S, d, Ns, Ns, Ns).prod(axis=1)                    # Eq. 25, per (s, x)
            full = T2.prod(axis=0)                                           # Eq. 26
            C[r - 1] += full.sum()
            for f, (a, b, c) in enumerate(fps):
                for ch in range(12):
                    pa, pb = comp_dirs(mu, ch // 2)
                    thP = plaq(th, pa, pb)
                    O = 1 - np.cos(thP) if ch % 2 == 0 else np.sin(thP)
                    O = shift(shift(shift(O, mu, r // 2 + a), nu, b), rho, c)   # O(x + off, t)
                    # Eq. 34 on one configuration: sum_t O(x0,t) prod_t' T(x,t') (each slab's TO times the others' T)
                    G[r - 1, f, ch] += (O.sum(axis=0) * full).sum()
    Vs = Ns ** 3
    return C / (3 * Vs), G / (3 * Vs * Nt)


FPS = [(0, 0, 0), (0, 1, 0), (1, 0, 0), (0, 0, 1), (-1, 2, 1)]


# ----------------------------------------------------------------------------- plaquette
def test_plaquette_cold_and_constant_flux(ulo):
    o = ulo.Oracle(4, 4, 1.0, 1)
    o.init(0)
    assert np.allclose(o.plaquette(), 1.0)
    links, phi = inputs.constant_flux_links(8, 4, m=1)
    o = ulo.Oracle(8, 4, 1.0, 1)
    o.set_links(links)
    p = o.plaquette()
    assert abs(p[0] - (5 + np.cos(phi)) / 6) < 1e-6        # closed form, SURVEY 8(c) pins
    assert abs(p[1] - 1.0) < 1e-6                           # time-like untouched
    assert abs(p[2] - (2 + np.cos(phi)) / 3) < 1e-6


def test_plaquette_matches_numpy(ulo):
    links = inputs.hot_links(4, 6, 5)
    o = ulo.Oracle(4, 6, 1.0, 1)
    o.set_links(links)
    th = links.astype(np.float64)
    st = np.mean([np.cos(plaq(th, 0, b)).mean() for b in (1, 2, 3)])
    ss = np.mean([np.cos(plaq(th, a, b)).mean() for a, b in ((1, 2), (1, 3), (2, 3))])
    p = o.plaquette()
    assert np.allclose(p, [(st + ss) / 2, st, ss], atol=1e-13)


# ----------------------------------------------------------------------------- Eq. 23 and closed forms
def test_eq23_product_of_two_link_operators_is_polyakov_correlator(ulo):
    # P^dagger(x) P(x + r mu) = prod_t T(x,t,r mu), on any configuration, any slab thickness
    Ns, Nt = 6, 4
    o = ulo.Oracle(Ns, Nt, 1.0, 3)
    naive, meanP = o.polyakov_naive(3)
    for d in (1, 2, 4):
        o.multilevel(d, 0, 3)
        corr, _, _ = o.read_correlators()
        assert np.allclose(corr, naive, atol=1e-13)
    # independent numpy value of <P> (Eq. 15-16)
    th0 = o.get_links()[0].astype(np.float64)
    assert abs(np.exp(1j * th0.sum(axis=0)).mean() - meanP) < 1e-13


def test_correlator_closed_form_winding(ulo):
    # theta_0(x,t) = g(x)/Nt, g = 2 pi m x1/Ns  ->  C_{mu=1}(r) = e^{2 pi i m r/Ns}, C_{mu=2,3}(r) = 1
    Ns, Nt, m = 8, 4, 1
    links = np.zeros((4, Nt, Ns, Ns, Ns))
    links[0] = (2 * np.pi * m * np.arange(Ns) / Ns / Nt).reshape(1, 1, 1, Ns)
    links = (links - 2 * np.pi * np.round(links / (2 * np.pi))).astype(np.float32)
    o = ulo.Oracle(Ns, Nt, 1.0, 1)
    o.set_links(links)
    o.multilevel(2, 0, 4, FPS)
    corr, field, vac = o.read_correlators()
    want = np.array([(np.exp(2j * np.pi * m * r / Ns) + 2) / 3 for r in range(1, 5)])
    assert np.allclose(corr, want, atol=2e-6)


def test_cold_configuration(ulo):
    o = ulo.Oracle(4, 4, 1.0, 1)
    o.init(0)
    o.multilevel(2, 0, 2, FPS)
    corr, field, vac = o.read_correlators()
    assert np.allclose(corr, 1.0) and np.allclose(field, 0.0) and np.allclose(vac, 0.0)


def test_field_channels_on_constant_flux(ulo):
    # every (1,2) plaquette = phi, temporal links 0 -> T = 1 and G(ch) = frame average of O_ch:
    # (1,2) is comp 5 (mu,nu) for mu=1, comp 4 (rho,mu) for mu=2, comp 3 (nu,rho) for mu=3, each with sign +
    links, phi = inputs.constant_flux_links(8, 4, m=1)
    o = ulo.Oracle(8, 4, 1.0, 1)
    o.set_links(links)
    o.multilevel(2, 0, 3, FPS)
    corr, field, vac = o.read_correlators()
    assert np.allclose(corr, 1.0, atol=1e-12)
    want = np.zeros(12)
    for comp in (3, 4, 5):
        want[2 * comp] = (1 - np.cos(phi)) / 3
        want[2 * comp + 1] = np.sin(phi) / 3
    assert np.allclose(vac, want, atol=1e-6)
    for r in range(3):
        for f in range(len(FPS)):
            assert np.allclose(field[r, f], want, atol=1e-6)


@pytest.mark.parametrize("Ns,Nt,d", [(4, 4, 2), (4, 6, 3), (6, 4, 1), (4, 4, 4)])
def test_single_configuration_estimator_against_brute_force(ulo, Ns, Nt, d):
    # rows a7, a8, a10 with n_sub = 0 against the np.roll restatement of Eqs. 22-34 (index/offset/sign pin)
    links = inputs.hot_links(Ns, Nt, 100 + Ns + Nt)
    o = ulo.Oracle(Ns, Nt, 1.0, 1)
    o.set_links(links)
    r_max = Ns // 2
    o.multilevel(d, 0, r_max, FPS)
    corr, field, vac = o.read_correlators()
    C, G = brute_force_single_config(links, d, r_max, FPS)
    assert np.allclose(corr, C, atol=1e-12)
    assert np.allclose(field, G, atol=1e-12)
    # vacuum = frame-averaged lattice mean of O_ch
    th = links.astype(np.float64)
    for ch in range(12):
        vals = []
        for mu in (1, 2, 3):
            thP = plaq(th, *comp_dirs(mu, ch // 2))
            vals.append((1 - np.cos(thP)).mean() if ch % 2 == 0 else np.sin(thP).mean())
        assert abs(vac[ch] - np.mean(vals)) < 1e-12
    # slab averages on one configuration are the T^(d) themselves (unit modulus)
    sa = o.read_slab_averages()
    assert np.allclose(np.abs(sa), 1.0, atol=1e-12)
    th0 = th[0]
    T = np.exp(1j * (shift(th0, 2, 1) - th0)).reshape(Nt // d, d, -1).prod(axis=1)     # mu=2, r=1
    assert np.allclose(sa[1, 0], T, atol=1e-12)


def test_gauge_invariance(ulo):
    # BJ check (b): plaquette, C(r) and G invariant under theta_mu(x) -> theta_mu(x) + lam(x) - lam(x+mu);
    # a single-slab T^(2) is only covariant, the product over slabs is invariant
    Ns, Nt = 4, 4
    links = inputs.hot_links(Ns, Nt, 17)
    lam = inputs.gauge_function(Ns, Nt, 18)
    res = []
    for cfg in (links, inputs.gauge_transform(links, lam)):
        o = ulo.Oracle(Ns, Nt, 1.0, 1)
        o.set_links(cfg)
        o.multilevel(2, 0, 2, FPS)
        res.append((o.plaquette(), *o.read_correlators(), o.read_slab_averages()))
    (p0, c0, f0, v0, s0), (p1, c1, f1, v1, s1) = res
    assert np.allclose(p0, p1, atol=3e-7)
    assert np.allclose(c0, c1, atol=3e-6) and np.allclose(f0, f1, atol=3e-6) and np.allclose(v0, v1, atol=3e-6)
    assert not np.allclose(s0, s1, atol=1e-3)


def test_accumulate_hooks_equal_multilevel(ulo):
    # measure_begin / accumulate / measure_end reproduce ulo_multilevel's slab sums exactly
    Ns, Nt = 4, 4
    a = ulo.Oracle(Ns, Nt, 0.95, 1)
    b = ulo.Oracle(Ns, Nt, 0.95, 1)
    a.multilevel(2, 3, 2, FPS[:2])
    b.measure_begin(2, 2, FPS[:2])
    for _ in range(3):
        for k in range(1):
            # one masked compound sweep = 1 HB + 3 OR masked sweeps
            for parity in (0, 1):
                for mu in range(4):
                    b.substep(0, parity, mu, 2)
            b.set_counter(b.get_counter() + 1)
            for _ in range(3):
                for parity in (0, 1):
                    for mu in range(4):
                        b.substep(1, parity, mu, 2)
        b.accumulate()
    b.measure_end()
    for x, y in zip(a.read_correlators(), b.read_correlators()):
        assert np.array_equal(x, y)
    assert np.array_equal(a.get_links(), b.get_links())


def test_slab_average_is_mean_of_sub_update_values(ulo):
    # [T] = (1/n_sub) sum_j T^(2)_j with the configurations after each sub-update (S8(c)-O6): the start
    # configuration is not measured
    Ns, Nt, n = 4, 4, 3
    a = ulo.Oracle(Ns, Nt, 0.95, 5)
    b = ulo.Oracle(Ns, Nt, 0.95, 5)
    a.multilevel(2, n, 1)
    acc = 0
    for _ in range(n):
        b.multilevel(2, 1, 1)          # one sub-update + one measurement, chained from b's own state
        acc = acc + b.read_slab_averages()
    assert np.allclose(a.read_slab_averages(), acc / n, atol=1e-14)
    assert np.array_equal(a.get_links(), b.get_links())


def test_two_level_reduces_to_single_level(ulo):
    # d_in = d_out, n_out = 1: T^(4) = [T^(2)], so multilevel2 = one masked compound sweep + multilevel
    Ns, Nt = 4, 4
    a = ulo.Oracle(Ns, Nt, 0.95, 2)
    b = ulo.Oracle(Ns, Nt, 0.95, 2)
    a.multilevel2(2, 3, 2, 1, 2, FPS[:2])
    b.multilevel(2, 0, 1)                      # no-op measurement
    # the outer masked sweep
    for parity in (0, 1):
        for mu in range(4):
            b.substep(0, parity, mu, 2)
    b.set_counter(b.get_counter() + 1)
    for _ in range(3):
        for parity in (0, 1):
            for mu in range(4):
                b.substep(1, parity, mu, 2)
    b.multilevel(2, 3, 2, FPS[:2])
    for x, y in zip(a.read_correlators(), b.read_correlators()):
        assert np.allclose(x, y, atol=1e-14)


def test_two_level_combine_against_numpy(ulo):
    # Eqs. 32-33 (with the t+2 reading): one outer iteration; rebuild [T2], [TO2] from single-level runs and
    # combine them in numpy
    Ns, Nt, d_in, d_out, n_in, R = 4, 8, 2, 4, 2, 2
    fps = FPS[:2]
    a = ulo.Oracle(Ns, Nt, 0.9, 7)
    a.multilevel2(d_in, n_in, d_out, 1, R, fps)
    corr2, field2, vac2 = a.read_correlators()
    T4 = a.read_slab_averages()                                 # [3][R][Nt/d_out][Vs]
    b = ulo.Oracle(Ns, Nt, 0.9, 7)
    for parity in (0, 1):                                       # the outer (d_out-masked) compound sweep
        for mu in range(4):
            b.substep(0, parity, mu, d_out)
    b.set_counter(b.get_counter() + 1)
    for _ in range(3):
        for parity in (0, 1):
            for mu in range(4):
                b.substep(1, parity, mu, d_out)
    b.multilevel(d_in, n_in, R, fps)
    T2 = b.read_slab_averages()                                 # [3][R][Nt/d_in][Vs]
    want = T2[:, :, 0::2] * T2[:, :, 1::2]
    assert np.allclose(T4, want, atol=1e-14)
    C = want.prod(axis=2).sum(axis=(0, 2)) / (3 * Ns ** 3)
    assert np.allclose(corr2, C, atol=1e-14)


def eq34_from_slab_averages(avT, avTO, Nt):
    """C(r), G(r,fp,ch) from slab averages, straight from Eqs. 26 and 34:
    avT [3][R][S][Vs], avTO [3][R][S][F][12][Vs]."""
    Vs = avT.shape[-1]
    S = avT.shape[2]
    C = avT.prod(axis=2).sum(axis=(0, 2)) / (3 * Vs)
    G = 0
    for s in range(S):
        others = np.delete(avT, s, axis=2).prod(axis=2)                    # prod_{s' != s} [T](s'), [3][R][Vs]
        G = G + (avTO[:, :, s] * others[:, :, None, None, :]).sum(axis=(0, 4))
    return C, G / (3 * Vs * Nt)


def outer_masked_compound_sweep(o, d_out, n_or=3):
    """The d_out-masked compound sweep (1 heatbath + 3 overrelaxation, the default sub-update) by sub-steps."""
    for parity in (0, 1):
        for mu in range(4):
            o.substep(0, parity, mu, d_out)
    o.set_counter(o.get_counter() + 1)
    for _ in range(n_or):
        for parity in (0, 1):
            for mu in range(4):
                o.substep(1, parity, mu, d_out)


@pytest.mark.parametrize("Nt,d_in,d_out,n_in", [(8, 2, 4, 2), (12, 2, 6, 2), (8, 1, 4, 3)])
def test_two_level_field_combine_against_numpy(ulo, Nt, d_in, d_out, n_in):
    # Eq. 33 with the t+2 reading R7, for m = d_out/d_in = 2 (the paper's case), 3 and 4 inner slabs per
    # outer slab: TO^(d_out)(S) = sum_i [TO](s_i) prod_{i' != i} [T](s_i'), rebuilt in numpy from the single-level
    # slab averages of the same trajectory; then Eq. 34 on the outer averages; then the vacuum.
    Ns, R = 4, 2
    fps = FPS[:3]
    m = d_out // d_in
    a = ulo.Oracle(Ns, Nt, 0.9, 7)
    a.multilevel2(d_in, n_in, d_out, 1, R, fps)
    corr2, field2, vac2 = a.read_correlators()
    T4, TO4 = a.read_slab_averages(), a.read_slab_field_averages()
    b = ulo.Oracle(Ns, Nt, 0.9, 7)
    outer_masked_compound_sweep(b, d_out)
    b.multilevel(d_in, n_in, R, fps)
    T2, TO2 = b.read_slab_averages(), b.read_slab_field_averages()       # [3][R][Nt/d_in][Vs], [3][R][Nt/d_in][F][12][Vs]
    _, _, vac1 = b.read_correlators()
    assert np.array_equal(a.get_links(), b.get_links())
    n_outer = Nt // d_out
    T2g = T2.reshape(3, R, n_outer, m, -1)
    TO2g = TO2.reshape(3, R, n_outer, m, len(fps), 12, -1)
    wantT = T2g.prod(axis=3)                                               # Eq. 32
    wantTO = 0
    for i in range(m):                                                     # Eq. 33
        others = np.delete(T2g, i, axis=3).prod(axis=3)
        wantTO = wantTO + TO2g[:, :, :, i] * others[:, :, :, None, None, :]
    assert np.abs(TO2).max() > 0.1                                         # the comparison is not vacuous
    assert np.allclose(T4, wantT, atol=1e-14)
    assert np.allclose(TO4, wantTO, atol=1e-14)
    C, G = eq34_from_slab_averages(wantT, wantTO, Nt)
    assert np.allclose(corr2, C, atol=1e-15) and np.allclose(field2, G, atol=1e-15)
    assert np.allclose(vac2, vac1, atol=1e-15)


@pytest.mark.parametrize("Nt,d_in,d_out", [(8, 2, 4), (12, 2, 6)])
def test_two_level_on_one_configuration_equals_brute_force(ulo, Nt, d_in, d_out):
    # n_in = n_out = 1: every average is over ONE configuration, so Eqs. 32-34 must give the plain single-configuration
    # C and G of the final links (np.roll restatement of Eqs. 22-34, no slab structure at all): pins the cross terms
    # of Eq. 33 and every 1/n factor without reading any intermediate of the oracle
    Ns, R = 4, 2
    a = ulo.Oracle(Ns, Nt, 0.9, 21)
    a.multilevel2(d_in, 1, d_out, 1, R, FPS)
    corr, field, vac = a.read_correlators()
    C, G = brute_force_single_config(a.get_links(), d_out, R, FPS)
    assert np.allclose(corr, C, atol=1e-13)
    assert np.allclose(field, G, atol=1e-13)
    assert np.abs(G).max() > 1e-3


def test_two_level_outer_average_is_mean_of_chained_runs(ulo):
    # Alg. 1 lines 5-17, Eq. 27: [T4], [TO4] and the vacuum over n_out outer iterations are
    # the means of the single-iteration values along the same trajectory; C and G follow from the means by Eq. 34
    Ns, Nt, R, n_in, n_out = 4, 8, 2, 2, 3
    fps = FPS[:2]
    a = ulo.Oracle(Ns, Nt, 0.95, 9)
    a.multilevel2(2, n_in, 4, n_out, R, fps)
    b = ulo.Oracle(Ns, Nt, 0.95, 9)
    T4, TO4, vac = 0, 0, 0
    for _ in range(n_out):
        b.multilevel2(2, n_in, 4, 1, R, fps)                               # chained from b's own state
        T4 = T4 + b.read_slab_averages()
        TO4 = TO4 + b.read_slab_field_averages()
        vac = vac + b.read_correlators()[2]
    assert np.array_equal(a.get_links(), b.get_links()) and a.get_counter() == b.get_counter()
    assert np.allclose(a.read_slab_averages(), T4 / n_out, atol=1e-15)
    assert np.allclose(a.read_slab_field_averages(), TO4 / n_out, atol=1e-15)
    corr, field, vac_a = a.read_correlators()
    C, G = eq34_from_slab_averages(T4 / n_out, TO4 / n_out, Nt)
    assert np.allclose(corr, C, atol=1e-15) and np.allclose(field, G, atol=1e-15)
    assert np.allclose(vac_a, vac / n_out, atol=1e-15)
    # and the mean is not the single-iteration value
    assert not np.allclose(a.read_slab_averages(), b.read_slab_averages(), atol=1e-3)


def test_two_level_hooks_equal_multilevel2(ulo):
    # measure2_begin / accumulate / combine / measure2_end with the sweeps done by hand reproduce ulo_multilevel2
    Ns, Nt, R, n_in, n_out = 4, 8, 2, 3, 2
    fps = FPS[:2]
    a = ulo.Oracle(Ns, Nt, 0.95, 3)
    b = ulo.Oracle(Ns, Nt, 0.95, 3)
    a.multilevel2(2, n_in, 4, n_out, R, fps)
    b.measure2_begin(2, 4, R, fps)
    for _ in range(n_out):
        outer_masked_compound_sweep(b, 4)
        for _ in range(n_in):
            outer_masked_compound_sweep(b, 2)
            b.accumulate()
        b.combine()
    b.measure2_end()
    for x, y in zip(a.read_correlators(), b.read_correlators()):
        assert np.array_equal(x, y)
    assert np.array_equal(a.read_slab_field_averages(), b.read_slab_field_averages())
    assert np.array_equal(a.get_links(), b.get_links())
    # state errors: end with configurations pending, combine with nothing accumulated
    b.measure2_begin(2, 4, R, fps)
    with pytest.raises(ulo.OracleError):
        b.combine()
    b.accumulate()
    with pytest.raises(ulo.OracleError):
        b.measure2_end()
    with pytest.raises(ulo.OracleError):
        b.measure_end()


# ----------------------------------------------------------------------------- theory (statistical)
def _series_mean_err(x, nbins=10):
    x = np.asarray(x, dtype=float)
    b = x[: len(x) // nbins * nbins].reshape(nbins, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / np.sqrt(nbins)


def test_strong_coupling_plaquette(ulo):
    # BJ check (c): <cos theta_P> = I1(beta)/I0(beta) + O(u^5) = 0.0499376 at beta = 0.1
    from scipy import special
    o = ulo.Oracle(6, 6, 0.1, 11)
    o.sweep(5, 0)
    vals = []
    for _ in range(120):
        o.sweep(1, 1)
        vals.append(o.plaquette()[0])
    m, e = _series_mean_err(vals)
    want = special.iv(1, 0.1) / special.iv(0, 0.1)
    assert abs(want - 0.0499376) < 1e-7
    assert e < 1.5e-3 and abs(m - want) < 4 * e, (m, e, want)


def test_weak_coupling_plaquette(ulo):
    # BJ check (d): <1 - cos theta_P> ~ 1/(4 beta) = 0.05 at beta = 5 from a cold start (within 5 %)
    o = ulo.Oracle(6, 6, 5.0, 12)
    o.init(0)
    o.sweep(30, 30)
    vals = []
    for _ in range(60):
        o.sweep(1, 2)
        vals.append(1 - o.plaquette()[0])
    m, e = _series_mean_err(vals)
    assert abs(m - 0.05) < 0.05 * 0.05 + 4 * e, (m, e)


def test_equilibrium_heatbath_identity(ulo):
    # <cos theta_P> = <k I1(beta k)/I0(beta k)>_links / 6 in equilibrium (multihit form)
    from scipy import special
    beta = 0.9
    o = ulo.Oracle(4, 4, beta, 13)
    o.sweep(40, 40)
    lhs, rhs = [], []
    for _ in range(40):
        o.sweep(1, 2)
        lhs.append(o.plaquette()[0])
        ks = np.array([o.staple(mu, s)[0] for mu in range(4) for s in range(0, o.V, 3)])
        rhs.append(np.mean(ks * special.ive(1, beta * ks) / special.ive(0, beta * ks)) / 6)
    diff = np.array(lhs) - np.array(rhs)
    m, e = _series_mean_err(diff, nbins=8)
    assert abs(m) < 4 * e + 1e-4, (m, e)


def test_multilevel_matches_naive_on_2x2x2x2(ulo):
    # BJ check (e): on a 2^4 lattice the multilevel estimator equals the naive Polyakov correlator average
    beta = 0.8
    o = ulo.Oracle(2, 2, beta, 14)
    o.set_subupdate(1, 1, 1)
    o.sweep(50, 50)
    naive, ml = [], []
    for _ in range(400):
        o.sweep(1, 1)
        naive.append(o.polyakov_naive(1)[0][0].real)
        o.multilevel(2, 6, 1)
        ml.append(o.read_correlators()[0][0].real)
    mn, en = _series_mean_err(naive)
    mm, em = _series_mean_err(ml)
    assert abs(mn - mm) < 3.5 * np.hypot(en, em), (mn, en, mm, em)
    assert em < en                                     # and it does reduce the variance


def test_multilevel_matches_naive_and_strong_coupling_4x4x4x2(ulo):
    # C(1) ~ u^{Nt} with u = I1/I0 at strong coupling (Ns >= 4); multilevel agrees with naive
    from scipy import special
    beta = 0.3
    o = ulo.Oracle(4, 2, beta, 15)
    o.set_subupdate(1, 1, 1)
    o.sweep(20, 20)
    naive, ml = [], []
    for _ in range(120):
        o.sweep(1, 1)
        naive.append(o.polyakov_naive(1)[0][0].real)
        o.multilevel(2, 4, 1)
        ml.append(o.read_correlators()[0][0].real)
    mn, en = _series_mean_err(naive)
    mm, em = _series_mean_err(ml)
    u = special.iv(1, beta) / special.iv(0, beta)
    assert abs(mn - mm) < 3.5 * np.hypot(en, em), (mn, en, mm, em)
    assert abs(mm - u ** 2) < 4 * em + 0.1 * u ** 2, (mm, em, u ** 2)
