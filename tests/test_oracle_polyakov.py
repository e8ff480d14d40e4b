"""Pins of the oracle's Polyakov-loop average with analytic multihit (Eqs. 15-16), -m "not gpu".

Closed forms (cold start: r(6 beta)^Nt; constant temporal angle; beta = 0), gauge invariance on random
configurations (a wrong sign of alpha breaks it), a numpy restatement from the pinned staple with scipy's Bessel
functions, and the statistical statement that the multihit estimator has the same mean and a smaller variance.
"""
import numpy as np
from scipy import special

from tests import inputs


def _ratio(a):
    return special.ive(1, a) / special.ive(0, a)


def test_closed_forms(ulo):
    Ns, Nt, beta = 4, 6, 0.8
    o = ulo.Oracle(Ns, Nt, beta, 1)
    o.init(0)
    assert abs(o.polyakov(0) - 1) < 1e-15
    assert abs(o.polyakov(1) - _ratio(6 * beta) ** Nt) < 1e-14           # every staple sum is 6
    links = np.zeros((4, Nt, Ns, Ns, Ns), dtype=np.float32)
    links[0] = 0.25                                                      # constant temporal angle: P = e^{i Nt phi}
    o.set_links(links)
    assert abs(o.polyakov(0) - np.exp(1j * Nt * float(np.float32(0.25)))) < 1e-14
    assert abs(o.polyakov(1) - _ratio(6 * beta) ** Nt * np.exp(1j * Nt * float(np.float32(0.25)))) < 1e-13   # plaquettes are all trivial
    z = ulo.Oracle(Ns, Nt, 0.0, 1)
    assert z.polyakov(1) == 0                                            # beta = 0: the link average vanishes
    assert abs(z.polyakov(0) - z.polyakov_naive(0)[1]) < 1e-15


def test_gauge_invariance(ulo):
    Ns, Nt = 4, 4
    links = inputs.hot_links(Ns, Nt, 8) * 0.5
    lam = inputs.gauge_function(Ns, Nt, 9)
    o = ulo.Oracle(Ns, Nt, 1.1, 1)
    vals = []
    for cfg in (links, inputs.gauge_transform(links, lam)):
        o.set_links(cfg)
        vals.append((o.polyakov(0), o.polyakov(1)))
    assert abs(vals[0][0] - vals[1][0]) < 2e-6 and abs(vals[0][1] - vals[1][1]) < 2e-6   # fp32 storage of the transformed links
    assert abs(vals[0][1]) > 1e-4


def test_numpy_restatement_from_the_staple(ulo):
    Ns, Nt, beta = 4, 4, 0.9
    o = ulo.Oracle(Ns, Nt, beta, 5)
    o.sweep(3, 1)
    Vs = Ns ** 3
    P = np.ones(Vs, dtype=complex)
    for t in range(Nt):
        for xs in range(Vs):
            k, alpha = o.staple(0, xs + Vs * t)
            P[xs] *= _ratio(beta * k) * np.exp(1j * alpha)
    assert abs(o.polyakov(1) - P.mean()) < 1e-13


def test_multihit_has_the_same_mean_and_less_noise(ulo):
    # Re <P conj(P_ref)> is not available without a reference phase, so compare <|mean_x P|^2>-free quantities:
    # the lattice means over an ensemble, real and imaginary parts, and their spreads.
    Ns, Nt, beta = 4, 2, 1.3                                             # deconfined, short time extent: |<P>| is sizeable
    o = ulo.Oracle(Ns, Nt, beta, 17)
    o.init(0)
    o.sweep(30, 30)
    plain, mh = [], []
    for _ in range(200):
        o.sweep(1, 2)
        plain.append(o.polyakov(0))
        mh.append(o.polyakov(1))
    plain, mh = np.array(plain), np.array(mh)
    d = mh - plain                                                       # same configurations: the difference has mean zero
    nb = 10
    db = d.reshape(nb, -1).mean(axis=1)
    err = np.hypot(db.real.std(ddof=1), db.imag.std(ddof=1)) / np.sqrt(nb)
    assert abs(d.mean()) < 4 * err + 1e-3, (d.mean(), err)
    assert abs(plain.mean()) > 0.05                                      # there is a signal to speak of
    assert np.abs(d).mean() < 0.5 * np.abs(plain).mean()                 # and the two estimators track each other


# ----------------------------------------------------------------- multihit inside the two-link operators (r >= 2)
def test_multihit_two_link_closed_forms_and_gauge_invariance(ulo):
    Ns, Nt, beta, R = 6, 4, 0.8, 3
    o = ulo.Oracle(Ns, Nt, beta, 1)
    o.init(0)
    o.set_multihit(1)
    o.multilevel(2, 0, R)
    c = o.read_correlators()[0]
    r = _ratio(6 * beta)
    assert abs(c[0] - 1) < 1e-14                                       # r = 1 keeps the plain links (they share plaquettes)
    assert np.abs(c[1:] - r ** (2 * Nt)).max() < 1e-13                 # 2 Nt multihit links per pair of lines
    links = inputs.hot_links(Ns, Nt, 3) * 0.6
    lam = inputs.gauge_function(Ns, Nt, 4)
    vals = []
    for cfg in (links, inputs.gauge_transform(links, lam)):
        o.set_links(cfg)
        o.multilevel(2, 0, R)
        vals.append(o.read_correlators()[0])
    assert np.abs(vals[0] - vals[1]).max() < 2e-6 and np.abs(vals[0][1:]).max() > 1e-6


def test_multihit_two_link_numpy_restatement(ulo):
    Ns, Nt, beta, d, R = 4, 4, 0.9, 2, 2
    o = ulo.Oracle(Ns, Nt, beta, 5)
    o.sweep(3, 1)
    o.set_multihit(1)
    o.multilevel(d, 0, R)
    got = o.read_slab_averages()                                        # [3][R][n_slab][Vs]
    Vs = Ns ** 3
    ubar = np.empty((Nt, Vs), dtype=complex)
    for t in range(Nt):
        for xs in range(Vs):
            k, alpha = o.staple(0, xs + Vs * t)
            ubar[t, xs] = _ratio(beta * k) * np.exp(1j * alpha)
    ubar = ubar.reshape(Nt, Ns, Ns, Ns)                                 # [t][x3][x2][x1]
    for mu in (1, 2, 3):
        shifted = np.roll(ubar, -2, axis=inputs.AXIS[mu])               # Ubar(x + 2 mu)
        T = (np.conj(ubar) * shifted).reshape(Nt // d, d, Vs).prod(axis=1)
        assert np.abs(got[mu - 1, 1] - T).max() < 1e-13
    o.set_multihit(0)
    o.multilevel(d, 0, R)
    plain = o.read_slab_averages()
    assert np.array_equal(plain[:, 0], got[:, 0]) and not np.allclose(plain[:, 1], got[:, 1])


def test_multihit_two_link_same_mean_smaller_error(ulo):
    """The estimator of C(2) with multihit links has the same expectation value and a smaller error (4^3 x 4,
    beta = 0.7: signal ~1e-3)."""
    Ns, Nt, beta = 4, 4, 0.7
    res = {}
    for on in (0, 1):
        o = ulo.Oracle(Ns, Nt, beta, 23)
        o.set_subupdate(1, 2, 1)
        o.set_multihit(on)
        o.sweep(20, 20)
        vals = []
        for _ in range(150):
            o.sweep(1, 2)
            o.multilevel(2, 6, 2)
            vals.append(o.read_correlators()[0][1].real)
        v = np.array(vals)
        b = v.reshape(10, -1).mean(axis=1)
        res[on] = (v.mean(), b.std(ddof=1) / np.sqrt(10))
    (m0, e0), (m1, e1) = res[0], res[1]
    assert abs(m0 - m1) < 4 * np.hypot(e0, e1), res
    assert e1 < e0, res
