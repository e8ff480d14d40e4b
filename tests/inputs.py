"""Seeded synthetic input generators shared by the oracle tests and the GPU parity tests.

This module holds none of the method's arithmetic (no staples, no updates, no
estimators): only configurations and gauge functions drawn from numpy's seeded
generators, in the canonical layout [mu][t][x3][x2][x1], fp32 radians.
Recipe: lattices are Ns^3 x Nt like the paper's 24^3 x Nt
(P:92); angles are either uniform on [-pi, pi) ("hot"), small Gaussian
fluctuations around 0 ("smooth", weak-coupling like), or produced by the
library under test from a hot start followed by thermalisation sweeps.
"""
import numpy as np


def hot_links(Ns, Nt, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(-np.pi, np.pi, size=(4, Nt, Ns, Ns, Ns)).astype(np.float32)


def smooth_links(Ns, Nt, seed, width=0.4):
    rng = np.random.default_rng(seed)
    return (width * rng.standard_normal(size=(4, Nt, Ns, Ns, Ns))).astype(np.float32)


def gauge_function(Ns, Nt, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(-np.pi, np.pi, size=(Nt, Ns, Ns, Ns))


# array axis of a [t][x3][x2][x1] field that direction mu (0=t,1=x1,2=x2,3=x3) runs along
AXIS = {0: 0, 1: 3, 2: 2, 3: 1}


def shift(field, mu, n=1):
    """field(x) -> field(x + n*mu_hat) on a [..., t, x3, x2, x1] array (periodic)."""
    return np.roll(field, -n, axis=field.ndim - 4 + AXIS[mu])


def gauge_transform(links, lam):
    """theta_mu(x) -> theta_mu(x) + lam(x) - lam(x + mu_hat), wrapped to [-pi, pi), fp32."""
    out = np.empty_like(links)
    for mu in range(4):
        v = links[mu].astype(np.float64) + lam - shift(lam, mu)
        v = v - 2 * np.pi * np.round(v / (2 * np.pi))
        out[mu] = v.astype(np.float32)
    return out


def constant_flux_links(Ns, Nt, m=1):
    """theta_2(x) = phi * x1 with phi = 2 pi m / Ns: every (1,2) plaquette equals phi, all others 0."""
    links = np.zeros((4, Nt, Ns, Ns, Ns), dtype=np.float64)
    phi = 2 * np.pi * m / Ns
    x1 = np.arange(Ns).reshape(1, 1, 1, Ns)
    links[2] = phi * x1
    links = links - 2 * np.pi * np.round(links / (2 * np.pi))
    return links.astype(np.float32), phi
