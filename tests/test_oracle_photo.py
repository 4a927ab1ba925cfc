"""Pins of the oracle's photolysis rate constants: what the definitions
fix without this code -- closed forms of a transparent atmosphere and of a grey uniform slab, a one-bin
cross-section, invariances and linearity."""
import numpy as np
import pytest


class P:
    def __init__(self, dl, abs_species, sigma_ext, sigma_ph):
        self.dlambda = np.asarray(dl, dtype=np.float64)
        self.abs_species = np.asarray(abs_species, dtype=np.int32)
        self.sigma_ext = np.asarray(sigma_ext, dtype=np.float64).reshape(len(abs_species), -1)
        self.sigma_ph = np.asarray(sigma_ph, dtype=np.float64).reshape(-1, self.dlambda.shape[0])


def slab(n_layers, n_species=3, ld=None, dens=2.0e12, thick=1.0e5):
    ld = ld or n_layers
    n = np.zeros((n_species, ld))
    n[:, :n_layers] = dens
    dz = np.full(ld, thick)
    return n, dz


def test_transparent_atmosphere_is_the_plain_quadrature(oracle):
    """sigma_ext = 0: tau = 0 everywhere, k_ph = t_f sum_b J0 sigma dlambda at every layer."""
    rng = np.random.default_rng(1)
    nb, L = 37, 9
    dl = rng.uniform(0.5, 2.0, nb)
    ph = P(dl, [0, 2], np.zeros((2, nb)), rng.uniform(0, 1e-17, (4, nb)))
    n, dz = slab(L)
    j0 = rng.uniform(1e9, 1e12, (1, nb))
    k, tau = oracle.photo_rates(ph, n, dz, j0, None, [0.6], [0.5], 1, L, want_tau=True)
    want = 0.5 * (ph.sigma_ph * (j0[0] * dl)[None, :]).sum(axis=1)
    assert np.all(tau == 0.0)
    assert np.allclose(k, want[:, None] * np.ones((1, L)), rtol=2e-15, atol=0)


def test_grey_uniform_slab_matches_beer_lambert_closed_form(oracle):
    """One absorber of constant density and a wavelength-independent cross-section: the optical depth at the
    centre of layer k (counted from the bottom) is kappa dz ((L - 1 - k) + 1/2) and
    k_ph(k) = t_f J0 sigma_ph Lambda exp(-tau_k / mu)  with Lambda the total width of the bins."""
    nb, L = 11, 20
    dl = np.linspace(0.7, 1.3, nb)
    sig_e, sig_p, dens, thick, mu, tf, j0v = 3.0e-18, 1.1e-18, 2.0e12, 1.0e5, 0.4, 1.0, 5.0e11
    ph = P(dl, [1], np.full((1, nb), sig_e), np.full((1, nb), sig_p))
    n, dz = slab(L, dens=dens, thick=thick)
    n[0] = 7e30                                            # a non-absorber must not matter
    k, tau = oracle.photo_rates(ph, n, dz, np.full((1, nb), j0v), None, [mu], [tf], 1, L, want_tau=True)
    depth = (L - 1 - np.arange(L) + 0.5) * sig_e * dens * thick
    assert np.allclose(tau, depth[None, :] * np.ones((nb, 1)), rtol=1e-15)
    want = tf * j0v * sig_p * dl.sum() * np.exp(-depth / mu)
    assert np.allclose(k[0], want, rtol=1e-14, atol=0)
    assert np.all(np.diff(k[0]) > 0), "the rate constant decreases downwards (layer 0 is the bottom)"


def test_one_bin_cross_section_reads_the_actinic_flux_of_that_bin(oracle):
    rng = np.random.default_rng(3)
    nb, L = 16, 6
    dl = rng.uniform(0.5, 2.0, nb)
    sig_e = rng.uniform(0, 4e-18, (2, nb))
    sp = np.zeros((1, nb))
    sp[0, 5] = 2.0e-17
    ph = P(dl, [0, 1], sig_e, sp)
    n, dz = slab(L)
    n *= rng.uniform(0.5, 2.0, n.shape)
    j0 = rng.uniform(1e9, 1e12, (1, nb))
    jd = rng.uniform(0, 1e9, (nb, L))
    k, tau = oracle.photo_rates(ph, n, dz, j0, jd, [0.8], [1.0], 1, L, want_tau=True)
    flux = j0[0, 5] * np.exp(-tau[5] / 0.8) + jd[5]
    assert np.allclose(k[0], flux * 2.0e-17 * dl[5], rtol=1e-15)
    # and tau itself, layer by layer from the top, by hand
    kap = sig_e[0, 5] * n[0] + sig_e[1, 5] * n[1]
    above = np.concatenate([np.cumsum((kap * dz)[::-1])[::-1][1:], [0.0]])
    assert np.allclose(tau[5], above + 0.5 * kap * dz, rtol=1e-15)


def test_invariances_and_linearity(oracle):
    rng = np.random.default_rng(4)
    nb, L, A = 23, 8, 2
    dl = rng.uniform(0.5, 2.0, nb)
    ph = P(dl, [0, 2], rng.uniform(0, 5e-18, (2, nb)), rng.uniform(0, 1e-17, (3, nb)))
    n = rng.uniform(1e11, 1e13, (3, A * L))
    dz = rng.uniform(5e4, 2e5, A * L)
    j0 = rng.uniform(1e9, 1e12, (A, nb))
    jd = rng.uniform(0, 1e10, (nb, A * L))
    mu, tf = np.array([0.5, 0.9]), np.array([1.0, 0.5])
    base = oracle.photo_rates(ph, n, dz, j0, jd, mu, tf, A, L)
    # tau / mu only: scaling the extinction and mu together changes nothing
    ph2 = P(dl, [0, 2], 3.0 * ph.sigma_ext, ph.sigma_ph)
    assert np.allclose(oracle.photo_rates(ph2, n, dz, j0, jd, 3.0 * mu, tf, A, L), base, rtol=1e-14)
    # the same for density x thickness
    assert np.allclose(oracle.photo_rates(ph, 4.0 * n, dz / 4.0, j0, jd, mu, tf, A, L), base, rtol=1e-14)
    # linear in (J0, J_diff), in sigma_ph and in t_f
    assert np.allclose(oracle.photo_rates(ph, n, dz, 2 * j0, 2 * jd, mu, tf, A, L), 2 * base, rtol=1e-14)
    ph3 = P(dl, [0, 2], ph.sigma_ext, 5.0 * ph.sigma_ph)
    assert np.allclose(oracle.photo_rates(ph3, n, dz, j0, jd, mu, 0.2 * tf, A, L), base, rtol=1e-14)
    # the diffuse term alone: J0 = 0 gives t_f sum_b J_diff sigma dlambda, no attenuation
    only = oracle.photo_rates(ph, n, dz, 0 * j0, jd, mu, tf, A, L)
    want = np.repeat(tf, L)[None, :] * ((ph.sigma_ph * dl[None, :]) @ jd)
    assert np.allclose(only, want, rtol=1e-14)
    # atmospheres are independent: the second one alone gives the same numbers
    solo = oracle.photo_rates(ph, n[:, L:].copy(), dz[L:].copy(), j0[1:], jd[:, L:].copy(), mu[1:], tf[1:], 1, L)
    assert np.array_equal(solo, base[:, L:])
    # night side
    assert np.all(oracle.photo_rates(ph, n, dz, j0, jd, mu, 0 * tf, A, L) == 0.0)


def test_synthetic_tables_give_rates_in_the_range_the_configs_draw(oracle, network):
    """The stand-in spectra and cross-sections produce J values that overlap BASELINE config 1's range
    (1e-10..1e-2 s^-1) near the top of the atmosphere and vanish at depth."""
    from paper_2512_06729_b200 import synth
    net = network(2)
    atm = synth.config_atmosphere(2, net)
    ph = synth.make_photo(31, net, n_bins=400)
    dz, j0, jd, mu, tf = synth.make_irradiation(32, net, atm, ph, with_diffuse=False)
    k = oracle.photo_rates(ph, atm.n, dz, j0, None, mu, tf, 1, atm.ncol)
    top, bottom = k[:, atm.ncol - 1], k[:, 0]
    assert np.all(top > 0) and np.median(top) > 1e-10 and np.median(top) < 1e2
    assert np.all(bottom <= top) and np.median(bottom) < 1e-30
