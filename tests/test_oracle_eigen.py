"""Pins for the oracle's k-eigenvalue mode (DESIGN.md Appendix H).  (H-a) one-group infinite
medium: every particle is absorbed sooner or later, so each generation's k has the expectation nu Sigma_f / Sigma_a
whatever the spatial distribution; (H-b) a non-scattering bare slab with a uniform isotropic source: generation 0 has
k = nu Sigma_f / Sigma_t * (1 - P_esc) with the textbook escape probability P_esc = (1/2 - E_3(tau)) / tau, and the
track length per source particle is (1 - P_esc) / Sigma_t; (H-c) multigroup infinite medium with one fission spectrum:
the fission operator has rank one, so from generation 1 on E[k] = (nu Sigma_f)^T (diag Sigma_t - S^T)^-1 chi;
(H-d) nothing depends on the order in which a generation's bank is processed."""
import numpy as np
import pytest
from scipy.special import expn

from oracle import Oracle
from workloads import configs as W


def test_Ha_one_group_infinite_medium_k_is_nu_sigf_over_siga():
    p = W.as_eigenvalue(W.config0_infinite_medium(n_histories=4000, n_batches=1))
    o = Oracle(p)
    N, n_in, n_act = 4000, 5, 35
    k = o.run_eigenvalue(N, p.seed, n_in, n_act)
    assert k.shape == (40,) and np.all(k > 0.6) and np.all(k < 1.0)
    # per source particle: fission with probability 0.4, then exactly 2 children -> variance 4 * 0.4 * 0.6
    sigma_g = np.sqrt(0.96 / N)
    assert np.all(np.abs(k - 0.8) < 5.0 * sigma_g * 1.05)
    assert abs(k.mean() - 0.8) < 4.0 * sigma_g / np.sqrt(40)
    wa, na = o.census_after()
    assert abs(na[0] / 39 - N) < 5.0 * np.sqrt(N)             # the control between generations holds the population at N
    assert wa[0] == float(na[0])                              # ... with unit weights
    # flux per source particle in the single (space, time) bin: 1 / Sigma_a = 2 cm, batch = active generation
    mean, sdev = o.tallies()
    assert mean.shape == (1, 1, 1, 1, 1)
    assert abs(mean.ravel()[0] - 2.0) < 4.0 * sdev.ravel()[0] and 0 < sdev.ravel()[0] < 0.05
    c = o.counters()
    assert c["histories"] == N * n_act and c["batches"] == n_act and c["census_events"] == 0


@pytest.mark.parametrize("thickness", [0.5, 2.0, 6.0])
def test_Hb_bare_slab_first_generation_against_the_escape_probability(thickness):
    N = 200_000
    p = W.bare_slab_absorber(thickness=thickness, n_histories=N)
    o = Oracle(p)
    k = o.run_eigenvalue(N, p.seed, 0, 1)
    tau = 1.0 * thickness
    p_esc = (0.5 - expn(3, tau)) / tau
    p_fis = 0.4 * (1.0 - p_esc)                               # Sigma_f / Sigma_t = 0.4, no scattering
    var = 6.5 * p_fis - (2.5 * p_fis) ** 2                    # n = 2 or 3 with equal probability: E[n^2] = 6.5
    assert abs(k[0] - 2.5 * p_fis) < 4.0 * np.sqrt(var / N)
    mean, _ = o.tallies()
    flux = mean.sum()                                         # cm of track per source particle
    # track length per particle: exponential truncated by the faces; its mean is (1 - P_esc) / Sigma_t
    assert abs(flux - (1.0 - p_esc)) < 4.0 * np.sqrt(1.0 / N)
    prof = mean.ravel()
    assert np.allclose(prof, prof[::-1], rtol=0.05)           # symmetric in x
    c = o.counters()
    assert c["leak"] / N == pytest.approx(p_esc, abs=4.0 * np.sqrt(p_esc * (1 - p_esc) / N))


def test_Hc_multigroup_rank_one_fission_operator():
    p = W.as_eigenvalue(W.infinite_medium_multigroup(material=0, n_histories=3000, n_batches=1))
    st, sf, nu, chi, ss = p.sigma_t[0], p.sigma_f[0], p.nu[0], p.chi[0], p.sigma_s[0]
    assert sf.sum() > 0 and chi.sum() == pytest.approx(1.0)
    phi = np.linalg.solve(np.diag(st) - ss.T, chi)            # Sigma_t phi_g = sum_g' Sigma_s[g'->g] phi_g' + chi_g
    k_exact = float((nu * sf) @ phi)
    o = Oracle(p)
    N = 3000
    k = o.run_eigenvalue(N, p.seed, 1, 40)
    kk = k[1:]                                                # generation 0 starts from the source pdf, not chi
    se = kk.std(ddof=1) / np.sqrt(len(kk))
    assert abs(kk.mean() - k_exact) < 4.0 * se and se < 0.01
    # group flux per source particle = phi (active generations only)
    mean, sdev = o.tallies()
    z = (mean.ravel() - phi) / sdev.ravel()
    assert np.abs(z).max() < 4.5


def test_Hd_order_independence_and_argument_checks():
    p = W.as_eigenvalue(W.config3_pin_lattice(n_histories=1500, n_batches=1))
    a = Oracle(p); ka = a.run_eigenvalue(1500, p.seed, 2, 4)
    b = Oracle(p); kb = b.run_eigenvalue(1500, p.seed, 2, 4, reverse_order=True)
    assert np.array_equal(ka, kb)
    sa, _ = a.tally_sums(); sb, _ = b.tally_sums()
    assert np.abs(sa - sb).max() <= 1e-12 * np.abs(sa).max()
    ca, cb = a.counters(), b.counters()
    for key in ("collisions", "surf_hits", "children", "pc_removed", "pc_added"):
        assert ca[key] == cb[key]
    assert 0.5 < ka[2:].mean() < 1.3                          # the lattice is built for k_inf ~ 0.95, less axial leakage
    c = Oracle(p); kc = c.run_eigenvalue(1500, p.seed + 1, 2, 4)
    assert not np.array_equal(ka, kc)
    with pytest.raises(RuntimeError):
        a.run_eigenvalue(1500, p.seed, 0, 0)
