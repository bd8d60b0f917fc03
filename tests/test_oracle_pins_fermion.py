"""Pins for the fermionic LPA loop at finite chemical potential (orc_lpa_fermion, DESIGN.md
reading A22) against textbook closed forms:
  * flat spatial regulator on [0,k]:  I_F = C (2 k^(d+2)/d) (1/d-free radial integral) T sum_n Re 1/((nu_n + i mu)^2 + E^2) and
        T sum_{all n} 1/((nu_n + i mu)^2 + E^2) = (1 - n_F(E - mu) - n_F(E + mu)) / (2E),   n_F(x) = 1/(e^(x/T) + 1)
    with the truncation tail sum_{n > N} [1/(n + z1) - 1/(n + z2)] = psi(N+1+z2) - psi(N+1+z1) (mpmath digamma);
  * mu = 0: tanh(E/2T)/(2E);  the m2 derivative by mpmath differentiation of the closed form;
  * exponential spatial regulator: the same closed form under an mpmath radial quadrature.
CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle

PI = math.pi


def truncated_fermi_sum(E2, T, mu, N):
    """T sum_{n=-N-1..N} 1/((nu_n + i mu)^2 + E2), nu_n = (2n+1) pi T  (real).  mpmath, closed form."""
    E = mp.sqrt(mp.mpf(E2))
    nF = lambda x: 1 / (mp.exp(x / T) + 1)
    full = (1 - nF(E - mu) - nF(E + mu)) / (2 * E)
    # 1/((nu + i mu)^2 + E^2) = [1/(nu + i(mu - E)) - 1/(nu + i(mu + E))] / (2 i E),  nu = 2 pi T (n + 1/2)
    z1 = mp.mpf(1) / 2 + 1j * (mu - E) / (2 * mp.pi * T)
    z2 = mp.mpf(1) / 2 + 1j * (mu + E) / (2 * mp.pi * T)
    tail = (mp.digamma(N + 1 + z2) - mp.digamma(N + 1 + z1)) / (2j * E) / (2 * mp.pi * T)   # sum_{n > N}
    return full - 2 * T * mp.re(tail)


def test_truncated_sum_closed_form_is_the_finite_sum():
    """The closed form used as the pin, checked against the finite sum it stands for (both in mpmath, 30 digits)."""
    mp.mp.dps = 30
    for T, mu, E2, N in ((0.1, 0.3, 1.7, 5), (0.05, 0.9, 0.8, 12), (0.3, 0.0, 2.0, 3)):
        direct = T * sum(mp.re(1 / (((2 * n + 1) * mp.pi * T + 1j * mu) ** 2 + E2)) for n in range(-N - 1, N + 1))
        assert abs(truncated_fermi_sum(E2, T, mu, N) / direct - 1) < mp.mpf(10) ** -25


@pytest.mark.parametrize("d", [3, 4])
@pytest.mark.parametrize("T,mu,n_max", [(0.1, 0.3, 10), (0.05, 0.9, 20), (0.3, 0.0, 4), (0.02, 1.3, 30)])
def test_fermion_litim_closed_form(d, T, mu, n_max):
    mp.mp.dps = 30
    k, C = 1.1, 0.37
    xq, wq = oracle.gl_rule(32, 0.0, k)
    m2 = np.array([-0.4, 0.0, 0.3, 2.5, 40.0])
    I, dI, dmin, sens, sens_d = oracle.lpa_fermion(d, T, n_max, mu, C, oracle.REG_LITIM, 1, k, xq, wq, m2)
    for j, m in enumerate(m2):
        E2 = k * k + m
        ref = C * (2 * k ** (d + 2) / d) * truncated_fermi_sum(E2, T, mu, n_max)
        assert abs(I[j] - float(ref)) <= 1e-13 * sens[j], (j, I[j], float(ref))
        dref = C * (2 * k ** (d + 2) / d) * mp.diff(lambda e2: truncated_fermi_sum(e2, T, mu, n_max), mp.mpf(E2))
        assert abs(dI[j] - float(dref)) <= 1e-12 * sens_d[j], (j, dI[j], float(dref))
        # |D| at the node closest to the pole: q-independent for the flat regulator
        nu0 = PI * T
        assert abs(dmin[j] - abs(complex(nu0 * nu0 - mu * mu + E2, 2 * nu0 * mu)) / (k * k)) < 1e-13 * (1 + dmin[j])


def test_fermion_mu0_tanh_limit_and_symmetry_in_mu():
    k, T = 1.0, 0.2
    xq, wq = oracle.gl_rule(24, 0.0, k)
    m2 = np.array([0.5])
    I_big = oracle.lpa_fermion(3, T, 20000, 0.0, 1.0, oracle.REG_LITIM, 1, k, xq, wq, m2)[0][0]
    E = math.sqrt(1.5)
    ref = (2.0 / 3.0) * math.tanh(E / (2 * T)) / (2 * E)
    assert abs(I_big / ref - 1) < 5e-5                      # tail of the truncated sum ~ 1/(2 pi^2 T N E-ish)
    a = oracle.lpa_fermion(3, T, 7, 0.4, 1.0, oracle.REG_EXP_POLY, 1, k, xq, wq, m2)
    b = oracle.lpa_fermion(3, T, 7, -0.4, 1.0, oracle.REG_EXP_POLY, 1, k, xq, wq, m2)
    assert a[0][0] == b[0][0] and a[1][0] == b[1][0]        # nu + i mu or nu - i mu (the paper's p0f - i mu): same real part


def test_fermion_exp_regulator_vs_mpmath_quadrature():
    mp.mp.dps = 25
    k, T, mu, n_max, d, C = 1.0, 0.15, 0.5, 8, 3, 1.0
    xq, wq = oracle.gl_rule(96, 0.0, 8.0 * k)
    m2 = np.array([0.2, 1.5])
    I, dI, _, sens, _ = oracle.lpa_fermion(d, T, n_max, mu, C, oracle.REG_EXP_POLY, 1, k, xq, wq, m2, zk=1.2, eta=0.1)
    for j, m in enumerate(m2):
        def integrand(q):
            x = q * q / (k * k)
            R = 1.2 * k * k * mp.exp(-x)
            Rd = 1.2 * (2 * k * k * mp.exp(-x) * (1 + x) - 0.1 * k * k * mp.exp(-x))
            return q ** (d - 1) * Rd * truncated_fermi_sum(q * q + R + m, T, mu, n_max)
        ref = C * mp.quad(integrand, [0, 0.5, 1, 2, 4, 8])
        assert abs(I[j] / float(ref) - 1) < 1e-11
