"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pins one piece of oracle/emri_oracle.cpp to
something other than itself: a library routine of different construction (scipy/mpmath/numpy), a
closed form, an identity, a limit, a convergence order, or brute force on a tiny input.
"""
import math
import os

import mpmath
import numpy as np
import pytest
import scipy.integrate
import scipy.optimize
import scipy.special

from paper_2311_17174_b200 import workloads as W

MSUN = 4.925490947e-6
GPC = 1.0292712503e17
AU = 499.004783836
YEAR = 31557600.0
TWOPI = 2.0 * math.pi


def base_row(**kw):
    """Fig. 1 / Fig. 2 geometry of the paper: M=1e6, mu=10, thS=pi/4, phS=0,
    thK=pi/8, phK=0, lambda=pi/6, D=1 Gpc; nu0 chosen well below plunge."""
    p = np.zeros(W.NPAR)
    p[W.P_M], p[W.P_MU], p[W.P_A], p[W.P_E0] = 1e6, 10.0, 0.4, 0.3
    p[W.P_NU0] = 1.0e-3
    p[W.P_PHI0], p[W.P_GAM0], p[W.P_ALP0] = 0.3, 1.1, 2.2
    p[W.P_LAM], p[W.P_THS], p[W.P_PHS], p[W.P_THK], p[W.P_PHK] = math.pi / 6, math.pi / 4, 0.0, math.pi / 8, 0.0
    p[W.P_DL], p[W.P_XI0], p[W.P_NXI], p[W.P_DELT] = 1.0, 1.0, 0.0, 0.0
    for k, v in kw.items():
        p[getattr(W, "P_" + k)] = v
    return p


def circ_diff(a, b):
    """difference of two phases in cycles, wrapped to [-1/2, 1/2)"""
    d = (a - b) % 1.0
    return d - (d >= 0.5)


# ------------------------------------------------------------------ Bessel (S5.6)
def test_bessel_against_scipy_and_mpmath(oracle):
    mpmath.mp.dps = 50
    worst = worst_hi = 0.0
    for n in range(1, 33):
        for e in (0.0, 1e-3, 0.05, 0.1, 0.3, 0.5, 0.7):
            for k in range(n - 2, n + 3):
                x = n * e
                got = oracle.bessel_j(k, x)
                ref = float(mpmath.besselj(k, mpmath.mpf(x)))
                assert got == pytest.approx(scipy.special.jv(k, x), rel=1e-12, abs=1e-300)
                if ref == 0.0:
                    assert got == 0.0
                elif e <= 0.5:
                    worst = max(worst, abs(got - ref) / abs(ref))
                else:
                    worst_hi = max(worst_hi, abs(got - ref) / abs(ref))
    # the alternating series loses ~1 digit in the configs' range e <= 0.5, ~2.5 digits at e = 0.7, n ~ 30
    assert worst < 5e-15 and worst_hi < 2e-13


def test_bessel_identities(oracle):
    for x in (0.3, 1.7, 4.0, 7.5):
        J = [oracle.bessel_j(k, x) for k in range(0, 60)]
        assert J[0] ** 2 + 2.0 * sum(v * v for v in J[1:]) == pytest.approx(1.0, abs=1e-13)
        for k in range(1, 30):
            assert J[k - 1] + J[k + 1] == pytest.approx(2.0 * k / x * J[k], rel=1e-10, abs=1e-18)
    assert oracle.bessel_j(0, 0.0) == 1.0 and oracle.bessel_j(3, 0.0) == 0.0
    assert oracle.bessel_j(-1, 0.4) == -oracle.bessel_j(1, 0.4)


# ------------------------------------------------------------------ Peters-Mathews brackets
def g_from_brackets(oracle, n, e):
    Ba, Bb, Bc = oracle.brackets(n, e)      # Bb already carries sqrt(1-e^2)
    return n ** 4 / 32.0 * (Ba * Ba + Bb * Bb + 4.0 / (3.0 * n * n) * Bc * Bc)


@pytest.mark.parametrize("e", [0.1, 0.2, 0.3, 0.4, 0.5, 0.6, 0.7])
def test_peters_mathews_power_sum(oracle, e):
    """sum_n g(n,e) = (1 + 73 e^2/24 + 37 e^4/96) / (1-e^2)^{7/2}  (BASELINE.json north_star)"""
    total = sum(g_from_brackets(oracle, n, e) for n in range(1, 201))
    closed = (1.0 + 73.0 * e * e / 24.0 + 37.0 * e ** 4 / 96.0) / (1.0 - e * e) ** 3.5
    assert total == pytest.approx(closed, rel=2e-10)


@pytest.mark.parametrize("n_max,e,bound", [(5, 0.1, 2e-5), (10, 0.3, 5e-5), (20, 0.4, 5e-5), (30, 0.5, 5e-8)])
def test_power_sum_truncation_at_config_nmax(oracle, n_max, e, bound):
    total = sum(g_from_brackets(oracle, n, e) for n in range(1, n_max + 1))
    closed = (1.0 + 73.0 * e * e / 24.0 + 37.0 * e ** 4 / 96.0) / (1.0 - e * e) ** 3.5
    assert 0.0 <= 1.0 - total / closed < bound


def test_brackets_at_zero_eccentricity(oracle):
    """R18: J_k(0) = delta_k0, so only n = 2 survives"""
    for n in range(1, 12):
        Ba, Bb, Bc = oracle.brackets(n, 0.0)
        want = 1.0 if n == 2 else 0.0
        assert (Ba, Bb, Bc) == (want, want, 0.0)


# ------------------------------------------------------------------ plunge frequency
def test_nu_lso_closed_forms(oracle):
    M = 1e6
    assert oracle.nu_lso(M, 0.0) == pytest.approx(1.0 / (TWOPI * M * MSUN * 6.0 ** 1.5), rel=1e-15)
    e = 0.3
    assert oracle.nu_lso(M, e) == pytest.approx(((1 - e * e) / (6 + 2 * e)) ** 1.5 / (TWOPI * M * MSUN), rel=1e-15)
    # the input generator's copy of the same formula agrees (it places nu0 below plunge)
    assert W.nu_lso_hz(M, e) == pytest.approx(oracle.nu_lso(M, e), rel=1e-14)


# ------------------------------------------------------------------ cosmology / propagation (S1)
@pytest.mark.parametrize("DL", [0.5, 1.0, 3.0])
def test_redshift_and_lookback_against_scipy(oracle, DL):
    H0, Om = 67.4, 0.315
    tH = 3.0856775814913673e22 / (H0 * 1000.0)
    E = lambda z: math.sqrt(Om * (1 + z) ** 3 + 1 - Om)
    dL = lambda z: (1 + z) * tH * scipy.integrate.quad(lambda x: 1 / E(x), 0, z, epsabs=0, epsrel=1e-13)[0]
    z_ref = scipy.optimize.brentq(lambda z: dL(z) - DL * GPC, 0.0, 20.0, xtol=1e-15, rtol=1e-15)
    tlb_ref = tH * scipy.integrate.quad(lambda x: 1 / ((1 + x) * E(x)), 0, z_ref, epsabs=0, epsrel=1e-13)[0]
    z, tlb, dl_back = oracle.cosmology(DL)
    assert z == pytest.approx(z_ref, rel=1e-12)
    assert tlb == pytest.approx(tlb_ref, rel=1e-12)
    assert dl_back == pytest.approx(DL * GPC, rel=1e-13)


def test_survey_magnitudes_of_delay(oracle):
    z, tlb, _ = oracle.cosmology(1.0)
    assert z == pytest.approx(0.19724, abs=1e-5) and tlb == pytest.approx(7.858e16, rel=1e-3)
    s = oracle.walker_scalars(base_row(DELT=1e-15))
    assert s["dT"] == pytest.approx(-1e-15 * tlb, rel=1e-14) and abs(s["dT"]) < 80.0


def test_xi_gr_limits(oracle):
    """Eq. 6: Xi0 = 1 => Xi = 1 for every n; n = 0 => Xi = 1; z = 0 => Xi = 1"""
    for n in (0.0, 1.0, 2.5):
        assert oracle.xi(1.0, n, 0.7) == 1.0
    assert oracle.xi(0.8, 0.0, 0.7) == 1.0
    assert oracle.xi(0.8, 2.0, 0.0) == 1.0
    assert oracle.xi(0.8, 2.0, 0.5) == pytest.approx(0.8 + 0.2 / 1.5 ** 2, rel=1e-15)
    assert oracle.xi(0.8, 2.0, 1e9) == pytest.approx(0.8, rel=1e-12)


def test_walker_scalars_units(oracle):
    p = base_row(XI0=0.9, NXI=2.0)
    s = oracle.walker_scalars(p)
    assert s["Ms"] == pytest.approx(1e6 * MSUN, rel=1e-15) and s["mus"] == pytest.approx(10 * MSUN, rel=1e-15)
    assert s["Ds"] == pytest.approx(GPC, rel=1e-15)
    assert s["amp"] == pytest.approx(s["mus"] / (s["Xi"] * s["Ds"]), rel=1e-15)
    assert s["Xi"] == pytest.approx(0.9 + 0.1 / (1 + s["z"]) ** 2, rel=1e-14)
    assert s["status"] == 0
    for bad in (dict(M=-1.0), dict(E0=1.0), dict(A=1.5), dict(NU0=0.0), dict(DL=0.0), dict(MU=float("nan"))):
        assert oracle.walker_scalars(base_row(**bad))["status"] == 1


# ------------------------------------------------------------------ right-hand side (S2)
def test_rhs_leading_order_chirp_coefficient(oracle):
    """a=0, e=0, PN terms off: nu' = K nu^{11/3} with the chirp-mass form
    K = (96/5) pi^{8/3} Mc^{5/3} for GW frequency f = 2 nu, i.e. (48/5) pi^{8/3} 2^{11/3} mu M^{2/3}"""
    p = base_row(A=0.0, E0=0.0)
    nu = 2.0e-3
    f = oracle.rhs(p, [0.1, nu, 0.2, 0.0, 0.3], pn_mask=0)
    M, mu = 1e6 * MSUN, 10 * MSUN
    K = 48.0 / 5.0 * math.pi ** (8.0 / 3.0) * 2.0 ** (11.0 / 3.0) * mu * M ** (2.0 / 3.0)
    assert f[1] == pytest.approx(K * nu ** (11.0 / 3.0), rel=1e-14)
    # same thing from the standard chirp df/dt = (96/5) pi^{8/3} Mc^{5/3} f^{11/3}, f = 2 nu
    Mc = mu ** 0.6 * M ** 0.4
    fgw = 2 * nu
    assert 2.0 * f[1] == pytest.approx(96.0 / 5.0 * math.pi ** (8.0 / 3.0) * Mc ** (5.0 / 3.0) * fgw ** (11.0 / 3.0), rel=1e-13)
    assert f[0] == nu and f[3] == 0.0 and f[4] == 0.0


def test_rhs_1pn_circular_coefficient(oracle):
    """1PN circular term: 1273/336 = 6 - 743/336 (radial-to-azimuthal frequency shift 3u twice,
    plus the standard -743/336 chirp coefficient)"""
    p = base_row(A=0.0, E0=0.0)
    nu = 2.0e-3
    f0 = oracle.rhs(p, [0, nu, 0, 0, 0], pn_mask=0)[1]
    f1 = oracle.rhs(p, [0, nu, 0, 0, 0], pn_mask=1)[1]
    u = (TWOPI * 1e6 * MSUN * nu) ** (2.0 / 3.0)
    assert f1 / f0 - 1.0 == pytest.approx((6.0 - 743.0 / 336.0) * u, rel=1e-12)


def test_rhs_eccentric_newtonian_is_peters(oracle):
    """0PN: nu'(e)/nu'(0) = Peters' enhancement f(e); e' = Peters' de/dt with a = (M/(2 pi nu)^2)^{1/3}"""
    nu = 1.5e-3
    M, mu = 1e6 * MSUN, 10 * MSUN
    for e in (0.1, 0.4, 0.7):
        p = base_row(A=0.0)
        f = oracle.rhs(p, [0, nu, 0, e, 0], pn_mask=0)
        f_circ = oracle.rhs(p, [0, nu, 0, 0.0, 0], pn_mask=0)
        enh = (1 + 73 / 24 * e * e + 37 / 96 * e ** 4) / (1 - e * e) ** 3.5
        assert f[1] / f_circ[1] == pytest.approx(enh, rel=1e-13)
        a_sma = (M / (TWOPI * nu) ** 2) ** (1.0 / 3.0)
        dedt = -304.0 / 15.0 * e * mu * M * M / a_sma ** 4 / (1 - e * e) ** 2.5 * (1 + 121.0 / 304.0 * e * e)
        assert f[3] == pytest.approx(dedt, rel=1e-13)


def test_rhs_precession_limits(oracle):
    """gamma~' -> 3 (2 pi nu) u/(1-e^2) (Schwarzschild periapsis advance), alpha' = 2 a M (2 pi nu)^2
    (1-e^2)^{-3/2} (Lense-Thirring), spin part of gamma~' = -3 cos(lambda) alpha'"""
    nu, e, a, lam = 1.0e-3, 0.25, 0.6, 0.7
    p = base_row(A=a, LAM=lam)
    M = 1e6 * MSUN
    x = TWOPI * M * nu
    u, q = x ** (2.0 / 3.0), 1 - e * e
    y = [0, nu, 0, e, 0]
    f00 = oracle.rhs(p, y, pn_mask=0)
    f10 = oracle.rhs(p, y, pn_mask=1)
    f01 = oracle.rhs(p, y, pn_mask=2)
    assert TWOPI * f00[2] == pytest.approx(3 * TWOPI * nu * u / q, rel=1e-13)
    assert TWOPI * f01[4] == pytest.approx(2 * a * M * (TWOPI * nu) ** 2 * q ** -1.5, rel=1e-13)
    assert f01[2] - f00[2] == pytest.approx(-3 * math.cos(lam) * f01[4], rel=1e-12)
    assert f10[2] / f00[2] - 1 == pytest.approx(0.25 * u / q * (26 - 15 * e * e), rel=1e-11)
    assert f00[4] == 0.0


def test_rhs_spin_flux_coefficient_73_12(oracle):
    """circular spin-orbit correction of the flux: -(73/12) a cos(lambda) x (known test-mass value)"""
    nu, a, lam = 1.0e-3, 0.5, 0.4
    p = base_row(A=a, LAM=lam, E0=0.0)
    y = [0, nu, 0, 0.0, 0]
    f0 = oracle.rhs(p, y, pn_mask=0)[1]
    f2 = oracle.rhs(p, y, pn_mask=2)[1]
    x = TWOPI * 1e6 * MSUN * nu
    assert f2 / f0 - 1 == pytest.approx(-73.0 / 12.0 * a * math.cos(lam) * x, rel=1e-11)


def test_rhs_full_is_sum_of_parts(oracle):
    """the PN switches only remove terms: full - 0PN = (1PN - 0PN) + (spin - 0PN) for nu', e', gamma~'"""
    p = base_row(A=0.7, LAM=1.0)
    y = [0.1, 1.3e-3, 0.2, 0.35, 0.3]
    f = {m: oracle.rhs(p, y, pn_mask=m) for m in range(4)}
    for c in (1, 3):
        assert f[3][c] - f[0][c] == pytest.approx((f[1][c] - f[0][c]) + (f[2][c] - f[0][c]), rel=1e-9)


# ------------------------------------------------------------------ RK4 orbit (S3)
def test_orbit_0pn_circular_chirp_closed_form(oracle):
    """a=0, e=0, PN off: nu(t) = nu0 (1 - t/tau)^{-3/8}, Phi(t) = Phi0 + 2 pi nu0 tau (8/5)[1 - (1-t/tau)^{5/8}]"""
    p = base_row(A=0.0, E0=0.0, NU0=1.2e-3, PHI0=0.7)
    N, dt, S = 1 << 18, 15.0, 256
    orb = oracle.orbit(p, N, dt, S, pn_mask=0)
    assert orb["status"] == 0
    M, mu = 1e6 * MSUN, 10 * MSUN
    K = 96.0 / (10.0 * math.pi) * mu / M ** 3 * (TWOPI * M) ** (11.0 / 3.0)
    nu0 = p[W.P_NU0]
    tau = 3.0 / (8.0 * K * nu0 ** (8.0 / 3.0))
    j = np.arange(-1, orb["Nn"] - 1)
    t = j * S * dt
    nu_cf = nu0 * (1 - t / tau) ** -0.375
    np.testing.assert_allclose(orb["val"][1], nu_cf, rtol=2e-13)
    # closed-form phase in cycles, evaluated in 50-digit arithmetic so that the frac() is exact
    mpmath.mp.dps = 50
    for jj in (0, 1, 2, 100, orb["Nn"] - 1):
        tt = mpmath.mpf(float(t[jj]))
        ph = mpmath.mpf(0.7) / (2 * mpmath.pi) + mpmath.mpf(nu0) * tau * mpmath.mpf(8) / 5 * (1 - (1 - tt / tau) ** mpmath.mpf(0.625))
        assert abs(circ_diff(orb["val"][0][jj], float(ph % 1))) < 2e-10
    assert np.all(orb["val"][3] == 0.0) and np.all(orb["val"][4] == p[W.P_ALP0] / TWOPI)


def test_orbit_1pn_circular_time_of_frequency(oracle):
    """1PN on, a=0, e=0: t(nu) = int dnu / (K nu^{11/3} (1 + c1 nu^{2/3})) by independent quadrature"""
    p = base_row(A=0.0, E0=0.0, NU0=1.2e-3)
    N, dt, S = 1 << 18, 15.0, 256
    orb = oracle.orbit(p, N, dt, S, pn_mask=1)
    M, mu = 1e6 * MSUN, 10 * MSUN
    K = 96.0 / (10.0 * math.pi) * mu / M ** 3 * (TWOPI * M) ** (11.0 / 3.0)
    c1 = (6.0 - 743.0 / 336.0) * (TWOPI * M) ** (2.0 / 3.0)
    for jj in (0, 300, orb["Nn"] - 1):
        nu = orb["val"][1][jj]
        t_ref = scipy.integrate.quad(lambda v: 1.0 / (K * v ** (11.0 / 3.0) * (1 + c1 * v ** (2.0 / 3.0))),
                                     p[W.P_NU0], nu, epsabs=0, epsrel=1e-13)[0]
        assert t_ref == pytest.approx((jj - 1) * S * dt, rel=1e-10, abs=1e-4)


def test_orbit_peters_invariant_along_0pn_flow(oracle):
    """Peters 1964: a(e) ~ e^{12/19} (1+121e^2/304)^{870/2299}/(1-e^2), and a ~ nu^{-2/3}"""
    p = base_row(A=0.0, E0=0.45, NU0=9e-4)
    orb = oracle.orbit(p, 1 << 19, 15.0, 256, pn_mask=0)
    assert orb["status"] == 0
    nu, e = orb["val"][1], orb["val"][3]
    inv = e ** (12 / 19) * (1 + 121 * e * e / 304) ** (870 / 2299) / (1 - e * e) * nu ** (2 / 3)
    assert np.ptp(inv) / inv[0] < 1e-12
    assert e[-1] < e[0] and nu[-1] > nu[0]


def test_orbit_against_dop853(oracle):
    """full model vs scipy DOP853 (rtol 1e-13) driven by the oracle's right-hand side"""
    cfg = W.CONFIGS[2]
    P = W.draw_params(cfg, K=3)
    for p in P:
        N, dt, S = 1 << 19, 15.0, 256
        orb = oracle.orbit(p, N, dt, S)
        assert orb["status"] == 0
        y0 = [orb["val"][q][1] for q in range(5)]
        T = (orb["Nn"] - 2) * S * dt
        sol = scipy.integrate.solve_ivp(lambda t, y: oracle.rhs(p, y), (0.0, T), y0, method="DOP853",
                                        rtol=1e-13, atol=[1e-9, 1e-19, 1e-9, 1e-16, 1e-9])
        yT = sol.y[:, -1]
        assert orb["val"][1][-1] == pytest.approx(yT[1], rel=5e-12)
        assert orb["val"][3][-1] == pytest.approx(yT[3], rel=5e-11, abs=1e-14)
        for q in (0, 2, 4):
            assert abs(circ_diff(orb["val"][q][-1], yT[q] % 1.0)) < 2e-8


def test_rk4_is_fourth_order(oracle_ld):
    """halving the step cuts the phase error at the last node 16x (80-bit build, where rounding does not
    mask it; at the default stride S=256 the truncation error is ~4e-15 cycles, below fp64 rounding)"""
    p = W.draw_params(W.CONFIGS[1], K=1)[0]
    N, dt = 1 << 19, 15.0
    ref = oracle_ld.orbit(p, N, dt, 64)
    errs = [abs(circ_diff(oracle_ld.orbit(p, N, dt, S)["val"][0][-2], ref["val"][0][-2])) for S in (8192, 4096, 2048, 1024)]
    assert errs[0] > 1e-10
    for a, b in zip(errs[:-1], errs[1:]):
        assert 14.0 < a / b < 18.0


def test_orbit_guard_node_and_increments(oracle):
    """node -1 + inc[-1] = node 0; node j + inc[j] = node j+1 (mod 1 for the angles); slopes = rhs"""
    p = W.draw_params(W.CONFIGS[2], K=1)[0]
    orb = oracle.orbit(p, 1 << 16, 15.0, 256)
    v, inc, sl = orb["val"], orb["inc"], orb["slope"]
    for q in (0, 2, 4):
        assert np.max(np.abs(circ_diff(v[q][:-1] + inc[q][:-1], v[q][1:]))) < 1e-14
    for q in (1, 3):
        np.testing.assert_allclose(v[q][:-1] + inc[q][:-1], v[q][1:], rtol=1e-15)
    for jj in (0, 1, 17, orb["Nn"] - 1):
        np.testing.assert_array_equal(sl[:, jj], oracle.rhs(p, v[:, jj]))
    assert np.all((v[0] >= 0) & (v[0] < 1) & (v[2] >= 0) & (v[2] < 1) & (v[4] >= 0) & (v[4] < 1))
    np.testing.assert_allclose(v[:, 1], [(p[W.P_PHI0] / TWOPI) % 1, p[W.P_NU0], (p[W.P_GAM0] / TWOPI) % 1, p[W.P_E0],
                                         (p[W.P_ALP0] / TWOPI) % 1], rtol=1e-15)


def test_orbit_plunge_truncation(oracle):
    """R8: nu0 just below nu_LSO => status bit 2, nodes from j_pl on are copies of node j_pl - 1"""
    p = base_row(E0=0.2, A=0.3)
    p[W.P_NU0] = 0.97 * oracle.nu_lso(1e6, 0.2)
    orb = oracle.orbit(p, 1 << 17, 15.0, 256)
    assert orb["status"] == 2 and 0 < orb["jpl"] < orb["Nn"] - 1
    jj = orb["jpl"] + 1   # column of node j_pl
    assert orb["val"][1][jj - 1] < oracle.nu_lso(1e6, orb["val"][3][jj - 1])
    assert np.all(orb["val"][:, jj:] == orb["val"][:, jj - 1:jj]) and np.all(orb["inc"][:, jj:] == 0)
    hI, hII, st = oracle.waveform(p, 1 << 17, 15.0, 4)
    first_zero = (orb["jpl"] - 1) * 256
    assert st == 2 and np.all(hI[first_zero:] == 0) and np.all(hII[first_zero:] == 0) and np.any(hI[:first_zero] != 0)
    # already plunged at t = 0
    p[W.P_NU0] = 1.01 * oracle.nu_lso(1e6, 0.2)
    hI, hII, st = oracle.waveform(p, 1 << 12, 15.0, 4)
    assert st == 2 and not hI.any() and not hII.any()


# ------------------------------------------------------------------ Hermite (S4)
def test_hermite_reproduces_cubics(oracle):
    rng = np.random.default_rng(7)
    for _ in range(20):
        c = rng.standard_normal(4)
        Delta = 3840.0
        poly = lambda t: ((c[3] * t + c[2]) * t + c[1]) * t + c[0]
        dpoly = lambda t: (3 * c[3] * t + 2 * c[2]) * t + c[1]
        for s in (0.0, 0.1, 0.5, 0.77, 1.0):
            got = oracle.hermite1(poly(0.0), poly(1.0) - poly(0.0), dpoly(0.0) / Delta, dpoly(1.0) / Delta, Delta, s)
            assert got == pytest.approx(poly(s), rel=1e-13, abs=1e-13)


def test_orbit_at_matches_nodes_and_delay_split(oracle):
    p = base_row(DELT=1e-15)     # dT ~ -78.6 s: sample 0 falls into the guard interval -1... no: dT<0 => t' > t
    N, dt, S = 1 << 14, 15.0, 256
    orb = oracle.orbit(p, N, dt, S)
    sc = oracle.walker_scalars(p)
    idx = np.array([0, 1, 255, 256, 257, N - 1])
    got = oracle.orbit_at(p, N, dt, idx, S)
    # independent evaluation of the interpolant from the node arrays with plain float arithmetic
    for m, i in enumerate(idx):
        tprime = i * dt - sc["dT"]
        j = int(math.floor(tprime / (S * dt)))
        s = tprime / (S * dt) - j
        jj = j + 1
        for q in range(5):
            y = (orb["val"][q][jj] + (3 * s * s - 2 * s ** 3) * orb["inc"][q][jj]
                 + S * dt * ((s ** 3 - 2 * s * s + s) * orb["slope"][q][jj] + (s ** 3 - s * s) * orb["slope"][q][jj + 1]))
            assert got[q][m] == pytest.approx(y, rel=1e-10, abs=1e-12)
    # positive delay: first samples come from the backward guard interval
    p2 = base_row(DELT=-1e-15)
    got2 = oracle.orbit_at(p2, N, dt, np.array([0]), S)
    orb2 = oracle.orbit(p2, N, dt, S)
    assert got2[1][0] < orb2["val"][1][1]        # nu(t' < 0) < nu0


# ------------------------------------------------------------------ geometry (S5.2, S5.3, S5.7)
def _vec(th, ph):
    return np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])


def test_geometry_against_vector_algebra(oracle):
    rng = np.random.default_rng(11)
    z = np.array([0.0, 0.0, 1.0])
    for _ in range(300):
        thS, thK = np.arccos(rng.uniform(-0.999, 0.999, 2))
        phS, phK, alpha, phibar = rng.uniform(0, TWOPI, 4)
        lam = rng.uniform(0.01, math.pi - 0.01)
        p = base_row(THS=thS, PHS=phS, THK=thK, PHK=phK, LAM=lam)
        g = oracle.geometry(p, alpha, phibar)
        n, Sv = _vec(thS, phS), _vec(thK, phK)
        L = (Sv * math.cos(lam) + (z - Sv * math.cos(thK)) / math.sin(thK) * math.sin(lam) * math.cos(alpha)
             + np.cross(Sv, z) / math.sin(thK) * math.sin(lam) * math.sin(alpha))
        assert np.dot(L, L) == pytest.approx(1.0, abs=1e-14) and np.dot(L, Sv) == pytest.approx(math.cos(lam), abs=1e-14)
        Lo = np.array([g["sthL"] * math.cos(g["phL"]), g["sthL"] * math.sin(g["phL"]), g["cthL"]])
        np.testing.assert_allclose(Lo, L, atol=3e-15)
        Ln = np.dot(L, n)
        assert g["Ln"] == pytest.approx(Ln, abs=3e-15) and g["Sn"] == pytest.approx(np.dot(Sv, n), abs=3e-15)
        if 1 - Ln * Ln > 1e-4:
            rt = math.sqrt(1 - Ln * Ln)
            phat = (Sv - L * math.cos(lam)) / math.sin(lam)
            xhat = (L * Ln - n) / rt
            sinb = np.dot(phat, xhat)
            cosb = np.dot(phat, np.cross(L, n)) / rt
            assert g["sinb"] == pytest.approx(sinb, abs=2e-11) and g["cosb"] == pytest.approx(cosb, abs=2e-11)
            assert g["sinb"] ** 2 + g["cosb"] ** 2 == pytest.approx(1.0, abs=1e-10)
            assert g["beta"] == pytest.approx(math.atan2(sinb, cosb), abs=3e-11)
        zd = np.array([-math.sqrt(3) / 2 * math.cos(phibar), -math.sqrt(3) / 2 * math.sin(phibar), 0.5])
        assert g["cthd"] == pytest.approx(np.dot(zd, n), abs=3e-15)
        assert g["Npsi"] == pytest.approx(np.dot(L, zd) - Ln * np.dot(zd, n), abs=5e-15)
        assert g["Dpsi"] == pytest.approx(np.dot(n, np.cross(L, zd)), abs=5e-15)
        assert g["psi"] == pytest.approx(math.atan2(g["Npsi"], g["Dpsi"]), abs=1e-15)


def _detector_axes(phibar):
    """Explicit unit vectors of the rolling LISA frame (Cutler 1998; S5.7 with phibar0 = alphabar0 = 0), in ecliptic
    coordinates: the normal z_d is tilted 60 degrees from the ecliptic pole and follows the orbit; e2 points along the
    orbital motion and e1 = e2 x z_d completes the in-plane pair; the arms' frame (x_d, y_d) counter-rotates in that plane
    once per orbit, starting at t = 0 from x_d = -e2, y_d = e1 (which is what S5.7's phi_d says at phibar = 0:
    sin(th_d) cos(phi_d) = -n_y, sin(th_d) sin(phi_d) = (n_x + sqrt3 n_z)/2)."""
    zd = np.array([-math.sqrt(3) / 2 * math.cos(phibar), -math.sqrt(3) / 2 * math.sin(phibar), 0.5])
    e2 = np.array([-math.sin(phibar), math.cos(phibar), 0.0])
    e1 = np.cross(e2, zd)
    xd = -math.cos(phibar) * e2 - math.sin(phibar) * e1
    yd = -math.sin(phibar) * e2 + math.cos(phibar) * e1
    return xd, yd, zd


def test_detector_azimuth_against_rotating_frame(oracle):
    """phi_d is the azimuth of n^ in the rolling frame built from explicit axes: NO modulo (a quarter-turn slip, which
    would flip the sign of both channels, fails here)"""
    rng = np.random.default_rng(5)
    for _ in range(200):
        thS = math.acos(rng.uniform(-0.99, 0.99))
        phS, phibar = rng.uniform(0, TWOPI, 2)
        g = oracle.geometry(base_row(THS=thS, PHS=phS), 0.3, phibar)
        n = _vec(thS, phS)
        xd, yd, zd = _detector_axes(phibar)
        assert abs(np.dot(xd, yd)) < 1e-15 and abs(np.dot(xd, zd)) < 1e-15 and abs(np.dot(yd, zd)) < 1e-15
        np.testing.assert_allclose(np.cross(xd, yd), zd, atol=1e-15)
        assert g["cthd"] == pytest.approx(np.dot(n, zd), abs=1e-15)
        az = math.atan2(np.dot(n, yd), np.dot(n, xd))
        assert abs(math.remainder(g["phid"] - az, TWOPI)) < 1e-12         # full turns only: cos/sin(phi_d) are what enter
        sthd = math.sqrt(1 - g["cthd"] ** 2)
        assert sthd * math.cos(g["phid"]) == pytest.approx(np.dot(n, xd), abs=1e-14)
        assert sthd * math.sin(g["phid"]) == pytest.approx(np.dot(n, yd), abs=1e-14)


def test_antenna_patterns_from_the_detector_tensor(oracle):
    """The whole response chain geometry() -> antenna() against tensors written out from vectors, with no angle and no
    modulo anywhere: detector tensors D_I = (x_d x_d - y_d y_d)/2, D_II = (x_d y_d + y_d x_d)/2 (the second two-arm
    combination = the first rotated by 45 degrees) from the explicit rolling axes; polarisation tensors of BC Eqs. 5-6,
    e+ = p p - q q, ex = p q + q p with p = n x L / |n x L|, q = p x n; F = D : e.  Pins the sign and quadrant of phi_d
    and psi and every sign of BC 15-16 (a quarter-turn slip of phi_d flips all four)."""
    rng = np.random.default_rng(17)
    z = np.array([0.0, 0.0, 1.0])
    for _ in range(300):
        thS, thK = np.arccos(rng.uniform(-0.99, 0.99, 2))
        phS, phK, alpha, phibar = rng.uniform(0, TWOPI, 4)
        lam = rng.uniform(0.05, math.pi - 0.05)
        g = oracle.geometry(base_row(THS=thS, PHS=phS, THK=thK, PHK=phK, LAM=lam), alpha, phibar)
        F = oracle.antenna(g["cthd"], g["phid"], g["psi"])
        n, Sv = _vec(thS, phS), _vec(thK, phK)
        L = (Sv * math.cos(lam) + (z - Sv * math.cos(thK)) / math.sin(thK) * math.sin(lam) * math.cos(alpha)
             + np.cross(Sv, z) / math.sin(thK) * math.sin(lam) * math.sin(alpha))
        nxL = np.cross(n, L)
        if np.linalg.norm(nxL) < 1e-3:
            continue
        ph = nxL / np.linalg.norm(nxL)
        q = np.cross(ph, n)
        ep = np.outer(ph, ph) - np.outer(q, q)
        ex = np.outer(ph, q) + np.outer(q, ph)
        xd, yd, zd = _detector_axes(phibar)
        DI = 0.5 * (np.outer(xd, xd) - np.outer(yd, yd))
        DII = 0.5 * (np.outer(xd, yd) + np.outer(yd, xd))
        want = [np.sum(DI * ep), np.sum(DI * ex), np.sum(DII * ep), np.sum(DII * ex)]
        np.testing.assert_allclose(F, want, atol=5e-12)


# ------------------------------------------------------------------ antenna patterns (S5.8)
def test_antenna_identities(oracle):
    rng = np.random.default_rng(3)
    for _ in range(200):
        c, ph, ps = rng.uniform(-1, 1), rng.uniform(0, TWOPI), rng.uniform(0, TWOPI)
        F = oracle.antenna(c, ph, ps)
        h = 0.5 * (1 + c * c)
        assert F[0] ** 2 + F[1] ** 2 == pytest.approx(h * h * math.cos(2 * ph) ** 2 + c * c * math.sin(2 * ph) ** 2, abs=1e-14)
        assert F[2] ** 2 + F[3] ** 2 == pytest.approx(h * h * math.sin(2 * ph) ** 2 + c * c * math.cos(2 * ph) ** 2, abs=1e-14)
        assert np.sum(F ** 2) == pytest.approx(h * h + c * c, abs=1e-14)
        # channel II is channel I rotated by 45 degrees in phi_d
        F45 = oracle.antenna(c, ph - math.pi / 4, ps)
        np.testing.assert_allclose(F[2:], F45[:2], atol=1e-14)
        # psi -> psi + pi/4 swaps + and x
        Fp = oracle.antenna(c, ph, ps + math.pi / 4)
        np.testing.assert_allclose([Fp[0], Fp[1]], [-F[1], F[0]], atol=1e-14)


def test_antenna_sky_average_is_one_fifth(oracle):
    xs, ws = np.polynomial.legendre.leggauss(8)
    acc = np.zeros(4)
    m = 16
    for c, w in zip(xs, ws):
        for a in range(m):
            for b in range(m):
                F = oracle.antenna(c, TWOPI * a / m, TWOPI * b / m)
                acc += 0.5 * w * F ** 2 / (m * m)
    np.testing.assert_allclose(acc, 0.2, atol=1e-13)


def test_antenna_normal_incidence(oracle):
    """source at the detector zenith, psi = 0: F+ = cos 2 phi, Fx = sin 2 phi (textbook 90-degree
    interferometer), and channel II = same at 45 degrees"""
    F = oracle.antenna(1.0, 0.0, 0.0)
    np.testing.assert_allclose(F, [1.0, 0.0, 0.0, -1.0], atol=1e-15)


# ------------------------------------------------------------------ waveform (S5)
def test_circular_orbit_is_textbook_quadrupole(oracle):
    """e = 0: A+ = 2A(1+(L.n)^2) cos(2 Phi_tot + 2 gamma), Ax = -4A (L.n) sin(2 Phi_tot + 2 gamma),
    A = (2 pi nu M)^{2/3} mu / D; the phase, Doppler term, L^ and beta are rebuilt here by vector algebra"""
    p = base_row(E0=0.0, A=0.6, NU0=1.1e-3, THS=1.0, PHS=0.5, THK=0.7, PHK=2.0, LAM=0.9)
    N, dt, S = 1 << 14, 15.0, 256
    idx = np.array([0, 3, 1000, 5555, N - 1])
    hI, hII, st, Ap, Ax = oracle.waveform(p, N, dt, 6, S, idx=idx, amplitudes=True)
    assert st == 0
    y = oracle.orbit_at(p, N, dt, idx, S)
    z = np.array([0.0, 0.0, 1.0])
    n, Sv = _vec(1.0, 0.5), _vec(0.7, 2.0)
    for m, i in enumerate(idx):
        Phic, nu, gamc, e, alpc = y[:, m]
        assert e == 0.0
        alpha = TWOPI * alpc
        L = (Sv * math.cos(0.9) + (z - Sv * math.cos(0.7)) / math.sin(0.7) * math.sin(0.9) * math.cos(alpha)
             + np.cross(Sv, z) / math.sin(0.7) * math.sin(0.9) * math.sin(alpha))
        Ln = np.dot(L, n)
        rt = math.sqrt(1 - Ln * Ln)
        phat = (Sv - L * math.cos(0.9)) / math.sin(0.9)
        beta = math.atan2(np.dot(phat, (L * Ln - n) / rt), np.dot(phat, np.cross(L, n)) / rt)
        phibar = TWOPI * i * dt / YEAR
        Phitot = TWOPI * Phic + TWOPI * nu * AU * math.sin(1.0) * math.cos(phibar - 0.5)
        gam = TWOPI * gamc + beta
        A = (TWOPI * nu * 1e6 * MSUN) ** (2.0 / 3.0) * 10 * MSUN / GPC
        assert Ap[m] == pytest.approx(2 * A * (1 + Ln * Ln) * math.cos(2 * Phitot + 2 * gam), abs=2e-11 * A)
        assert Ax[m] == pytest.approx(-4 * A * Ln * math.sin(2 * Phitot + 2 * gam), abs=2e-11 * A)
        # and the projection onto the two channels
        g = oracle.geometry(p, alpha, phibar)
        F = oracle.antenna(g["cthd"], g["phid"], g["psi"])
        assert hI[m] == pytest.approx(math.sqrt(3) / 2 * (F[0] * Ap[m] + F[1] * Ax[m]), rel=1e-13, abs=1e-40)
        assert hII[m] == pytest.approx(math.sqrt(3) / 2 * (F[2] * Ap[m] + F[3] * Ax[m]), rel=1e-13, abs=1e-40)


def test_harmonic_sum_against_direct_python(oracle):
    """eccentric case: rebuild A+, Ax at a few samples from scipy Bessel functions and BC Eqs. 7-9"""
    p = base_row(E0=0.35, A=0.5, NU0=8e-4)
    N, dt, S, n_max = 1 << 13, 15.0, 256, 12
    idx = np.array([1, 777, 4096, N - 2])
    hI, hII, st, Ap, Ax = oracle.waveform(p, N, dt, n_max, S, idx=idx, amplitudes=True)
    y = oracle.orbit_at(p, N, dt, idx, S)
    for m, i in enumerate(idx):
        Phic, nu, gamc, e, alpc = y[:, m]
        phibar = TWOPI * i * dt / YEAR
        g = oracle.geometry(p, TWOPI * alpc, phibar)
        Phitot = TWOPI * (Phic + nu * AU * math.sin(p[W.P_THS]) * math.cos(phibar - p[W.P_PHS]))
        gam = TWOPI * gamc + g["beta"]
        A = (TWOPI * nu * 1e6 * MSUN) ** (2.0 / 3.0) * 10 * MSUN / GPC
        ap = ax = 0.0
        for n in range(1, n_max + 1):
            J = lambda k: scipy.special.jv(k, n * e)
            a_n = -n * A * (J(n - 2) - 2 * e * J(n - 1) + 2.0 / n * J(n) + 2 * e * J(n + 1) - J(n + 2)) * math.cos(n * Phitot)
            b_n = -n * A * math.sqrt(1 - e * e) * (J(n - 2) - 2 * J(n) + J(n + 2)) * math.sin(n * Phitot)
            c_n = 2 * A * J(n) * math.cos(n * Phitot)
            ap += -(1 + g["Ln"] ** 2) * (a_n * math.cos(2 * gam) - b_n * math.sin(2 * gam)) + (1 - g["Ln"] ** 2) * c_n
            ax += 2 * g["Ln"] * (b_n * math.cos(2 * gam) + a_n * math.sin(2 * gam))
        scale = A * n_max
        assert Ap[m] == pytest.approx(ap, abs=1e-10 * scale) and Ax[m] == pytest.approx(ax, abs=1e-10 * scale)


def test_doppler_term_bound_and_period(oracle):
    """the Doppler phase enters as nu R sin(thS) cos(phibar - phS) cycles: bounded by nu R sin(thS),
    absent at sin(thS) -> 0 (compare A+ phase with a source at the ecliptic pole direction changed)"""
    N, dt, S = 1 << 12, 15.0, 256
    p = base_row(E0=0.0, THS=1e-8)
    idx = np.arange(0, N, 97)
    _, _, _, Ap, Ax = oracle.waveform(p, N, dt, 3, S, idx=idx, amplitudes=True)
    y = oracle.orbit_at(p, N, dt, idx, S)
    # at thS = 1e-8 the Doppler term is < nu R 1e-8 ~ 5e-9 cycles: phase = 2 Phi + 2 gamma only
    for m, i in enumerate(idx):
        g = oracle.geometry(p, TWOPI * y[4][m], TWOPI * i * dt / YEAR)
        A = (TWOPI * y[1][m] * 1e6 * MSUN) ** (2.0 / 3.0) * 10 * MSUN / GPC
        ph = 2 * TWOPI * y[0][m] + 2 * (TWOPI * y[2][m] + g["beta"])
        assert Ap[m] == pytest.approx(2 * A * (1 + g["Ln"] ** 2) * math.cos(ph), abs=1e-6 * A)


def test_waveform_scalings_and_gr_limit(oracle):
    """h ~ 1/(Xi D_L) exactly (Eq. 4-6); Xi0=1 or n=0 or delta_T=0 are the GR waveform"""
    N, dt, n_max = 1 << 12, 15.0, 6
    p = base_row()
    hI, hII, st = oracle.waveform(p, N, dt, n_max)
    assert st == 0 and np.max(np.abs(hI)) > 0
    hI2, hII2, _ = oracle.waveform(base_row(DL=2.0), N, dt, n_max)
    np.testing.assert_allclose(hI2 * 2.0, hI, rtol=0, atol=1e-14 * np.max(np.abs(hI)))
    np.testing.assert_allclose(hII2 * 2.0, hII, rtol=0, atol=1e-14 * np.max(np.abs(hII)))
    for kw in (dict(XI0=1.0, NXI=2.0), dict(XI0=0.8, NXI=0.0)):
        a, b, _ = oracle.waveform(base_row(**kw), N, dt, n_max)
        np.testing.assert_array_equal(a, hI)
        np.testing.assert_array_equal(b, hII)
    pm = base_row(XI0=0.8, NXI=2.0)
    Xi = oracle.walker_scalars(pm)["Xi"]
    a, b, _ = oracle.waveform(pm, N, dt, n_max)
    np.testing.assert_allclose(a * Xi, hI, rtol=0, atol=1e-14 * np.max(np.abs(hI)))
    # typical strain magnitude of a 10+1e6 Msun EMRI at 1 Gpc: 1e-23..1e-21
    assert 1e-24 < np.max(np.abs(hI)) < 1e-20


def test_waveform_phase_invariances(oracle):
    """only frac of the phases matters: Phi0 + 2 pi, gamma~0 + pi (2 gamma enters), alpha0 + 2 pi"""
    N, dt, n_max = 1 << 11, 15.0, 5
    p = base_row()
    hI, hII, _ = oracle.waveform(p, N, dt, n_max)
    sc = np.max(np.abs(hI))
    for kw in (dict(PHI0=p[W.P_PHI0] + TWOPI), dict(GAM0=p[W.P_GAM0] + math.pi), dict(ALP0=p[W.P_ALP0] + TWOPI),
               dict(PHS=p[W.P_PHS] + TWOPI), dict(PHK=p[W.P_PHK] + TWOPI)):
        a, b, _ = oracle.waveform(base_row(**kw), N, dt, n_max)
        assert np.max(np.abs(a - hI)) < 1e-11 * sc and np.max(np.abs(b - hII)) < 1e-11 * sc


def test_gw_speed_delay_is_an_arrival_delay(oracle):
    """R9: with dT = m dt the source quantities at sample i are those of sample i-m at dT = 0; only the
    detector angles (3e-6 rad apart) differ => h(i; dT) ~ h(i-m; 0) to ~1e-5"""
    N, dt, n_max, m = 1 << 12, 15.0, 6, 3
    tlb = oracle.cosmology(1.0)[1]
    p_del = base_row(DELT=-(m * dt) / tlb)     # dT = -delta_T t_lb = +m dt  (slower GW: arrives later)
    assert oracle.walker_scalars(p_del)["dT"] == pytest.approx(m * dt, rel=1e-13)
    a, b, st = oracle.waveform(p_del, N, dt, n_max)
    hI, hII, _ = oracle.waveform(base_row(), N, dt, n_max)
    sc = np.max(np.abs(hI))
    assert st == 0
    assert np.max(np.abs(a[m:] - hI[:-m])) < 3e-5 * sc and np.max(np.abs(b[m:] - hII[:-m])) < 3e-5 * sc
    assert np.max(np.abs(a[m:] - hI[m:])) > 1e-2 * sc      # and it is not a no-op
    # |dT| > Delta => status bit 4, zero waveform
    a, b, st = oracle.waveform(base_row(DELT=5e-14), N, dt, n_max)
    assert st & 4 and not a.any() and not b.any()


def test_double_and_long_double_builds_agree(oracle, oracle_ld):
    """conditioning: the fp64 oracle's own rounding error is far below the 1e-9 parity tolerance"""
    cfg = W.CONFIGS[2]
    P = W.draw_params(cfg, K=4)
    N = cfg.N
    idx = np.concatenate([np.arange(0, 64), np.arange(N - 64, N), np.random.default_rng(0).integers(0, N, 200)])
    for p in P:
        o1, o2 = oracle.orbit(p, N, cfg.dt, 256), oracle_ld.orbit(p, N, cfg.dt, 256)
        for q in (0, 2, 4):                                                       # phases, cycles, after one year
            assert np.max(np.abs(circ_diff(o1["val"][q], o2["val"][q]))) < 1e-11
        assert np.max(np.abs(o1["val"][1] / o2["val"][1] - 1)) < 1e-15
        a1, b1, _ = oracle.waveform(p, N, cfg.dt, cfg.n_max, idx=idx)
        a2, b2, _ = oracle_ld.waveform(p, N, cfg.dt, cfg.n_max, idx=idx)
        assert np.max(np.abs(a1 - a2)) < 1e-10 * np.max(np.abs(a2)) and np.max(np.abs(b1 - b2)) < 1e-10 * np.max(np.abs(b2))


# ------------------------------------------------------------------ transform (S6)
def test_fft_against_naive_dft_and_numpy(oracle):
    rng = np.random.default_rng(2)
    for N in (1, 2, 4, 8, 64, 256):
        h = rng.standard_normal(N)
        H = oracle.rfft(h)
        np.testing.assert_allclose(H, oracle.dft_naive(h), atol=1e-12)
        np.testing.assert_allclose(H, np.fft.rfft(h), atol=1e-12)
    # the naive DFT itself against its definition written out here
    h = rng.standard_normal(12)
    ref = np.array([sum(h[i] * np.exp(-2j * np.pi * i * m / 12) for i in range(12)) for m in range(7)])
    np.testing.assert_allclose(oracle.dft_naive(h), ref, atol=1e-13)
    h = rng.standard_normal(1 << 16)
    np.testing.assert_allclose(oracle.rfft(h), np.fft.rfft(h), atol=1e-9, rtol=1e-11)
    with pytest.raises(ValueError):
        oracle.rfft(np.zeros(12))


def test_fft_parseval_and_delta(oracle):
    rng = np.random.default_rng(4)
    N = 1 << 12
    h = rng.standard_normal(N)
    H = oracle.rfft(h)
    rhs = (abs(H[0]) ** 2 + 2 * np.sum(np.abs(H[1:N // 2]) ** 2) + abs(H[N // 2]) ** 2) / N
    assert np.sum(h * h) == pytest.approx(rhs, rel=1e-13)
    d = np.zeros(N)
    d[3] = 1.0
    np.testing.assert_allclose(oracle.rfft(d), np.exp(-2j * np.pi * 3 * np.arange(N // 2 + 1) / N), atol=1e-14)


# ------------------------------------------------------------------ likelihood (S7)
def _small_problem(oracle, K=3, N=1 << 12, n_max=5):
    cfg = W.scaled(W.CONFIGS[1], K=K, N=N, n_max=n_max)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    h, st = oracle.waveform_batch(P, N, cfg.dt, n_max)
    H = np.stack([[oracle.rfft(h[k, c]) for c in range(2)] for k in range(K)])
    return cfg, P, psd, h, H


def test_loglike_zero_at_injection_and_quadratic_identity(oracle):
    cfg, P, psd, h, H = _small_problem(oracle)
    N, dt = cfg.N, cfg.dt
    assert oracle.loglike(H[0], H[0], psd, N, dt) == 0.0
    logL, st = oracle.loglike_batch(P, N, dt, cfg.n_max, H[0], psd)
    assert logL[0] == 0.0 and np.all(logL[1:] < 0) and not st.any()
    for k in (1, 2):
        dd, hh, dh = (oracle.inner(H[0], H[0], psd, N, dt), oracle.inner(H[k], H[k], psd, N, dt),
                      oracle.inner(H[0], H[k], psd, N, dt))
        assert logL[k] == pytest.approx(-0.5 * (dd - 2 * dh + hh), rel=1e-11)
        assert logL[k] == pytest.approx(oracle.loglike(H[k], H[0], psd, N, dt), rel=1e-15)


def test_loglike_definition_written_out(oracle):
    """-(1/2) <d-h|d-h>, <a|b> = 4 Re sum a~* b~ / S_n df, a~ = dt A (Eq. 8 / reading R12), via numpy"""
    cfg, P, psd, h, H = _small_problem(oracle, K=2)
    N, dt = cfg.N, cfg.dt
    ok = np.isfinite(psd) & (psd > 0)
    r = (np.fft.rfft(h[0], axis=-1) - np.fft.rfft(h[1], axis=-1)) * dt
    df = 1.0 / (N * dt)
    want = -0.5 * 4.0 * np.sum(np.abs(r[:, ok]) ** 2 / psd[ok]) * df
    assert oracle.loglike(H[1], H[0], psd, N, dt) == pytest.approx(want, rel=1e-10)
    assert not ok[0] and not ok[-1]


def test_snr_scales_inversely_with_distance(oracle):
    N, dt, n_max = 1 << 12, 15.0, 5
    psd = W.lisa_psd_barack_cutler(N, dt)
    rho2 = []
    for DL in (1.0, 2.0, 4.0):
        hI, hII, _ = oracle.waveform(base_row(DL=DL), N, dt, n_max)
        H = np.stack([oracle.rfft(hI), oracle.rfft(hII)])
        rho2.append(oracle.inner(H, H, psd, N, dt))
    assert rho2[0] / rho2[1] == pytest.approx(4.0, rel=1e-12) and rho2[0] / rho2[2] == pytest.approx(16.0, rel=1e-12)


def test_loglike_noise_expectation(oracle):
    """d = h + n with the recipe's noise: E[logL(theta*)] = -(number of unmasked bins) x 2 channels x ... = -(N-2);
    variance N-2  => |logL + (N-2)| < 6 sqrt(N)"""
    N, dt = 1 << 14, 15.0
    psd = W.lisa_psd_barack_cutler(N, dt)
    noise = W.noise_fft(N, dt, psd, seed=99)
    zero = np.zeros_like(noise)
    logL = oracle.loglike(zero, noise, psd, N, dt)
    assert abs(logL + (N - 2)) < 6 * math.sqrt(N)
    assert noise[0, 0] == 0 and noise[1, -1] == 0


def test_loglike_masks_bad_psd_bins(oracle):
    N, dt = 64, 15.0
    rng = np.random.default_rng(1)
    H = rng.standard_normal((2, 33)) + 1j * rng.standard_normal((2, 33))
    D = rng.standard_normal((2, 33)) + 1j * rng.standard_normal((2, 33))
    psd = np.full(33, 2.0)
    base = oracle.loglike(H, D, psd, N, dt)
    for bad in (0.0, -1.0, np.inf, np.nan):
        psd2 = psd.copy()
        psd2[5] = bad
        want = base + (2 * dt / N) * np.sum(np.abs(D[:, 5] - H[:, 5]) ** 2) / 2.0
        assert oracle.loglike(H, D, psd2, N, dt) == pytest.approx(want, rel=1e-13)


def test_invalid_walker_gets_minus_infinity(oracle):
    cfg, P, psd, h, H = _small_problem(oracle, K=2)
    P2 = P.copy()
    P2[1, W.P_E0] = 1.2
    logL, st = oracle.loglike_batch(P2, cfg.N, cfg.dt, cfg.n_max, H[0], psd)
    assert st[1] == 1 and logL[1] == -np.inf and logL[0] == 0.0


# ------------------------------------------------------------------ input recipe
def test_configs_have_no_plunge_and_sane_parameters(oracle):
    for cfg in W.CONFIGS:
        P = W.draw_params(cfg, K=min(cfg.K, 48))
        assert P.shape[1] == W.NPAR and np.all(np.isfinite(P))
        for p in P:
            assert oracle.orbit(p, cfg.N, cfg.dt, 256)["status"] == 0
            assert p[W.P_NU0] < oracle.nu_lso(p[W.P_M], p[W.P_E0])
        np.testing.assert_array_equal(P, W.draw_params(cfg, K=min(cfg.K, 48)))     # seeded


def test_psd_models_are_positive_and_masked_at_ends():
    for fn in (W.lisa_psd_barack_cutler, W.lisa_psd_robson):
        s = fn(1 << 12, 15.0)
        assert np.isinf(s[0]) and np.isinf(s[-1]) and np.all(s[1:-1] > 0) and np.all(np.isfinite(s[1:-1]))
        # LISA bucket near a few mHz
        f = W.freqs(1 << 12, 15.0)
        assert 1e-3 < f[np.argmin(s[1:-1]) + 1] < 2e-2


# ----------------------------------------------------------------------------- frequency-dependent propagation (Eq. 7)
def _fdep_case(seed=3, N=256, dt=15.0):
    rng = np.random.default_rng(seed)
    Nf = N // 2 + 1
    H = rng.normal(size=(2, Nf)) + 1j * rng.normal(size=(2, Nf))
    D = rng.normal(size=(2, Nf)) + 1j * rng.normal(size=(2, Nf))
    psd = rng.uniform(0.5, 2.0, Nf)
    psd[0] = psd[-1] = np.inf
    return H, D, psd, N, dt


def test_fdep_reduces_to_eq8_when_the_series_vanish(oracle):
    H, D, psd, N, dt = _fdep_case()
    assert oracle.loglike_fdep(H, D, psd, N, dt, np.zeros(6)) == oracle.loglike(H, D, psd, N, dt)


def test_fdep_factor_restated_with_numpy(oracle):
    """G = exp(-Dm(f)) exp(-2 pi i f tau(f)) applied to H, then Eq. 8"""
    H, D, psd, N, dt = _fdep_case(4)
    fc, fstar = np.array([0.3, -0.2, 0.05, 40.0, -15.0, 6.0]), 2e-3
    f = np.arange(N // 2 + 1) / (N * dt)
    x = f / fstar
    G = np.exp(-(fc[0] * x + fc[1] * x ** 2 + fc[2] * x ** 3)) * np.exp(-2j * np.pi * f * (fc[3] * x + fc[4] * x ** 2 + fc[5] * x ** 3))
    ok = np.isfinite(psd)
    want = -(2 * dt / N) * np.sum(np.abs(D - G * H)[:, ok] ** 2 / psd[ok])
    assert abs(oracle.loglike_fdep(H, D, psd, N, dt, fc, fstar) - want) <= 1e-12 * abs(want)
    # it equals the plain likelihood of the pre-multiplied spectrum
    assert abs(oracle.loglike(G * H, D, psd, N, dt) - want) <= 1e-12 * abs(want)


def test_fdep_pure_delay_leaves_signal_power_unchanged_and_damping_scales_it(oracle):
    H, D, psd, N, dt = _fdep_case(5)
    Z = np.zeros_like(D)
    base = oracle.loglike(H, Z, psd, N, dt)
    # a speed-only modification is a pure phase: <h|h> is invariant
    assert abs(oracle.loglike_fdep(H, Z, psd, N, dt, [0, 0, 0, 30.0, 5.0, -2.0]) - base) <= 1e-13 * abs(base)
    # a single unmasked bin: friction a1 scales the power by exp(-2 a1 f/f*)
    m0, fstar = 37, 1e-3
    psd1 = np.full_like(psd, np.inf)
    psd1[m0] = 1.3
    f0 = m0 / (N * dt)
    b1 = oracle.loglike(H, Z, psd1, N, dt)
    got = oracle.loglike_fdep(H, Z, psd1, N, dt, [0.7, 0, 0, 0, 0, 0], fstar)
    assert abs(got - b1 * np.exp(-2 * 0.7 * f0 / fstar)) <= 1e-13 * abs(b1)
    # data that carries exactly the delayed, damped signal gives logL = 0
    fc = np.array([0.1, 0.0, 0.0, 12.0, 0.0, 0.0])
    f = np.arange(N // 2 + 1) / (N * dt)
    G = np.exp(-fc[0] * f / fstar) * np.exp(-2j * np.pi * f * fc[3] * f / fstar)
    assert abs(oracle.loglike_fdep(H, G * H, psd, N, dt, fc, fstar)) <= 1e-25


def test_fdep_linear_in_f_delay_is_a_quadratic_phase_ie_a_dispersion(oracle):
    """tau(f) = b1 f/f*: the phase -2 pi b1 f^2/f* has group delay d(phase)/d(2 pi f) = -2 b1 f/f*, twice tau:
    checked through the factor the oracle applies, extracted with a one-bin probe"""
    N, dt, fstar, b1 = 128, 10.0, 5e-3, 3.0
    Nf = N // 2 + 1
    psd = np.ones(Nf)
    for m0 in (5, 20, 41):
        H = np.zeros((2, Nf), dtype=complex)
        H[0, m0] = 1.0
        f0 = m0 / (N * dt)
        # logL(D = c) = -(2dt/N) |c - G|^2 is maximal (zero) at c = G: scan the phase of c
        ph = -2 * np.pi * f0 * b1 * f0 / fstar
        Dm = np.zeros_like(H)
        Dm[0, m0] = np.exp(1j * ph)
        assert abs(oracle.loglike_fdep(H, Dm, psd, N, dt, [0, 0, 0, b1, 0, 0], fstar)) <= 1e-28
        Dm[0, m0] = np.exp(1j * (ph + 0.01))
        assert oracle.loglike_fdep(H, Dm, psd, N, dt, [0, 0, 0, b1, 0, 0], fstar) < -1e-6


# ----------------------------------------------------------------------------- the paper's IC convention: anchored at the LSO
@pytest.fixture()
def lso():
    """an oracle instance of its own, anchored at the LSO (the anchor is an explicit argument of every library call and a
    property of the instance: nothing here can leak into the session-wide forward-anchored `oracle`)"""
    from oracle.oracle import Oracle
    return Oracle(anchor=True)


def _lso_params(e_lso=0.3):
    p = W.draw_params(W.CONFIGS[1], K=1)[0].copy()
    p[W.P_E0] = e_lso
    return p


def test_lso_anchor_sits_on_the_plunge_frequency(lso):
    """nu_LSO = c^3/(2 pi G M) ((1-e^2)/(6+2e))^{3/2} at the last coarse node, integrated backwards"""
    p = _lso_params(0.3)
    N, dt, S = 1 << 16, 15.0, 256
    orb = lso.orbit(p, N, dt, S)
    assert orb["status"] == 0 and orb["jpl"] == orb["Nn"]
    x = ((1 - 0.09) / 6.6) ** 1.5 / (2 * np.pi * p[W.P_M] * 4.925490947e-6)
    assert orb["val"][1][-2] == pytest.approx(x, rel=1e-15)
    assert orb["val"][3][-2] == 0.3
    # going back in time the orbit is wider and more eccentric, monotonically
    assert np.all(np.diff(orb["val"][1]) > 0) and np.all(np.diff(orb["val"][3]) < 0)
    for q, col in ((0, W.P_PHI0), (2, W.P_GAM0), (4, W.P_ALP0)):
        assert abs(circ_diff(orb["val"][q][-2], (p[col] / (2 * np.pi)) % 1.0)) < 1e-15


def test_lso_increments_and_slopes_are_consistent(lso):
    p = _lso_params(0.2)
    orb = lso.orbit(p, 1 << 16, 15.0, 256)
    v, inc, sl = orb["val"], orb["inc"], orb["slope"]
    for q in (0, 2, 4):
        assert np.max(np.abs(circ_diff(v[q][:-1] + inc[q][:-1], v[q][1:]))) < 1e-14
    for q in (1, 3):
        np.testing.assert_allclose(v[q][:-1] + inc[q][:-1], v[q][1:], rtol=1e-15)
    for jj in (0, 1, 17, orb["Nn"] - 2, orb["Nn"] - 1):
        np.testing.assert_array_equal(sl[:, jj], lso.rhs(p, v[:, jj]))


def test_lso_backward_orbit_against_dop853_and_forward_rerun(lso):
    p = _lso_params(0.3)
    N, dt, S = 1 << 18, 15.0, 256
    orb = lso.orbit(p, N, dt, S)
    assert orb["status"] == 0
    yA = [orb["val"][q][-2] for q in range(5)]
    T = (orb["Nn"] - 3) * S * dt                     # from node Nc back to node 0
    sol = scipy.integrate.solve_ivp(lambda t, y: lso.rhs(p, y), (0.0, -T), yA, method="DOP853", rtol=1e-13,
                                    atol=[1e-9, 1e-19, 1e-9, 1e-16, 1e-9])
    y0 = sol.y[:, -1]
    assert orb["val"][1][1] == pytest.approx(y0[1], rel=5e-11)
    assert orb["val"][3][1] == pytest.approx(y0[3], rel=5e-10)
    for q in (0, 2, 4):
        assert abs(circ_diff(orb["val"][q][1], y0[q] % 1.0)) < 5e-7       # the last hours before plunge are stiff for RK4
    # the forward scheme started from node 0 of the backward orbit returns to the anchor (both are O(Delta^4) accurate)
    lso.set_anchor(False)
    q0 = p.copy()
    q0[W.P_NU0], q0[W.P_E0] = orb["val"][1][1], orb["val"][3][1]
    q0[W.P_PHI0], q0[W.P_GAM0], q0[W.P_ALP0] = (2 * np.pi * orb["val"][k][1] for k in (0, 2, 4))
    fwd = lso.orbit(q0, N - S, dt, S)                # stops short of the LSO node, so nothing plunges
    assert fwd["status"] == 0
    assert fwd["val"][1][-3] == pytest.approx(orb["val"][1][-4], rel=1e-8)
    assert fwd["val"][3][-3] == pytest.approx(orb["val"][3][-4], rel=1e-8)


def test_lso_waveform_ends_at_plunge_and_is_finite(lso):
    p = _lso_params(0.3)
    N, dt = 1 << 14, 15.0
    hI, hII, st = lso.waveform(p, N, dt, 10)
    assert st == 0 and np.all(np.isfinite(hI)) and np.abs(hI[-200:]).max() > 0
    # the window ends AT plunge: every sample is live (no truncation flag), unlike a forward orbit that crosses the LSO
    assert hI[-1] != 0.0 and hII[-1] != 0.0
    lso.set_anchor(False)
    q = p.copy()
    q[W.P_NU0] = 0.999 * lso.nu_lso(p[W.P_M], p[W.P_E0])
    _, _, st_fwd = lso.waveform(q, N, dt, 10)
    assert st_fwd == 2


# ----------------------------------------------------------------------------- the paper's Figure 1 set-up (inputs only)
FIG1 = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_fig1_parameters.txt")


def test_paper_fig1_grid_last_hour_before_plunge(lso):
    """nine waveforms over the last hour before the LSO.  What the text fixes: the orbit ends on nu_LSO
    (PAPER.md:120), the waveforms are finite and live to the last sample, and for e_LSO = 0 the signal is the n = 2
    quadrupole at 2 nu_LSO = 2 / (2 pi M 6^{3/2}) = 4.397 mHz for M = 1e6 Msun."""
    P = W.paper_fig1_params(FIG1)
    assert P.shape == (9, 17)
    dt, N, S = 15.0, 256, 256                        # 64 min: one coarse interval ending at plunge
    for p in P:
        hI, hII, st = lso.waveform(p, N, dt, 20, S=S)
        assert st == 0 and np.all(np.isfinite(hI)) and np.all(np.isfinite(hII))
        assert hI[-1] != 0.0 and 1e-24 < np.max(np.abs(hI)) < 1e-20           # strain of a 10 Msun body at 1 Gpc
        orb = lso.orbit(p, N, dt, S)
        assert orb["val"][1][-2] == pytest.approx(lso.nu_lso(p[W.P_M], p[W.P_E0]), rel=1e-15)
    # circular cases: only n = 2 survives, h ~ cos(2 Phi + 2 gamma): the GW frequency is twice the AZIMUTHAL frequency
    # nu + gamma~'/2pi (in the AK model nu is the radial frequency; at the LSO the periapsis advance gamma~' is as large as
    # nu itself), here from the rates at the two nodes bracketing the hour; count the zero crossings
    f_orb = 1.0 / (2 * np.pi * 1e6 * 4.925490947e-6 * 6 ** 1.5)
    assert f_orb == pytest.approx(2.1985e-3, rel=1e-3)             # nu_LSO(e = 0)
    for p in P[[0, 3, 6]]:
        hI, _, _ = lso.waveform(p, N, dt, 20, S=S)
        orb = lso.orbit(p, N, dt, S)
        assert orb["val"][1][-2] == pytest.approx(f_orb, rel=1e-12)
        f_az = 0.5 * ((orb["slope"][0][1] + orb["slope"][2][1]) + (orb["slope"][0][-2] + orb["slope"][2][-2]))
        assert 1.5 * f_orb < f_az < 2.5 * f_orb
        crossings = np.sum(np.signbit(hI[1:]) != np.signbit(hI[:-1]))
        # (with spin the precession of the orbital plane, alpha' ~ 0.1 nu at a = 0.8, shifts the observed phase by a few per cent)
        assert crossings == pytest.approx(2 * (2 * f_az) * N * dt, rel=0.10)


# ----------------------------------------------------------------------------- S3': adaptive embedded pair with dense output (f-3, D14)
DP_ATOL = np.array([1e-9, 1e-18, 1e-9, 1e-14, 1e-9])


def _cycles_state(p):
    return np.array([(p[W.P_PHI0] / TWOPI) % 1.0, p[W.P_NU0], (p[W.P_GAM0] / TWOPI) % 1.0, p[W.P_E0], (p[W.P_ALP0] / TWOPI) % 1.0])


def _dense(r, tq):
    """the oracle's dense output, unwrapped (turns + wrapped value + offset), at times tq"""
    idx = np.clip(np.searchsorted(np.abs(r["t"]), np.abs(tq), side="right") - 1, 0, len(r["t"]) - 1)
    th = (tq - r["t"][idx]) / r["h"][idx]
    Y = r["y"][idx] + sum(r["Q"][idx][:, :, j] * th[:, None] ** (j + 1) for j in range(4))
    for a, q in enumerate((0, 2, 4)):
        Y[:, q] += r["turns"][idx, a]
    return Y


@pytest.mark.parametrize("T,rtol", [(2 ** 16 * 15.0, 1e-9), (2 ** 20 * 15.0, 1e-12), (-50 * 3840.0, 1e-11)])
def test_adaptive_pair_takes_scipy_rk45_steps_and_dense_output(oracle, T, rtol):
    """the paper integrates with SciPy's solve_ivp.  The oracle's Dormand-Prince 5(4) + step controller +
    continuous extension against solve_ivp(method="RK45") on the same right-hand side (in cycles): the same number of
    accepted steps at the same times, the same dense output -- forward over 11 days and half a year, and backwards.
    (A wrong tableau entry, controller constant, exponent, first-step rule or dense-output coefficient fails this.)"""
    P = W.draw_params(W.CONFIGS[1], K=3)
    for k in range(3):
        p = P[k]
        r = oracle.dp5_steps(p, T, rtol, DP_ATOL)
        sol = scipy.integrate.solve_ivp(lambda t, y: oracle.rhs(p, y), (0.0, T), _cycles_state(p), method="RK45", rtol=rtol,
                                        atol=DP_ATOL, dense_output=True)
        assert r["stop"] == 0 and r["t_reached"] == T
        np.testing.assert_allclose(r["t"][:4], sol.t[:4], rtol=1e-12, atol=0)          # the first-step rule, exactly
        tq = np.sort(np.random.default_rng(k).uniform(min(0.0, T), max(0.0, T), 300))
        Y, S = _dense(r, tq), sol.sol(tq).T
        if rtol >= 1e-9 or T < 0:
            # the error estimate is well above rounding: the same steps.  (SciPy carries the angles unwrapped, so its
            # estimate has 1e3 cycles x 1e-16 of rounding in it: equal to ~1e-6, not bit for bit.)
            assert len(r["t"]) == len(sol.t) - 1
            np.testing.assert_allclose(r["t"], sol.t[:-1], rtol=1e-5, atol=1e-9)
            for q in range(5):
                assert np.max(np.abs(Y[:, q] - S[:, q])) <= 2e-15 * max(1.0, np.max(np.abs(S[:, q]))) + 1e-24
        else:
            # near rounding the estimate is partly noise (|Phi| ~ 1e4 cycles in SciPy's state): the step sizes agree to a
            # per cent, the count to a step or two, and the two solutions to the accuracy the tolerance buys
            assert abs(len(r["t"]) - (len(sol.t) - 1)) <= 2
            m = min(len(r["t"]), len(sol.t) - 1)
            np.testing.assert_allclose(r["t"][:m], sol.t[:m], rtol=2e-2, atol=1e-9)
            for q in range(5):
                assert np.max(np.abs(Y[:, q] - S[:, q])) <= 100 * rtol * max(1.0, np.max(np.abs(S[:, q])))


def test_forced_error_norms_are_scipys_and_the_free_run_obeys_the_controller(oracle):
    """dp5_forced_errors (the validity half of the teacher-forced protocol, D14) returns, for a prescribed step
    sequence, the norm the controller would have judged each step by.  Pins: (1) SciPy's own RK45 machinery (`rk_step` and
    the rms of K^T E h / scale, the code path of solve_ivp) gives the same number for arbitrary -- not controller-chosen --
    step sizes, good steps and bad ones alike; (2) the oracle's free run satisfies its own rule exactly: every accepted
    norm is below 1 and the next step is h min(10, 0.9 norm^-1/5)."""
    from scipy.integrate._ivp.rk import RK45, rk_step
    P = W.draw_params(W.CONFIGS[1], K=2)
    for k in range(2):
        p = P[k]
        fun = lambda t, y: oracle.rhs(p, y)                                     # noqa: E731
        for rtol, sign in ((1e-8, 1.0), (1e-11, -1.0)):
            atol = DP_ATOL * (rtol / 1e-9)
            # arbitrary multiples of the largest step the controller itself takes, so that the norms straddle 1
            h_star = np.max(np.abs(oracle.dp5_steps(p, sign * 2 ** 20 * 15.0, rtol, atol)["h"][:-1]))
            hs = [sign * c * h_star for c in (0.3, 1.5, 0.6, 1.0)]
            got = oracle.dp5_forced_errors(p, rtol, atol, hs)
            t, y = 0.0, _cycles_state(p)
            f = fun(t, y)
            want = []
            Kbuf = np.empty((7, 5))
            for h in hs:
                y_new, f_new = rk_step(fun, t, y, f, h, RK45.A, RK45.B, RK45.C, Kbuf)
                scale = atol + np.maximum(np.abs(y), np.abs(y_new)) * rtol
                want.append(np.linalg.norm(np.dot(Kbuf.T, RK45.E) * h / scale) / 5 ** 0.5)
                t, y, f = t + h, y_new, f_new
            assert len(got) == len(hs)
            np.testing.assert_allclose(got, want, rtol=1e-6, atol=1e-8)         # (SciPy's state is unwrapped: rounding noise)
            assert max(want) > 1.0 > min(want)                                  # both verdicts occur in the sample
        for rtol in (1e-8, 1e-11):
            atol = DP_ATOL * (rtol / 1e-9)
            r = oracle.dp5_steps(p, 2 ** 18 * 15.0, rtol, atol)
            err = oracle.dp5_forced_errors(p, rtol, atol, r["h"])
            assert len(err) == len(r["h"]) and np.all(err < 1.0)
            # (a step after a rejection is smaller than the rule allows, and the last one is cut to the bound)
            ratio, fac = r["h"][1:-1] / r["h"][:-2], np.minimum(10.0, 0.9 * err[:-2] ** -0.2)
            assert np.all(ratio <= fac * (1 + 1e-12)) and np.mean(np.abs(ratio / fac - 1) < 1e-12) > 0.9


def test_adaptive_orbit_nodes_are_consistent_and_converge_to_the_rk4_orbit(oracle):
    """the node table sampled from the dense output: increments and values agree, slopes are the right-hand side at the
    node, and with a tight tolerance it is the same orbit as the fixed-step scheme (both converge to the ODE solution)"""
    from oracle.oracle import Oracle
    p = W.draw_params(W.CONFIGS[1], K=1)[0]
    N, dt, S = 1 << 18, 15.0, 256
    ada = Oracle(adaptive=(1e-13, DP_ATOL * 1e-4))
    a, f = ada.orbit(p, N, dt, S), oracle.orbit(p, N, dt, S)
    assert a["status"] == 0 and a["Nn"] == f["Nn"] and a["jpl"] == a["Nn"]
    v, inc, sl = a["val"], a["inc"], a["slope"]
    for q in (0, 2, 4):
        assert np.max(np.abs(circ_diff(v[q][:-1] + inc[q][:-1], v[q][1:]))) < 2e-14
        assert np.max(np.abs(circ_diff(v[q], f["val"][q]))) < 1e-9            # 5th-order pair at 1e-13 against RK4 at 3840 s
        np.testing.assert_allclose(inc[q][:-1], f["inc"][q][:-1], rtol=1e-10, atol=1e-12)
    for q in (1, 3):
        np.testing.assert_allclose(v[q][:-1] + inc[q][:-1], v[q][1:], rtol=1e-15)
        np.testing.assert_allclose(v[q], f["val"][q], rtol=1e-12)
    for jj in (0, 1, 500, a["Nn"] - 1):
        np.testing.assert_array_equal(sl[:, jj], oracle.rhs(p, v[:, jj]))
    # the initial state sits on node 0 exactly
    np.testing.assert_array_equal(v[:, 1], _cycles_state(p))
    # and the waveform through the same Hermite + harmonic sum agrees at the level the two orbits do
    idx = np.arange(0, N, 997)
    hA = ada.waveform(p, N, dt, 10, idx=idx)[0]
    hF = oracle.waveform(p, N, dt, 10, idx=idx)[0]
    assert np.max(np.abs(hA - hF)) < 1e-6 * np.max(np.abs(hF))


def test_adaptive_orbit_plunge_and_lso_anchor(oracle):
    from oracle.oracle import Oracle
    p = W.draw_params(W.CONFIGS[1], K=1)[0].copy()
    N, dt, S = 1 << 14, 15.0, 256
    ada = Oracle(adaptive=(1e-12, DP_ATOL * 1e-3))
    # forward convention, plunging inside the window: same truncation node as the fixed-step scheme (or its neighbour)
    p[W.P_NU0] = 0.9995 * oracle.nu_lso(p[W.P_M], p[W.P_E0])
    a, f = ada.orbit(p, N, dt, S), oracle.orbit(p, N, dt, S)
    assert a["status"] == 2 and f["status"] == 2 and abs(a["jpl"] - f["jpl"]) <= 1 and 0 < a["jpl"] < a["Nn"] - 2
    jj = a["jpl"] + 1                                      # column of node j_pl
    np.testing.assert_array_equal(a["val"][:, jj], a["val"][:, jj - 1])      # copies of node j_pl - 1, zero increments
    assert not a["inc"][:, jj - 1:].any()
    # the LSO convention: anchored on nu_LSO at the last node, integrated backwards; agrees with the fixed-step LSO orbit
    p[W.P_E0] = 0.3
    adaL, fixL = Oracle(anchor=True, adaptive=(1e-13, DP_ATOL * 1e-4)), Oracle(anchor=True)
    a, f = adaL.orbit(p, N, dt, S), fixL.orbit(p, N, dt, S)
    assert a["status"] == 0 and f["status"] == 0
    assert a["val"][1][-2] == f["val"][1][-2] == pytest.approx(oracle.nu_lso(p[W.P_M], 0.3), rel=1e-15)
    np.testing.assert_allclose(a["val"][1], f["val"][1], rtol=1e-9)
    np.testing.assert_allclose(a["val"][3], f["val"][3], rtol=1e-9)
    assert np.max(np.abs(circ_diff(a["val"][0], f["val"][0]))) < 1e-6        # the last hours before plunge are stiff for RK4
    # a bad parameter row stays bad
    p[W.P_MU] = -1.0
    assert adaL.orbit(p, N, dt, S)["status"] == 1


def test_adaptive_forced_steps_reproduce_the_free_run(oracle):
    """teacher-forced mode: given its own accepted step sizes the integrator reproduces its own orbit bit for bit, and a
    different (coarser) step sequence gives a different but close orbit -- the step sizes are really taken from the list"""
    from oracle.oracle import Oracle
    p = W.draw_params(W.CONFIGS[1], K=1)[0]
    N, dt, S = 1 << 16, 15.0, 256
    rtol, atol = 1e-10, DP_ATOL * 0.1
    free = Oracle(adaptive=(rtol, atol))
    a = free.orbit(p, N, dt, S)
    Nc = N // S
    fw = free.dp5_steps(p, (Nc + 1) * S * dt, rtol, atol, stop_at_plunge=True)
    bw = free.dp5_steps(p, -S * dt, rtol, atol)
    forced = Oracle()
    forced.set_adaptive((rtol, atol), forced_fwd=fw["h"], forced_bwd=bw["h"])
    b = forced.orbit(p, N, dt, S)
    for key in ("val", "slope", "inc"):
        np.testing.assert_array_equal(a[key], b[key])
    # halve the number of forward steps (merge pairs): still an orbit, 5th order accurate, not the same bits
    h2 = fw["h"][:len(fw["h"]) // 2 * 2].reshape(-1, 2).sum(axis=1)
    if len(fw["h"]) % 2:
        h2 = np.append(h2, fw["h"][-1])
    forced.set_adaptive((rtol, atol), forced_fwd=h2, forced_bwd=bw["h"])
    c = forced.orbit(p, N, dt, S)
    assert c["status"] == 0 and not np.array_equal(a["val"], c["val"])
    np.testing.assert_allclose(c["val"][1], a["val"][1], rtol=1e-9)
