"""Seeded synthetic inputs for the EMRI_MC hot path (shared by tests, bench.py and the oracle tests).

This module holds NO arithmetic of the method itself (no orbit integration, no waveform, no
transform, no likelihood): only the recipes of DESIGN.md section 4 / SURVEY.md 8(d)-1 that turn
`BASELINE.json:configs[i]` into a parameter matrix, a noise curve and a noise realisation.  The
paper measures on no public dataset (its workload is a synthetic injection), so
these stand in for its "1 yr at 0.1 Hz, 8 walkers" run at the configs' shapes.

Parameter row (P = 17; first three are M, mu, S/M^2 as PAPER.md:149 asks):
  0 M [Msun]  1 mu [Msun]  2 a=S/M^2  3 e0  4 nu0 [Hz]  5 Phi0  6 gamma~0  7 alpha0  8 lambda
  9 theta_S  10 phi_S  11 theta_K  12 phi_K [rad]  13 D_L [Gpc]  14 Xi0  15 n_Xi  16 delta_T=c_T-1
"""
import dataclasses

import numpy as np

NPAR = 17
(P_M, P_MU, P_A, P_E0, P_NU0, P_PHI0, P_GAM0, P_ALP0, P_LAM, P_THS, P_PHS, P_THK, P_PHK, P_DL, P_XI0,
 P_NXI, P_DELT) = range(NPAR)

MSUN_SEC = 4.925490947e-6      # G Msun / c^3 [s]
YEAR_SEC = 31557600.0          # Julian year [s]


@dataclasses.dataclass(frozen=True)
class Config:
    """One entry of BASELINE.json:configs."""
    index: int
    K: int
    N: int
    dt: float
    n_max: int
    seed: int
    log10_M: tuple      # range, or a single value
    log10_mu: tuple
    a: tuple
    e0: tuple
    DL: tuple
    modified_gravity: bool
    noise_seed: int     # 0 = noise-less data (injection only)
    note: str = ""

    @property
    def T_obs(self):
        return self.N * self.dt


CONFIGS = (
    Config(0, 8, 1 << 16, 15.0, 5, 0, (6.0, 6.0), (1.0, 1.0), (0.5, 0.5), (0.0, 0.1), (1.0, 1.0), False, 0,
           "small case the oracle finishes in seconds"),
    Config(1, 64, 1 << 20, 15.0, 10, 1, (5.5, 6.5), (0.5, 1.5), (0.0, 0.95), (0.0, 0.3), (0.5, 3.0), False, 1001,
           "bench workload; injection + coloured noise"),
    Config(2, 256, 1 << 21, 15.0, 20, 2, (5.5, 6.5), (0.5, 1.5), (0.0, 0.95), (0.0, 0.4), (0.5, 3.0), True, 0,
           "1 yr, both channels, modified gravity"),
    Config(3, 1024, 1 << 21, 15.0, 30, 3, (5.0, 7.0), (0.0, 2.0), (0.0, 0.95), (0.0, 0.5), (0.5, 3.0), True, 1003,
           "logL only"),
    Config(4, 512, 1 << 21, 15.0, 20, 4, (5.5, 6.5), (0.5, 1.5), (0.0, 0.95), (0.0, 0.3), (0.5, 3.0), False, 1004,
           "ensemble MCMC, 200 stretch-move steps"),
    # not in BASELINE.json: the shape of the paper's own run: 8 walkers, 4 free parameters
    # (M, mu, S/M^2, Xi0), one year at 0.1 Hz (dt = 10 s; N = 3 * 2^20 = 364.1 d), noise-less data, orbit anchored at the
    # LSO with e_LSO = 0.3 and the angles of PAPER.md:147; n_max is not stated in the paper (20 here), nor n of Eq. 6 (2)
    Config(5, 8, 3 << 20, 10.0, 20, 5, (6.0, 6.0), (1.0, 1.0), (0.1, 0.1), (0.3, 0.3), (1.0, 1.0), False, 0,
           "the paper's run shape: 8 walkers, 4 free parameters, 1 yr at 0.1 Hz, anchored at the LSO"),
)
PAPER_RUN_FREE = (P_M, P_MU, P_A, P_XI0)


def scaled(cfg, K=None, N=None, n_max=None):
    """The same recipe at a reduced shape (parity tests that must finish in seconds)."""
    return dataclasses.replace(cfg, K=K or cfg.K, N=N or cfg.N, n_max=n_max or cfg.n_max)


# ----------------------------------------------------------------------------- nu0 rule
def nu_lso_hz(M_msun, e):
    """plunge frequency, used here only to place nu0 below it."""
    return ((1.0 - e * e) / (6.0 + 2.0 * e)) ** 1.5 / (2.0 * np.pi * M_msun * MSUN_SEC)


def nu0_for_plunge_after(M_msun, mu_msun, e0, t_plunge_sec):
    """"nu0 so plunge > T" (BASELINE.json:configs[0]).

    Closed-form estimate, not an integration: the leading-order circular chirp
    nu' = K nu^{11/3} reaches nu_LSO after (3/8K)(nu0^{-8/3} - nu_LSO^{-8/3}); eccentricity
    shortens that by roughly (1-e^2)^{7/2}.  The PN and spin terms of the real model make the true
    plunge time 0.58-0.85 of this estimate (more for the heaviest systems; measured with the oracle),
    so `draw_params` asks for 2.2-4.5 observation lengths to land on SURVEY 8(d)-1's strongly
    chirping regime, plunge 1.3-4 T_obs after the window starts (median 2-2.8); tests check that no
    walker of any config sets the plunge bit.
    """
    Ms, mus = M_msun * MSUN_SEC, mu_msun * MSUN_SEC
    Kc = 96.0 / (10.0 * np.pi) * mus / Ms ** 3 * (2.0 * np.pi * Ms) ** (11.0 / 3.0)
    F = (1.0 - e0 * e0) ** 3.5
    nl = nu_lso_hz(M_msun, e0)
    return (t_plunge_sec * 8.0 * Kc / (3.0 * F) + nl ** (-8.0 / 3.0)) ** (-3.0 / 8.0)


def _u(rng, lohi, size=None):
    lo, hi = lohi
    return rng.uniform(lo, hi, size) if hi > lo else (np.full(size, lo) if size else lo)


def _draw_row(rng, cfg):
    p = np.zeros(NPAR)
    while True:
        p[P_M] = 10.0 ** _u(rng, cfg.log10_M)
        p[P_MU] = 10.0 ** _u(rng, cfg.log10_mu)
        p[P_A] = _u(rng, cfg.a)
        p[P_E0] = _u(rng, cfg.e0)
        f_pl = rng.uniform(2.2, 4.5)               # ESTIMATED plunge time in units of T_obs (true: 0.58-0.85 of it)
        p[P_NU0] = nu0_for_plunge_after(p[P_M], p[P_MU], p[P_E0], f_pl * cfg.T_obs)
        p[P_PHI0], p[P_GAM0], p[P_ALP0] = rng.uniform(0.0, 2.0 * np.pi, 3)
        p[P_LAM] = rng.uniform(0.0, np.pi)
        p[P_THS] = np.arccos(rng.uniform(-1.0, 1.0))
        p[P_PHS] = rng.uniform(0.0, 2.0 * np.pi)
        p[P_THK] = np.arccos(rng.uniform(-1.0, 1.0))
        p[P_PHK] = rng.uniform(0.0, 2.0 * np.pi)
        p[P_DL] = _u(rng, cfg.DL)
        if cfg.modified_gravity:
            p[P_XI0] = rng.uniform(0.8, 1.2)
            p[P_NXI] = rng.uniform(1.0, 3.0)
            p[P_DELT] = rng.uniform(-1e-15, 1e-15)
        else:
            p[P_XI0], p[P_NXI], p[P_DELT] = 1.0, 0.0, 0.0
        # reading R16: reject draws within 1e-6 of a coordinate pole of the response
        if min(np.sin(p[P_LAM]), np.sin(p[P_THS]), np.sin(p[P_THK])) > 1e-6:
            return p


def draw_params(cfg, K=None):
    """params[K][17], walker-major draws from numpy default_rng(cfg.seed)."""
    rng = np.random.default_rng(cfg.seed)
    K = cfg.K if K is None else K
    if cfg.index == 4:
        return _draw_mcmc_ensemble(rng, cfg, K)
    if cfg.index == 5:
        return _draw_paper_run(rng, K)
    return np.stack([_draw_row(rng, cfg) for _ in range(K)])


def _draw_mcmc_ensemble(rng, cfg, K):
    """config 4: walkers in a small ball around the injected theta* (row 0 of the result is theta*)."""
    star = _draw_row(rng, cfg)
    P = np.tile(star, (K, 1))
    g = rng.standard_normal((K, NPAR))
    g[0] = 0.0
    P[:, :5] *= 1.0 + 1e-8 * g[:, :5]
    P[:, 5:13] += 1e-3 * g[:, 5:13]
    P[:, P_DL] *= 1.0 + 1e-3 * g[:, P_DL]
    P[:, P_XI0] += 1e-3 * g[:, P_XI0]
    P[:, P_NXI] = np.abs(1e-3 * g[:, P_NXI])
    P[:, P_DELT] = 1e-17 * g[:, P_DELT]
    return P


def _draw_paper_run(rng, K):
    """the paper's fiducial system at the LSO and K walkers in a small ball in its 4 free parameters"""
    star = np.zeros(NPAR)
    star[P_M], star[P_MU], star[P_A], star[P_E0], star[P_NU0] = 1e6, 10.0, 0.1, 0.3, 1e-3
    star[P_LAM], star[P_THS], star[P_PHS], star[P_THK], star[P_PHK] = np.pi / 6, np.pi / 4, 0.0, np.pi / 8, 0.0
    star[P_DL], star[P_XI0], star[P_NXI] = 1.0, 1.0, 2.0
    P = np.tile(star, (K, 1))
    g = rng.standard_normal((K, NPAR))
    g[0] = 0.0
    P[:, P_M] *= 1.0 + 1e-7 * g[:, P_M]
    P[:, P_MU] *= 1.0 + 1e-7 * g[:, P_MU]
    P[:, P_A] += 1e-7 * g[:, P_A]
    P[:, P_XI0] += 1e-2 * g[:, P_XI0]
    return P


def prior_box(cfg):
    """Uniform box prior of config 4: lo[17], hi[17] (the config-1 ranges + propagation ranges); config 5: only the paper's
    four free parameters have a range, every other column is held fixed (lo = hi)."""
    lo, hi = np.zeros(NPAR), np.zeros(NPAR)
    if cfg.index == 5:
        lo[P_M], hi[P_M] = 1e5, 1e7
        lo[P_MU], hi[P_MU] = 1.0, 100.0
        lo[P_A], hi[P_A] = 0.0, 0.95
        lo[P_XI0], hi[P_XI0] = 0.5, 1.5
        return lo, hi
    lo[P_M], hi[P_M] = 10.0 ** cfg.log10_M[0], 10.0 ** cfg.log10_M[1]
    lo[P_MU], hi[P_MU] = 10.0 ** cfg.log10_mu[0], 10.0 ** cfg.log10_mu[1]
    lo[P_A], hi[P_A] = 0.0, 0.95
    lo[P_E0], hi[P_E0] = 0.0, 0.5
    lo[P_NU0], hi[P_NU0] = 1e-5, 1e-1
    for c in (P_PHI0, P_GAM0, P_ALP0, P_PHS, P_PHK):
        lo[c], hi[c] = -2.0 * np.pi, 4.0 * np.pi
    for c in (P_LAM, P_THS, P_THK):
        lo[c], hi[c] = 1e-6, np.pi - 1e-6
    lo[P_DL], hi[P_DL] = 0.1, 10.0
    lo[P_XI0], hi[P_XI0] = 0.5, 1.5
    lo[P_NXI], hi[P_NXI] = 0.0, 4.0
    lo[P_DELT], hi[P_DELT] = -1e-14, 1e-14
    return lo, hi


# ----------------------------------------------------------------------------- noise curves
def freqs(N, dt):
    return np.arange(N // 2 + 1) / (N * dt)


def lisa_psd_barack_cutler(N, dt):
    """One-sided S_n(f_m) [1/Hz], the analytic model of the paper's example (PAPER.md:116, :171,
    ref. [1]); restated from the literature (fidelity: literature only -- it is an input).
    psd[0] = psd[N/2] = +inf masks DC and Nyquist."""
    f = freqs(N, dt)
    with np.errstate(divide="ignore", invalid="ignore", over="ignore"):
        s_inst = 9.18e-52 * f ** -4.0 + 1.59e-41 + 9.18e-38 * f ** 2.0
        s_gal = 2.1e-45 * f ** (-7.0 / 3.0)
        s_exgal = 4.2e-47 * f ** (-7.0 / 3.0)
        dNdf = 2e-3 * f ** (-11.0 / 3.0)
        kappa_over_T = 1.5 / YEAR_SEC
        s = np.minimum(s_inst * np.exp(np.minimum(kappa_over_T * dNdf, 700.0)), s_inst + s_gal) + s_exgal
    s[0] = np.inf
    s[-1] = np.inf
    return s


def lisa_psd_robson(N, dt):
    """Second noise model of the paper (refs. [51, 52]): sky-averaged sensitivity
    with the 1-yr galactic confusion fit; restated from the literature (an input only)."""
    f = freqs(N, dt)
    L, fstar = 2.5e9, 19.09e-3
    with np.errstate(divide="ignore", invalid="ignore", over="ignore"):
        p_oms = (1.5e-11) ** 2 * (1.0 + (2e-3 / f) ** 4)
        p_acc = (3e-15) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4)
        s = 10.0 / (3.0 * L * L) * (p_oms + 2.0 * (1.0 + np.cos(f / fstar) ** 2) * p_acc / (2.0 * np.pi * f) ** 4)
        s *= 1.0 + 0.6 * (f / fstar) ** 2
        s_c = 9e-45 * f ** (-7.0 / 3.0) * np.exp(-f ** 0.171 + 292.0 * f * np.sin(1020.0 * f))
        s_c *= 1.0 + np.tanh(1680.0 * (0.00215 - f))
        s = s + s_c
    s[0] = np.inf
    s[-1] = np.inf
    return s


def noise_fft(N, dt, psd, seed):
    """Coloured Gaussian noise directly in the frequency domain, un-normalised-DFT units:
    Re, Im ~ N(0, S_n N / (4 dt)) for unmasked bins, both channels: complex [2][N/2+1]."""
    rng = np.random.default_rng(seed)
    ok = np.isfinite(psd) & (psd > 0)
    sig = np.where(ok, np.sqrt(np.where(ok, psd, 0.0) * N / (4.0 * dt)), 0.0)
    out = np.empty((2, N // 2 + 1), dtype=np.complex128)
    for ch in range(2):
        out[ch] = sig * (rng.standard_normal(N // 2 + 1) + 1j * rng.standard_normal(N // 2 + 1))
    return out


def parity_walker_subset(params, n=16, seed=12345):
    """Seeded subset of walkers the oracle is run on at full N: indices 0-3,
    argmax e0, argmin M, argmax mu/M, then seeded draws."""
    K = params.shape[0]
    if K <= n:
        return np.arange(K)
    # the three extreme walkers come FIRST and are never dropped; then 0..3; then seeded draws up to n
    pick = []
    for k in (int(np.argmax(params[:, P_E0])), int(np.argmin(params[:, P_M])),
              int(np.argmax(params[:, P_MU] / params[:, P_M])), 0, 1, 2, 3):
        if k not in pick and len(pick) < n:
            pick.append(k)
    rng = np.random.default_rng(seed)
    for k in rng.permutation(K):
        if len(pick) >= n:
            break
        if int(k) not in pick:
            pick.append(int(k))
    return np.array(sorted(pick))


def paper_fig1_params(path):
    """params[9][17] of the paper's Figure 1 grid (tests/golden/paper_fig1_parameters.txt), for a
    plan anchored at the LSO: e0 = e_LSO, Phi0 = gamma0 = alpha0 = 0 at plunge; nu0 is ignored in that mode; GR."""
    rows = np.loadtxt(path)
    P = np.zeros((rows.shape[0], NPAR))
    P[:, P_M], P[:, P_MU], P[:, P_A], P[:, P_E0] = rows[:, 0], rows[:, 1], rows[:, 2], rows[:, 3]
    P[:, P_THS], P[:, P_PHS], P[:, P_THK], P[:, P_PHK], P[:, P_LAM], P[:, P_DL] = (rows[:, c] for c in range(4, 10))
    P[:, P_NU0] = 1e-3
    P[:, P_XI0] = 1.0
    return P
