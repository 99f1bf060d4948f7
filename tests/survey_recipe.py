"""SURVEY 8(d)-1's nu0 rule, run with the ORACLE's coarse orbit (test-side input preparation).

`workloads.draw_params` places nu0 with a closed-form estimate (reading D7: the generator module holds none of
the method's arithmetic), which leaves every walker 1.6-5 observation lengths from plunge.  The survey's own rule -- choose
nu0 by bisection in log nu0 so that the coarse RK4 orbit first reaches nu >= nu_LSO(e) at t_pl = f_pl * T_obs,
f_pl in [1.25, 3] -- needs the integrator, so it lives here, next to the tests, and calls only `oracle/`.
"""
import numpy as np

from paper_2311_17174_b200 import workloads as W


def nu0_for_plunge_at(oracle, p, N, dt, f_pl, S=256):
    """nu0 [Hz] for which walker `p` plunges at f_pl * N * dt (to within one coarse interval), by the oracle's RK4"""
    p = np.array(p, dtype=np.float64)
    n_long = int(np.ceil(f_pl * N / S)) * S
    lso = W.nu_lso_hz(p[W.P_M], p[W.P_E0])
    lo, hi = np.log(0.02 * lso), np.log(0.999 * lso)

    def plunges(lognu):
        q = p.copy()
        q[W.P_NU0] = np.exp(lognu)
        return (oracle.orbit(q, n_long, dt, S)["status"] & 2) != 0

    if not plunges(hi) or plunges(lo):
        raise ValueError("plunge time not bracketed")
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if plunges(mid):
            hi = mid
        else:
            lo = mid
    return float(np.exp(lo))          # the largest nu0 that does NOT plunge before f_pl * T_obs


def with_plunging_walkers(oracle, P, cfg, rows, f_pl=(1.25, 1.35, 1.5)):
    """copy of P whose `rows` chirp as the survey prescribes: plunge at f_pl[i] * T_obs after the window starts"""
    P = P.copy()
    for r, f in zip(rows, f_pl):
        P[r, W.P_NU0] = nu0_for_plunge_at(oracle, P[r], cfg.N, cfg.dt, f)
    return P
