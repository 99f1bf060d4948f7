"""ctypes binding of the CPU oracle (oracle/emri_oracle.cpp) -- TEST INFRASTRUCTURE.

`Oracle()` loads the double build, `Oracle(long_double=True)` the 80-bit diagnostic build;
`Oracle(anchor=True)` reads parameter rows as the state at plunge (reading D12) -- a property of the
instance, passed to the library as an explicit argument of every orbit / waveform call (no process-wide state).
Argument marshalling only; every number comes out of emri_oracle.cpp.
"""
import ctypes as C

import numpy as np

from . import build_oracle

NPAR = 17
H0_DEFAULT = 67.4
OM_DEFAULT = 0.315

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int64)
_i32p = C.POINTER(C.c_int32)


def _d(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    def __init__(self, long_double=False, anchor=False, adaptive=None):
        self.anchor = 1 if anchor else 0
        self.set_adaptive(adaptive)
        lib, lib_ld = build_oracle.build()
        self.lib = L = C.CDLL(lib_ld if long_double else lib)
        L.emri_o_real_bits.restype = C.c_int
        L.emri_o_bessel_j.restype = C.c_double
        L.emri_o_bessel_j.argtypes = [C.c_int, C.c_double]
        L.emri_o_brackets.argtypes = [C.c_int, C.c_double, _dp]
        L.emri_o_nu_lso.restype = C.c_double
        L.emri_o_nu_lso.argtypes = [C.c_double, C.c_double]
        L.emri_o_cosmology.argtypes = [C.c_double, C.c_double, C.c_double, _dp]
        L.emri_o_dL_sec.restype = C.c_double
        L.emri_o_dL_sec.argtypes = [C.c_double] * 3
        L.emri_o_xi.restype = C.c_double
        L.emri_o_xi.argtypes = [C.c_double] * 3
        L.emri_o_walker_scalars.argtypes = [_dp, C.c_double, C.c_double, _dp]
        L.emri_o_rhs.argtypes = [_dp, _dp, C.c_int, _dp]
        L.emri_o_orbit.argtypes = [_dp, C.c_int64, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double,
                                   _dp, _dp, _dp, _ip, C.c_int, _dp]
        L.emri_o_orbit_at.argtypes = [_dp, C.c_int64, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double,
                                      _ip, C.c_int64, _dp, C.c_int, _dp]
        L.emri_o_hermite1.restype = C.c_double
        L.emri_o_hermite1.argtypes = [C.c_double] * 6
        L.emri_o_geometry.argtypes = [_dp, C.c_double, C.c_double, _dp]
        L.emri_o_antenna.argtypes = [C.c_double, C.c_double, C.c_double, _dp]
        L.emri_o_waveform.restype = C.c_int
        L.emri_o_waveform.argtypes = [_dp, C.c_int64, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double,
                                      _ip, C.c_int64, _dp, _dp, _dp, _dp, C.c_int, _dp]
        L.emri_o_waveform_batch.argtypes = [_dp, C.c_int, C.c_int64, C.c_double, C.c_int, C.c_int,
                                            C.c_double, C.c_double, _dp, _i32p, C.c_int, _dp]
        L.emri_o_rfft.restype = C.c_int
        L.emri_o_rfft.argtypes = [_dp, C.c_int64, _dp]
        L.emri_o_dft_naive.argtypes = [_dp, C.c_int64, _dp]
        L.emri_o_loglike.restype = C.c_double
        L.emri_o_loglike.argtypes = [_dp, _dp, _dp, C.c_int64, C.c_double]
        L.emri_o_loglike_fdep.restype = C.c_double
        L.emri_o_loglike_fdep.argtypes = [_dp, _dp, _dp, C.c_int64, C.c_double, _dp, C.c_double]
        L.emri_o_inner.restype = C.c_double
        L.emri_o_inner.argtypes = [_dp, _dp, _dp, C.c_int64, C.c_double]
        L.emri_o_loglike_batch.restype = C.c_int
        L.emri_o_loglike_batch.argtypes = [_dp, C.c_int, C.c_int64, C.c_double, C.c_int, C.c_int, C.c_double,
                                           C.c_double, _dp, _dp, _dp, _i32p, _dp, C.c_int, _dp]

    def set_adaptive(self, adaptive, forced_fwd=None, forced_bwd=None):
        """None: the fixed-step RK4 of S3.  (rtol, atol[5]): the embedded Dormand-Prince pair with dense output (S3', D14).
        forced_fwd / forced_bwd: prescribed step sizes of the two branches (teacher-forced parity), else the controller's"""
        if adaptive is None:
            self._adaptive, self._adp = None, None
        else:
            rtol, atol = adaptive
            ff = np.zeros(0) if forced_fwd is None else np.asarray(forced_fwd, dtype=np.float64)
            fb = np.zeros(0) if forced_bwd is None else np.asarray(forced_bwd, dtype=np.float64)
            self._adaptive = np.ascontiguousarray(np.concatenate([[float(rtol)], np.broadcast_to(atol, (5,)),
                                                                  [float(ff.size), float(fb.size)], ff, fb]), dtype=np.float64)
            self._adp = self._adaptive.ctypes.data_as(_dp)

    def dp5_forced_errors(self, params, rtol, atol, h, pn_mask=3, H0=H0_DEFAULT, Om=OM_DEFAULT):
        """the controller's error norm (this implementation's) of each step of the prescribed sequence h taken from the
        row's state at t = 0 -- the validity half of the teacher-forced protocol (D14)"""
        p = _f64(params)
        at = np.ascontiguousarray(np.broadcast_to(atol, (5,)), dtype=np.float64)
        h = np.ascontiguousarray(h, dtype=np.float64)
        err = np.zeros(len(h))
        self.lib.emri_o_dp5_forced_errors.restype = C.c_int64
        self.lib.emri_o_dp5_forced_errors.argtypes = [_dp, C.c_double, _dp, C.c_int, C.c_double, C.c_double, _dp, C.c_int64, _dp]
        n = self.lib.emri_o_dp5_forced_errors(_d(p), float(rtol), _d(at), pn_mask, H0, Om, _d(h), len(h), _d(err))
        return err[:n]

    def dp5_steps(self, params, t_end, rtol, atol, pn_mask=3, stop_at_plunge=False, max_steps=200000,
                  H0=H0_DEFAULT, Om=OM_DEFAULT):
        """accepted steps of the adaptive integration from t = 0 to t_end -> dict(t, h, y[n][5], turns[n][3], Q[n][5][4], stop, t_reached)"""
        p = _f64(params)
        at = np.ascontiguousarray(np.broadcast_to(atol, (5,)), dtype=np.float64)
        t, h = np.zeros(max_steps), np.zeros(max_steps)
        y, tu, Q = np.zeros((max_steps, 5)), np.zeros((max_steps, 3)), np.zeros((max_steps, 5, 4))
        info = np.zeros(2)
        self.lib.emri_o_dp5_steps.restype = C.c_int64
        self.lib.emri_o_dp5_steps.argtypes = [_dp, C.c_double, C.c_double, _dp, C.c_int, C.c_double, C.c_double, C.c_int,
                                              C.c_int64, _dp, _dp, _dp, _dp, _dp, _dp]
        n = self.lib.emri_o_dp5_steps(_d(p), float(t_end), float(rtol), _d(at), pn_mask, H0, Om, 1 if stop_at_plunge else 0,
                                      max_steps, _d(t), _d(h), _d(y), _d(tu), _d(Q), _d(info))
        n = min(int(n), max_steps)
        return dict(t=t[:n], h=h[:n], y=y[:n], turns=tu[:n], Q=Q[:n], stop=int(info[0]), t_reached=float(info[1]))

    def set_anchor(self, at_lso):
        """False (default): the parameter row is the state at t = 0; True: at plunge, at the last coarse node (D12).
        Affects this instance only."""
        self.anchor = 1 if at_lso else 0

    # ---- scalars
    def real_bits(self):
        return self.lib.emri_o_real_bits()

    def bessel_j(self, k, x):
        return self.lib.emri_o_bessel_j(int(k), float(x))

    def brackets(self, n, e):
        out = np.zeros(3)
        self.lib.emri_o_brackets(int(n), float(e), _d(out))
        return out

    def nu_lso(self, M_msun, e):
        return self.lib.emri_o_nu_lso(float(M_msun), float(e))

    def cosmology(self, DL_gpc, H0=H0_DEFAULT, Om=OM_DEFAULT):
        """-> (z, lookback time [s], d_L(z) [s])"""
        out = np.zeros(3)
        self.lib.emri_o_cosmology(float(DL_gpc), H0, Om, _d(out))
        return tuple(out)

    def dL_sec(self, z, H0=H0_DEFAULT, Om=OM_DEFAULT):
        return self.lib.emri_o_dL_sec(float(z), H0, Om)

    def xi(self, Xi0, nXi, z):
        return self.lib.emri_o_xi(float(Xi0), float(nXi), float(z))

    def walker_scalars(self, params, H0=H0_DEFAULT, Om=OM_DEFAULT):
        """-> dict(Ms, mus, Ds, z, Xi, amp, dT, status)"""
        p = _f64(params)
        out = np.zeros(8)
        self.lib.emri_o_walker_scalars(_d(p), H0, Om, _d(out))
        keys = ("Ms", "mus", "Ds", "z", "Xi", "amp", "dT", "status")
        d = dict(zip(keys, out))
        d["status"] = int(d["status"])
        return d

    def rhs(self, params, y, pn_mask=3):
        p, yy, f = _f64(params), _f64(y), np.zeros(5)
        self.lib.emri_o_rhs(_d(p), _d(yy), int(pn_mask), _d(f))
        return f

    # ---- orbit
    def orbit(self, params, N, dt, S=256, pn_mask=3, H0=H0_DEFAULT, Om=OM_DEFAULT):
        """-> dict(val[5][Nn], slope[5][Nn], inc[5][Nn], Nn, jpl, status); node j at column j+1"""
        p = _f64(params)
        Nn = (N + S - 1) // S + 3
        val, slope, inc = (np.zeros((5, Nn)) for _ in range(3))
        info = np.zeros(3, dtype=np.int64)
        self.lib.emri_o_orbit(_d(p), N, dt, S, pn_mask, H0, Om, _d(val), _d(slope), _d(inc),
                              info.ctypes.data_as(_ip), self.anchor, self._adp)
        return dict(val=val, slope=slope, inc=inc, Nn=int(info[0]), jpl=int(info[1]), status=int(info[2]))

    def orbit_at(self, params, N, dt, idx, S=256, pn_mask=3, H0=H0_DEFAULT, Om=OM_DEFAULT):
        p = _f64(params)
        ii = np.ascontiguousarray(idx, dtype=np.int64)
        out = np.zeros((5, ii.size))
        self.lib.emri_o_orbit_at(_d(p), N, dt, S, pn_mask, H0, Om, ii.ctypes.data_as(_ip), ii.size, _d(out), self.anchor, self._adp)
        return out

    def hermite1(self, y0, inc, m0, m1, Delta, s):
        return self.lib.emri_o_hermite1(y0, inc, m0, m1, Delta, s)

    def geometry(self, params, alpha, phibar):
        p = _f64(params)
        out = np.zeros(13)
        self.lib.emri_o_geometry(_d(p), float(alpha), float(phibar), _d(out))
        keys = ("cthL", "sthL", "phL", "Ln", "Sn", "sinb", "cosb", "beta", "cthd", "phid", "psi", "Npsi", "Dpsi")
        return dict(zip(keys, out))

    def antenna(self, cthd, phid, psi):
        F = np.zeros(4)
        self.lib.emri_o_antenna(float(cthd), float(phid), float(psi), _d(F))
        return F

    # ---- waveform
    def waveform(self, params, N, dt, n_max, S=256, idx=None, H0=H0_DEFAULT, Om=OM_DEFAULT, amplitudes=False):
        """one walker -> (hI, hII, status) [+ (A+, Ax) if amplitudes]; idx selects samples"""
        p = _f64(params)
        if idx is None:
            ii, n, ptr = None, N, None
        else:
            ii = np.ascontiguousarray(idx, dtype=np.int64)
            n, ptr = ii.size, ii.ctypes.data_as(_ip)
        hI, hII = np.zeros(n), np.zeros(n)
        Ap, Ax = (np.zeros(n), np.zeros(n)) if amplitudes else (None, None)
        st = self.lib.emri_o_waveform(_d(p), N, dt, n_max, S, H0, Om, ptr, n, _d(hI), _d(hII),
                                      _d(Ap) if amplitudes else None, _d(Ax) if amplitudes else None, self.anchor, self._adp)
        return (hI, hII, st, Ap, Ax) if amplitudes else (hI, hII, st)

    def waveform_batch(self, params, N, dt, n_max, S=256, H0=H0_DEFAULT, Om=OM_DEFAULT):
        """-> h[K][2][N], status[K]; OpenMP over walkers"""
        p = _f64(params).reshape(-1, NPAR)
        K = p.shape[0]
        h = np.zeros((K, 2, N))
        st = np.zeros(K, dtype=np.int32)
        self.lib.emri_o_waveform_batch(_d(p), K, N, dt, n_max, S, H0, Om, _d(h), st.ctypes.data_as(_i32p), self.anchor, self._adp)
        return h, st

    # ---- transform and likelihood
    def rfft(self, h):
        h = _f64(h)
        N = h.size
        H = np.zeros(2 * (N // 2 + 1))
        rc = self.lib.emri_o_rfft(_d(h), N, _d(H))
        if rc:
            raise ValueError("oracle rfft needs a power-of-two length")
        return H.view(np.complex128)

    def dft_naive(self, h):
        h = _f64(h)
        N = h.size
        H = np.zeros(2 * (N // 2 + 1))
        self.lib.emri_o_dft_naive(_d(h), N, _d(H))
        return H.view(np.complex128)

    def loglike(self, H, D, psd, N, dt):
        """H, D: complex [2][N/2+1]"""
        Hc = np.ascontiguousarray(H, dtype=np.complex128)
        Dc = np.ascontiguousarray(D, dtype=np.complex128)
        s = _f64(psd)
        return self.lib.emri_o_loglike(_d(Hc.view(np.float64)), _d(Dc.view(np.float64)), _d(s), N, dt)

    def loglike_fdep(self, H, D, psd, N, dt, fcoef, fstar=1e-3):
        """Eq. 8 with the frequency-dependent propagation factor of Eq. 7 applied to H (reading D11)"""
        Hc = np.ascontiguousarray(H, dtype=np.complex128)
        Dc = np.ascontiguousarray(D, dtype=np.complex128)
        s, fc = _f64(psd), _f64(fcoef)
        return self.lib.emri_o_loglike_fdep(_d(Hc.view(np.float64)), _d(Dc.view(np.float64)), _d(s), N, dt, _d(fc), fstar)

    def inner(self, A, B, psd, N, dt):
        Ac = np.ascontiguousarray(A, dtype=np.complex128)
        Bc = np.ascontiguousarray(B, dtype=np.complex128)
        s = _f64(psd)
        return self.lib.emri_o_inner(_d(Ac.view(np.float64)), _d(Bc.view(np.float64)), _d(s), N, dt)

    def loglike_batch(self, params, N, dt, n_max, D, psd, S=256, H0=H0_DEFAULT, Om=OM_DEFAULT, spectra=False):
        """whole path for K walkers -> (logL[K], status[K]) [+ spectra[K][2][N/2+1] complex]"""
        p = _f64(params).reshape(-1, NPAR)
        K = p.shape[0]
        Dc = np.ascontiguousarray(D, dtype=np.complex128)
        s = _f64(psd)
        logL = np.zeros(K)
        st = np.zeros(K, dtype=np.int32)
        sp = np.zeros((K, 2, N // 2 + 1), dtype=np.complex128) if spectra else None
        rc = self.lib.emri_o_loglike_batch(_d(p), K, N, dt, n_max, S, H0, Om, _d(Dc.view(np.float64)), _d(s),
                                           _d(logL), st.ctypes.data_as(_i32p),
                                           _d(sp.view(np.float64)) if spectra else None, self.anchor, self._adp)
        if rc:
            raise ValueError("oracle loglike_batch failed (N must be a power of two)")
        return (logL, st, sp) if spectra else (logL, st)
