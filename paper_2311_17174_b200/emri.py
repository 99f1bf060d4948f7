"""Thin ctypes binding of include/emri.h -- argument marshalling only.

Every step of the path runs in the CUDA library (csrc/emri.cu).  PyTorch supplies device memory
(`tensor.data_ptr()`) and the stream (`torch.cuda.current_stream()`); nothing is computed here and
there is no CPU fallback: `load()` raises if libemri_b200.so is missing or does not load.
"""
import ctypes as C
import os

import numpy as np

NPAR = 17
NODE_STRIDE = 16
ST_BADPARAM, ST_PLUNGE, ST_DELAY, ST_STATE = 1, 2, 4, 8
_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libemri_b200.so")
_lib = None

EXPORTS = (
    "emri_strerror", "emri_plan_create", "emri_plan_destroy", "emri_plan_set_cosmology",
    "emri_plan_set_coarse_stride", "emri_plan_set_orbit_schedule", "emri_plan_set_anchor", "emri_plan_set_integrator", "emri_plan_orbit_steps", "emri_plan_orbit_report",
    "emri_plan_synth_report", "emri_plan_set_synth_debug", "emri_plan_set_unit_tiles", "emri_plan_set_series_tolerance", "emri_plan_set_transform", "emri_plan_transform_is_fused", "emri_plan_set_graphs", "emri_plan_graph_stats", "emri_plan_set_chunk", "emri_orbit", "emri_plan_num_nodes", "emri_waveform",
    "emri_waveform_fft", "emri_data_fft", "emri_loglike", "emri_loglike_fdep", "emri_loglike_host", "emri_plan_enable_timings",
    "emri_plan_get_timings", "emri_plan_last_cuda_error", "emri_plan_last_launch_count", "emri_plan_workspace_bytes", "emri_stretch_step",
    "emri_spectra_loglike_static", "emri_static_scratch_need", "emri_static_last_cuda_error",
)


class EmriError(RuntimeError):
    pass


def load():
    """dlopen libemri_b200.so and declare the prototypes of include/emri.h.  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise EmriError(f"{_LIB_PATH} is missing: build it with `python -m paper_2311_17174_b200.build` "
                        "(there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    vp, i32, i64, dbl, u64 = C.c_void_p, C.c_int, C.c_int64, C.c_double, C.c_uint64
    L.emri_strerror.restype = C.c_char_p
    L.emri_strerror.argtypes = [i32]
    L.emri_plan_create.argtypes = [C.POINTER(vp), i64, dbl, i32, i32, vp]
    L.emri_plan_destroy.argtypes = [vp]
    L.emri_plan_set_cosmology.argtypes = [vp, dbl, dbl]
    L.emri_plan_set_coarse_stride.argtypes = [vp, i32]
    L.emri_plan_set_chunk.argtypes = [vp, i32]
    L.emri_plan_set_orbit_schedule.argtypes = [vp, i32]
    L.emri_plan_orbit_report.argtypes = [vp, i32, vp]
    L.emri_plan_set_anchor.argtypes = [vp, i32]
    L.emri_plan_set_integrator.argtypes = [vp, i32, dbl, vp, i32]
    L.emri_plan_orbit_steps.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp]
    L.emri_plan_synth_report.argtypes = [vp, vp]
    L.emri_plan_set_synth_debug.argtypes = [vp, i32]
    L.emri_plan_set_unit_tiles.argtypes = [vp, i32]
    L.emri_plan_set_series_tolerance.argtypes = [vp, C.c_double]
    L.emri_plan_set_transform.argtypes = [vp, i32]
    L.emri_plan_set_graphs.argtypes = [vp, i32]
    L.emri_plan_graph_stats.argtypes = [vp, vp]
    L.emri_plan_transform_is_fused.argtypes = [vp]
    L.emri_orbit.argtypes = [vp, vp, i32, vp, vp, vp]
    L.emri_plan_num_nodes.restype = i64
    L.emri_plan_num_nodes.argtypes = [vp]
    L.emri_waveform.argtypes = [vp, vp, i32, vp, vp, vp, vp]
    L.emri_waveform_fft.argtypes = [vp, vp, i32, vp, vp, vp]
    L.emri_data_fft.argtypes = [vp, vp, vp, vp, vp]
    L.emri_loglike.argtypes = [vp, vp, i32, vp, vp, vp, vp]
    L.emri_loglike_host.argtypes = [vp, vp, i32, vp, vp, vp, vp]
    L.emri_loglike_fdep.argtypes = [vp, vp, i32, vp, dbl, vp, vp, vp, vp]
    L.emri_plan_enable_timings.argtypes = [vp, i32]
    L.emri_plan_get_timings.argtypes = [vp, C.POINTER(dbl)]
    L.emri_plan_last_cuda_error.argtypes = [vp]
    L.emri_plan_last_launch_count.argtypes = [vp]
    L.emri_plan_workspace_bytes.restype = i64
    L.emri_plan_workspace_bytes.argtypes = [vp]
    L.emri_stretch_step.argtypes = [vp, vp, vp, i32, vp, vp, vp, dbl, u64, i64, i32, vp, vp, vp]
    L.emri_spectra_loglike_static.argtypes = [vp, i32, i64, dbl, vp, vp, vp, vp]
    L.emri_static_scratch_need.restype = i64
    L.emri_static_scratch_need.argtypes = [i32, i64]
    L.emri_static_last_cuda_error.argtypes = []
    for name in EXPORTS:
        if name not in ("emri_strerror", "emri_plan_num_nodes", "emri_plan_workspace_bytes", "emri_static_scratch_need"):
            getattr(L, name).restype = i32
    _lib = L
    return L


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, dtype=None, shape=None):
    """device pointer of a contiguous CUDA tensor (None -> NULL)"""
    if t is None:
        return None
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise TypeError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


STATIC_SCRATCH_DOUBLES = 65536


def spectra_loglike_static(spectra, data_fft, psd, N, dt, logL):
    """emri_spectra_loglike_static: Eq. 8 from spectra the caller already holds, for code that must not allocate device
    memory (the whole card belongs to another pool, a fixed memory quota, or a host thread that cannot afford the
    device-wide synchronisation of cudaMalloc / cudaFree).  No plan is involved and this wrapper allocates nothing either,
    which is why `logL` is a required argument.  All tensors are contiguous CUDA tensors on the current device:
    spectra complex128 [K][2][N/2+1], data_fft complex128 [2][N/2+1], psd float64 [N/2+1] (masked like the `psd` of Plan),
    logL float64 [K].  Raises EmriError with the library's message when K ceil((N/2+1)/8192) > STATIC_SCRATCH_DOUBLES.
    Calls share one built-in scratch array per GPU: keep them on one stream.  The first call on a device also looks up that
    array's address; make it before any stream capture."""
    import torch
    L = load()
    K, Nf = spectra.shape[0], int(N) // 2 + 1
    rc = L.emri_spectra_loglike_static(_ptr(spectra, torch.complex128, (K, 2, Nf)), K, int(N), float(dt),
                                       _ptr(data_fft, torch.complex128, (2, Nf)), _ptr(psd, torch.float64, (Nf,)),
                                       _ptr(logL, torch.float64, (K,)), _stream())
    if rc != 0:
        raise EmriError(f"{L.emri_strerror(rc).decode()} (code {rc}, raw {L.emri_static_last_cuda_error()})")
    return logL


class Plan:
    """emri_plan_create(N, dt, n_max, K_max, psd) and the calls that use it (include/emri.h)."""

    def __init__(self, N, dt, n_max, K_max, psd=None):
        self._L = load()
        self._h = C.c_void_p()
        self.N, self.dt, self.n_max, self.K_max = int(N), float(dt), int(n_max), int(K_max)
        self.Nf = self.N // 2 + 1
        if psd is not None:
            psd = np.ascontiguousarray(psd, dtype=np.float64)
            if psd.shape != (self.Nf,):
                raise ValueError("psd must have N/2+1 entries")
        self._check(self._L.emri_plan_create(C.byref(self._h), self.N, self.dt, self.n_max, self.K_max,
                                              psd.ctypes.data_as(C.c_void_p) if psd is not None else None))

    def _check(self, rc):
        if rc != 0:
            raw = self._L.emri_plan_last_cuda_error(self._h) if self._h else 0
            raise EmriError(f"{self._L.emri_strerror(rc).decode()} (code {rc}, raw {raw})")

    def close(self):
        if getattr(self, "_h", None):
            self._L.emri_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- settings
    def set_cosmology(self, H0, Om):
        self._check(self._L.emri_plan_set_cosmology(self._h, H0, Om))

    def set_coarse_stride(self, S):
        self._check(self._L.emri_plan_set_coarse_stride(self._h, S))

    def set_orbit_schedule(self, schedule):
        """1 = parallel in time (default), 0 = sequential recursion (same scheme)"""
        self._check(self._L.emri_plan_set_orbit_schedule(self._h, int(schedule)))

    def set_anchor(self, at_lso):
        """False: the parameter row is the state at t = 0 (default); True: at plunge, at the end of the window"""
        self._check(self._L.emri_plan_set_anchor(self._h, 1 if at_lso else 0))

    def set_integrator(self, adaptive=None, max_steps=4096):
        """None: fixed-step RK4 (default).  (rtol, atol[5]): the embedded Dormand-Prince pair with dense output"""
        if adaptive is None:
            self._check(self._L.emri_plan_set_integrator(self._h, 0, 0.0, None, 0))
        else:
            rtol, atol = adaptive
            at = np.ascontiguousarray(np.broadcast_to(atol, (5,)), dtype=np.float64)
            self._check(self._L.emri_plan_set_integrator(self._h, 1, float(rtol), at.ctypes.data_as(C.c_void_p), int(max_steps)))

    def orbit_steps(self, k, branch=0, max_out=8192):
        """accepted steps of walker k's adaptive orbit -> dict(t, h, y[n][5], stop)"""
        t, h, y = np.zeros(max_out), np.zeros(max_out), np.zeros((max_out, 5))
        info = np.zeros(2, dtype=np.int32)
        self._check(self._L.emri_plan_orbit_steps(self._h, int(k), int(branch), max_out, t.ctypes.data_as(C.c_void_p),
                                                   h.ctypes.data_as(C.c_void_p), y.ctypes.data_as(C.c_void_p),
                                                   info.ctypes.data_as(C.c_void_p)))
        n = min(int(info[0]), max_out)
        return dict(t=t[:n], h=h[:n], y=y[:n], stop=int(info[1]), n=int(info[0]))

    def orbit_report(self, K):
        """modes of the last parallel-in-time orbit: 1 verified, 2 sequential tail, 3 zero rows"""
        m = np.zeros(K, dtype=np.int32)
        self._check(self._L.emri_plan_orbit_report(self._h, K, m.ctypes.data_as(C.c_void_p)))
        return m

    def synth_report(self):
        """path counters of stage (b) over the last call: dict(units, by_order[1..8], base_units, cbrt_samples, skipped_units)"""
        c = np.zeros(16, dtype=np.int64)
        self._check(self._L.emri_plan_synth_report(self._h, c.ctypes.data_as(C.c_void_p)))
        return dict(units=int(c[0]), by_order={m: int(c[m]) for m in range(1, 9)}, base_units=int(c[9]),
                    cbrt_samples=int(c[10]), skipped_units=int(c[11]), harmonics_evaluated=int(c[12]),
                    harmonics_first_range=int(c[13]), second_range_orders=int(c[14]))

    def set_synth_debug(self, force_base=False, force_cbrt=False):
        """test hook: force the data-selected slow paths of stage (b)"""
        self._check(self._L.emri_plan_set_synth_debug(self._h, (1 if force_base else 0) | (2 if force_cbrt else 0)))

    def set_unit_tiles(self, tiles):
        """test hook: tiles of 256 samples per synthesis unit (0 = chosen per call)"""
        self._check(self._L.emri_plan_set_unit_tiles(self._h, int(tiles)))

    def set_chunk(self, c):
        self._check(self._L.emri_plan_set_chunk(self._h, c))

    def num_nodes(self):
        return int(self._L.emri_plan_num_nodes(self._h))

    def launch_count(self):
        """kernels of this library enqueued by the last hot call"""
        return int(self._L.emri_plan_last_launch_count(self._h))

    def set_graphs(self, on):
        """True (default): emri_loglike replays a captured CUDA graph per argument set"""
        self._check(self._L.emri_plan_set_graphs(self._h, 1 if on else 0))

    def graph_stats(self):
        """(graphs captured, calls served by a replay)"""
        c = np.zeros(2, dtype=np.int64)
        self._check(self._L.emri_plan_graph_stats(self._h, c.ctypes.data_as(C.c_void_p)))
        return int(c[0]), int(c[1])

    def set_series_tolerance(self, tol):
        """relative truncation of the harmonic series of stage (b) (default 1e-14)"""
        self._check(self._L.emri_plan_set_series_tolerance(self._h, float(tol)))

    def set_transform(self, fused):
        """True (default where available): both transform passes and Eq. 8 in one kernel of the library; False: full cuFFT
        transform + streaming reduction kernel"""
        self._check(self._L.emri_plan_set_transform(self._h, 1 if fused else 0))

    def transform_is_fused(self):
        return bool(self._L.emri_plan_transform_is_fused(self._h))

    def like_kernel_name(self):
        return "fft2_like_kernel" if self.transform_is_fused() else "loglike_kernel"

    def workspace_bytes(self):
        return int(self._L.emri_plan_workspace_bytes(self._h))

    def enable_timings(self, on=True):
        self._check(self._L.emri_plan_enable_timings(self._h, 1 if on else 0))

    def timings(self):
        ms = (C.c_double * 4)()
        self._check(self._L.emri_plan_get_timings(self._h, ms))
        return dict(orbit=ms[0], synth=ms[1], fft=ms[2], like=ms[3])

    # ---- the path (device tensors; results are valid once the current stream has caught up)
    def orbit(self, params, nodes=None, status=None):
        import torch
        K = params.shape[0]
        if nodes is None:
            nodes = torch.empty((K, self.num_nodes(), NODE_STRIDE), dtype=torch.float64, device=params.device)
        self._check(self._L.emri_orbit(self._h, _ptr(params, torch.float64, (K, NPAR)), K,
                                       _ptr(nodes, torch.float64, (K, self.num_nodes(), NODE_STRIDE)),
                                       _ptr(status, torch.int32, (K,)), _stream()))
        return nodes

    def waveform(self, params, h_I=None, h_II=None, status=None):
        import torch
        K = params.shape[0]
        if h_I is None:
            h_I = torch.empty((K, self.N), dtype=torch.float64, device=params.device)
        if h_II is None:
            h_II = torch.empty((K, self.N), dtype=torch.float64, device=params.device)
        self._check(self._L.emri_waveform(self._h, _ptr(params, torch.float64, (K, NPAR)), K,
                                          _ptr(h_I, torch.float64, (K, self.N)), _ptr(h_II, torch.float64, (K, self.N)),
                                          _ptr(status, torch.int32, (K,)), _stream()))
        return h_I, h_II

    def waveform_fft(self, params, spectra=None, status=None):
        import torch
        K = params.shape[0]
        if spectra is None:
            spectra = torch.empty((K, 2, self.Nf), dtype=torch.complex128, device=params.device)
        self._check(self._L.emri_waveform_fft(self._h, _ptr(params, torch.float64, (K, NPAR)), K,
                                              _ptr(spectra, torch.complex128, (K, 2, self.Nf)),
                                              _ptr(status, torch.int32, (K,)), _stream()))
        return spectra

    def data_fft(self, d_I, d_II, out=None):
        import torch
        if out is None:
            out = torch.empty((2, self.Nf), dtype=torch.complex128, device=d_I.device)
        self._check(self._L.emri_data_fft(self._h, _ptr(d_I, torch.float64, (self.N,)),
                                          _ptr(d_II, torch.float64, (self.N,)),
                                          _ptr(out, torch.complex128, (2, self.Nf)), _stream()))
        return out

    def loglike(self, params, data_fft, logL=None, status=None):
        import torch
        K = params.shape[0]
        if logL is None:
            logL = torch.empty((K,), dtype=torch.float64, device=params.device)
        self._check(self._L.emri_loglike(self._h, _ptr(params, torch.float64, (K, NPAR)), K,
                                         _ptr(data_fft, torch.complex128, (2, self.Nf)),
                                         _ptr(logL, torch.float64, (K,)), _ptr(status, torch.int32, (K,)), _stream()))
        return logL

    def loglike_fdep(self, params, fcoef, f_star, data_fft, logL=None, status=None):
        """Eq. 8 with the frequency-dependent propagation factor of Eq. 7; fcoef: CUDA [K][6]"""
        import torch
        K = params.shape[0]
        if logL is None:
            logL = torch.empty((K,), dtype=torch.float64, device=params.device)
        self._check(self._L.emri_loglike_fdep(self._h, _ptr(params, torch.float64, (K, NPAR)), K,
                                              _ptr(fcoef, torch.float64, (K, 6)), float(f_star),
                                              _ptr(data_fft, torch.complex128, (2, self.Nf)),
                                              _ptr(logL, torch.float64, (K,)), _ptr(status, torch.int32, (K,)), _stream()))
        return logL

    def loglike_host(self, params, data_fft=None, logL=None, status=None):
        """HOST numpy arrays in and out (pinned or pageable); synchronises.  data_fft=None reuses the
        spectrum uploaded by the previous call."""
        params = np.ascontiguousarray(params, dtype=np.float64)
        K = params.shape[0]
        if data_fft is not None:
            data_fft = np.ascontiguousarray(data_fft, dtype=np.complex128)
            if data_fft.shape != (2, self.Nf):
                raise ValueError("data_fft must be complex [2][N/2+1]")
        logL = np.empty(K) if logL is None else logL
        self._check(self._L.emri_loglike_host(
            self._h, params.ctypes.data_as(C.c_void_p), K,
            data_fft.ctypes.data_as(C.c_void_p) if data_fft is not None else None,
            logL.ctypes.data_as(C.c_void_p),
            status.ctypes.data_as(C.c_void_p) if status is not None else None, _stream()))
        return logL

    def loglike_host_ptr(self, params_ptr, K, data_ptr, logL_ptr, status_ptr=None):
        """same, with raw host addresses (pinned torch tensors' data_ptr())"""
        self._check(self._L.emri_loglike_host(
            self._h, C.c_void_p(params_ptr), K, C.c_void_p(data_ptr) if data_ptr else None,
            C.c_void_p(logL_ptr), C.c_void_p(status_ptr) if status_ptr else None, _stream()))

    def stretch_step(self, X, logL, data_fft, lo, hi, a, seed, step, half, accepted=None, log_buf=None):
        import torch
        K = X.shape[0]
        self._check(self._L.emri_stretch_step(
            self._h, _ptr(X, torch.float64, (K, NPAR)), _ptr(logL, torch.float64, (K,)), K,
            _ptr(data_fft, torch.complex128, (2, self.Nf)), _ptr(lo, torch.float64, (NPAR,)),
            _ptr(hi, torch.float64, (NPAR,)), float(a), int(seed), int(step), int(half),
            _ptr(accepted, torch.int32, (K,)), _ptr(log_buf, torch.float64, (K // 2, NPAR + 4)), _stream()))
