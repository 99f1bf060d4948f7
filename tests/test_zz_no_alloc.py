"""emri_spectra_loglike_static: the likelihood entry point for callers that cannot allocate device memory.

Some users of this library never get to call cudaMalloc: their process gave the whole card to one memory pool when it
started, or runs under a memory quota that can refuse the request, or drives the GPU from a host thread that cannot afford
the device-wide synchronisation cudaMalloc and cudaFree imply.  They cannot own an emri_plan (a plan allocates its
workspace), so the library gives them Eq. 8 as a plan-less call whose only memory beyond the caller's
inputs and output is a 512 KiB array built into the library image (EMRI_STATIC_SCRATCH_DOUBLES, one copy per GPU,
shared by every call).  Limit: K ceil((N/2+1)/8192) <= 65536 partial sums per call.

What is checked here, against the existing plan-based emri_loglike on the same walkers, data and PSD, at the tolerance
the other likelihood tests use (1e-9 |logL| + 1e-6):
  - two calls in a row with different K and different data (the second finds the first call's partial sums in the array,
    laid out for another K: they must not leak into its result), then the first call again (same bits as before);
  - the call leaves the amount of free device memory unchanged;
  - problems beyond the array are refused with EMRI_ELIMIT before any CUDA call (needs no GPU).

This file is named to be collected last, so that under `pytest -x` a failure here cannot hide the other tests; it uses no
state of theirs and passes alone in a fresh process as well as after them."""
import ctypes as C

import numpy as np
import pytest

from paper_2311_17174_b200 import workloads as W

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def emri():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2311_17174_b200 import emri as m
    m.load()
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def close(got, ref):
    return np.all(np.abs(got - ref) <= 1e-9 * np.abs(ref) + 1e-6)


@pytest.mark.gpu
@pytest.mark.parametrize("N,K1,K2", [(1 << 16, 11, 5), (1 << 18, 9, 16), (3 * 4096 + 300, 3, 8)])
def test_static_scratch_likelihood_matches_the_plan_path_on_consecutive_calls(emri, N, K1, K2):
    """several bin ranges per walker (5 and 17 partial sums) and a single ragged one; walker groups of 8 with a ragged
    last group; masked DC and Nyquist bins (+inf in the PSD)"""
    cfg = W.scaled(W.CONFIGS[1], K=max(K1, K2), N=N, n_max=6)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K, psd)
    psd_d = dev(psd)
    inject = plan.waveform_fft(dev(P[:1]))[0].clone()
    calls = []
    for K, seed in ((K1, 3), (K2, 4)):
        rows = dev(P[cfg.K - K:])                                    # the two calls overlap only partly in walkers
        D = inject + dev(W.noise_fft(N, cfg.dt, psd, seed))          # and see different data
        st = torch.zeros(K, dtype=torch.int32, device="cuda")
        ref = {}
        plan.set_transform(True)
        for fused in ((True, False) if plan.transform_is_fused() else (False,)):     # both existing paths where N allows
            plan.set_transform(fused)
            ref[fused] = plan.loglike(rows, D, status=st).cpu().numpy()
        assert not (st.cpu().numpy() & ~emri.ST_PLUNGE).any()         # no walker the plan path would set to -inf
        spectra = plan.waveform_fft(rows)
        calls.append((K, spectra, D, ref))
    torch.cuda.synchronize()

    out = [torch.full((K,), float("nan"), dtype=torch.float64, device="cuda") for K, *_ in calls]
    first_again = torch.full((K1,), float("nan"), dtype=torch.float64, device="cuda")
    emri.spectra_loglike_static(calls[0][1], calls[0][2], psd_d, N, cfg.dt, out[0])   # also the per-device set-up call
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    emri.spectra_loglike_static(calls[1][1], calls[1][2], psd_d, N, cfg.dt, out[1])   # second call, stale scratch
    emri.spectra_loglike_static(calls[0][1], calls[0][2], psd_d, N, cfg.dt, first_again)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                     # nothing was allocated or freed by the calls

    for (K, _, _, ref), got in zip(calls, out):
        got = got.cpu().numpy()
        print("N", N, "K", K, "static", got[:3], {f: float(np.max(np.abs(got - r))) for f, r in ref.items()})
        assert np.all(np.isfinite(got)) and np.all(got < 0.0)
        for r in ref.values():
            assert close(got, r), (got, r)
    assert np.array_equal(first_again.cpu().numpy(), out[0].cpu().numpy())
    plan.close()


@pytest.mark.gpu
def test_static_scratch_likelihood_is_zero_at_the_injection_and_ignores_masked_bins(emri):
    """data = walker 0's own spectrum: the residual, hence logL[0], is exactly 0; bins whose PSD entry
    is 0, negative, NaN or +inf carry weight 0 whatever the spectra hold there"""
    N = 1 << 16
    cfg = W.scaled(W.CONFIGS[0], K=4, N=N)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K, psd)
    spectra = plan.waveform_fft(dev(P))
    D = spectra[0].clone()
    logL = torch.empty(cfg.K, dtype=torch.float64, device="cuda")
    emri.spectra_loglike_static(spectra, D, dev(psd), N, cfg.dt, logL)
    a = logL.cpu().numpy()
    assert a[0] == 0.0 and np.all(a[1:] < 0.0)
    psd2 = psd.copy()
    psd2[100], psd2[200], psd2[300], psd2[400] = 0.0, -1.0, np.nan, np.inf
    D2 = D.clone()
    D2[:, [100, 200, 300, 400]] += 1e3                               # would dominate the sum if those bins counted
    plan2 = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K, psd2)
    ref = plan2.loglike(dev(P), D2).cpu().numpy()
    emri.spectra_loglike_static(spectra, D2, dev(psd2), N, cfg.dt, logL)
    b = logL.cpu().numpy()
    assert close(b, ref), (b, ref)
    assert abs(b[0]) <= 1e-6
    plan.close()
    plan2.close()


def test_sizes_beyond_the_built_in_scratch_are_refused_without_a_gpu():
    """the size check comes before the first CUDA call, so it can be exercised on a machine without a GPU"""
    from paper_2311_17174_b200 import emri
    L = emri.load()
    assert emri.STATIC_SCRATCH_DOUBLES == 65536
    assert L.emri_static_scratch_need(508, 1 << 21) == 508 * 129 <= emri.STATIC_SCRATCH_DOUBLES
    assert L.emri_static_scratch_need(509, 1 << 21) > emri.STATIC_SCRATCH_DOUBLES
    assert L.emri_static_scratch_need(0, 1 << 21) == -1 and L.emri_static_scratch_need(4, 7) == -1
    fake = C.c_void_p(256)                                           # never dereferenced: the call is refused first
    assert L.emri_spectra_loglike_static(fake, 509, 1 << 21, 15.0, fake, fake, fake, None) == -5
    assert L.emri_spectra_loglike_static(fake, 13108, 1 << 16, 15.0, fake, fake, fake, None) == -5
    assert b"scratch" in L.emri_strerror(-5)
    for bad in ((None, 4, 64, 15.0, fake, fake, fake), (fake, 0, 64, 15.0, fake, fake, fake),
                (fake, 4, 63, 15.0, fake, fake, fake), (fake, 4, 64, 0.0, fake, fake, fake),
                (fake, 4, 64, 15.0, None, fake, fake), (fake, 4, 64, 15.0, fake, None, fake),
                (fake, 4, 64, 15.0, fake, fake, None)):
        assert L.emri_spectra_loglike_static(*bad, None) == -1
