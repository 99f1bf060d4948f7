"""GPU-vs-oracle parity, stage by stage, through the C ABI (run on the B200 box: pytest -m gpu).

Tolerances are BASELINE.json's north_star: |h_gpu - h_ref| <= 1e-9 max|h_ref| per channel and
|dlogL| <= 1e-9 |logL_ref| + 1e-6.  Sizes here span several 256-sample tiles, several coarse
intervals and ragged tails, and the oracle finishes them in seconds; the full-size configs are in
test_gpu_configs.py.
"""
import numpy as np
import pytest

from paper_2311_17174_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

H_TOL = 1e-9


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


@pytest.fixture(scope="module")
def emri():
    _need_gpu()
    from paper_2311_17174_b200 import emri as m
    m.load()
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def circ_diff(a, b):
    d = (a - b) % 1.0
    return d - (d >= 0.5)


def h_err(got, ref):
    """max |got-ref| / max|ref| per row"""
    scale = np.max(np.abs(ref), axis=-1)
    scale = np.where(scale > 0, scale, 1.0)
    return np.max(np.abs(got - ref), axis=-1) / scale


def small_cfg(i, K, N, n_max=None):
    return W.scaled(W.CONFIGS[i], K=K, N=N, n_max=n_max)


# ------------------------------------------------------------------ stage (a): orbit nodes
@pytest.mark.parametrize("ci,S", [(0, 256), (1, 256), (2, 64), (3, 256)])
def test_orbit_nodes_match_oracle(emri, oracle, ci, S):
    cfg = small_cfg(ci, K=6, N=1 << 16)
    P = W.draw_params(cfg)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    plan.set_coarse_stride(S)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    nodes = plan.orbit(dev(P), status=st)
    torch.cuda.synchronize()
    nodes, st = nodes.cpu().numpy(), st.cpu().numpy()
    for k in range(cfg.K):
        ref = oracle.orbit(P[k], cfg.N, cfg.dt, S)
        assert nodes.shape[1] == ref["Nn"] and st[k] == ref["status"] == 0
        val, slope, inc = nodes[k, :, 0:5].T, nodes[k, :, 5:10].T, nodes[k, :, 10:15].T
        for q in (0, 2, 4):     # phases, cycles
            assert np.max(np.abs(circ_diff(val[q], ref["val"][q]))) < 2e-11
            np.testing.assert_allclose(inc[q], ref["inc"][q], rtol=1e-13, atol=1e-15)
        for q in (1, 3):        # nu, e
            np.testing.assert_allclose(val[q], ref["val"][q], rtol=2e-14)
            np.testing.assert_allclose(inc[q], ref["inc"][q], rtol=1e-11, atol=1e-25)
        np.testing.assert_allclose(slope, ref["slope"], rtol=1e-12, atol=1e-30)
    plan.close()


# ------------------------------------------------------------------ stage (b): waveform
@pytest.mark.parametrize("ci,K,N", [(0, 8, 1 << 14), (1, 6, 5000), (2, 6, 1 << 13), (3, 8, 3 * 1024 + 2)])
def test_waveform_matches_oracle(emri, oracle, ci, K, N):
    cfg = small_cfg(ci, K=K, N=N)
    P = W.draw_params(cfg)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    st = torch.zeros(K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    torch.cuda.synchronize()
    h_ref, st_ref = oracle.waveform_batch(P, N, cfg.dt, cfg.n_max)
    assert np.array_equal(st.cpu().numpy(), st_ref) and not st_ref.any()
    eI, eII = h_err(hI.cpu().numpy(), h_ref[:, 0]), h_err(hII.cpu().numpy(), h_ref[:, 1])
    print(f"cfg{ci} max rel err h_I {eI.max():.2e} h_II {eII.max():.2e}")
    assert np.all(eI <= H_TOL) and np.all(eII <= H_TOL)
    plan.close()


def test_waveform_with_late_time_and_high_harmonics(emri, oracle):
    """a full-year orbit is integrated (N = 2^21) but only sampled outputs are compared: the last
    tiles carry the accumulated phase error of 8192 RK4 steps"""
    cfg = W.CONFIGS[2]
    P = W.draw_params(cfg, K=3)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, 3)
    hI, hII = plan.waveform(dev(P))
    torch.cuda.synchronize()
    rng = np.random.default_rng(5)
    idx = np.unique(np.concatenate([np.arange(0, 300), np.arange(cfg.N - 600, cfg.N), rng.integers(0, cfg.N, 1500)]))
    hI, hII = hI.cpu().numpy(), hII.cpu().numpy()
    for k in range(3):
        a, b, st = oracle.waveform(P[k], cfg.N, cfg.dt, cfg.n_max, idx=idx)
        sI, sII = np.max(np.abs(hI[k])), np.max(np.abs(hII[k]))
        eI, eII = np.max(np.abs(hI[k, idx] - a)) / sI, np.max(np.abs(hII[k, idx] - b)) / sII
        print(f"walker {k}: {eI:.2e} {eII:.2e}")
        assert st == 0 and eI <= H_TOL and eII <= H_TOL
    plan.close()


# ------------------------------------------------------------------ stage (c): spectrum
def test_spectrum_matches_oracle(emri, oracle):
    cfg = small_cfg(1, K=3, N=1 << 13)
    P = W.draw_params(cfg)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    sp = plan.waveform_fft(dev(P))
    torch.cuda.synchronize()
    sp = sp.cpu().numpy()
    h_ref, _ = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    for k in range(cfg.K):
        for c in range(2):
            H = oracle.rfft(h_ref[k, c])
            assert np.max(np.abs(sp[k, c] - H)) <= 1e-9 * np.max(np.abs(H))
    # emri_data_fft of the GPU's own time series gives the same spectrum
    hI, hII = plan.waveform(dev(P))
    D = plan.data_fft(hI[0].contiguous(), hII[0].contiguous())
    torch.cuda.synchronize()
    np.testing.assert_allclose(D.cpu().numpy(), sp[0], rtol=0, atol=1e-12 * np.max(np.abs(sp[0])))
    plan.close()


# ------------------------------------------------------------------ stage (d) and the whole path
@pytest.mark.parametrize("ci,K,N,noise", [(0, 8, 1 << 13, 0), (1, 6, 1 << 14, 1001), (2, 6, 1 << 13, 0), (3, 7, 1 << 12, 1003)])
def test_loglike_matches_oracle(emri, oracle, ci, K, N, noise):
    cfg = small_cfg(ci, K=K, N=N)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    # data from the ORACLE's injection (walker 0) + the generator's noise; the same array goes to both sides
    hI, hII, _ = oracle.waveform(P[0], N, cfg.dt, cfg.n_max)
    D = np.stack([oracle.rfft(hI), oracle.rfft(hII)])
    if noise:
        D = D + W.noise_fft(N, cfg.dt, psd, noise)
    ref, st_ref = oracle.loglike_batch(P, N, cfg.dt, cfg.n_max, D, psd)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, K, psd)
    st = torch.zeros(K, dtype=torch.int32, device="cuda")
    got = plan.loglike(dev(P), dev(D), status=st)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    print(f"cfg{ci} logL ref {ref[:4]} max abs diff {np.max(np.abs(got - ref)):.3e}")
    assert np.array_equal(st.cpu().numpy(), st_ref)
    assert np.all(np.abs(got - ref) <= 1e-9 * np.abs(ref) + 1e-6)
    # chunking does not change a bit
    plan.set_chunk(2)
    got2 = plan.loglike(dev(P), dev(D))
    torch.cuda.synchronize()
    assert np.array_equal(got2.cpu().numpy(), got)
    # host entry point
    got3 = plan.loglike_host(P, D)
    assert np.array_equal(got3, got)
    assert np.array_equal(plan.loglike_host(P), got)
    plan.close()


def test_loglike_is_zero_for_own_noiseless_injection(emri):
    """the mock data is the noise-less fiducial waveform => residual 0 at theta_0"""
    cfg = small_cfg(0, K=8, N=1 << 14)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    p_d = dev(P)
    hI, hII = plan.waveform(p_d)
    D = plan.data_fft(hI[0].contiguous(), hII[0].contiguous())
    logL = plan.loglike(p_d, D)
    torch.cuda.synchronize()
    logL = logL.cpu().numpy()
    assert abs(logL[0]) <= 1e-12 and np.all(logL[1:] < -1e-3)
    plan.close()


# ------------------------------------------------------------------ next row f-1: frequency-dependent propagation (Eq. 7)
@pytest.mark.parametrize("ci,K,N", [(2, 11, 1 << 13), (1, 5, 1 << 12)])
def test_loglike_fdep_matches_oracle(emri, oracle, ci, K, N):
    cfg = small_cfg(ci, K=K, N=N)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    rng = np.random.default_rng(77)
    fstar = 0.03                                           # ~ Nyquist (1/30 Hz): x = f/f* <= 1.1
    # friction series of order 0.1, delays of a few sample spacings at f ~ f*
    fc = np.column_stack([rng.uniform(-0.3, 0.3, K), rng.uniform(-0.1, 0.1, K), rng.uniform(-0.03, 0.03, K),
                          rng.uniform(-40, 40, K), rng.uniform(-10, 10, K), rng.uniform(-3, 3, K)])
    fc[1] = 0.0                                            # one walker without the frequency dependence
    hI, hII, _ = oracle.waveform(P[0], N, cfg.dt, cfg.n_max)
    D = np.stack([oracle.rfft(hI), oracle.rfft(hII)]) + W.noise_fft(N, cfg.dt, psd, 31)
    plain, st_ref, sp = oracle.loglike_batch(P, N, cfg.dt, cfg.n_max, D, psd, spectra=True)
    ref = np.array([oracle.loglike_fdep(sp[k], D, psd, N, cfg.dt, fc[k], fstar) for k in range(K)])
    plan = emri.Plan(N, cfg.dt, cfg.n_max, K, psd)
    st = torch.zeros(K, dtype=torch.int32, device="cuda")
    got = plan.loglike_fdep(dev(P), dev(fc), fstar, dev(D), status=st)
    base = plan.loglike(dev(P), dev(D))
    torch.cuda.synchronize()
    got, base = got.cpu().numpy(), base.cpu().numpy()
    print(f"fdep cfg{ci}: ref {ref[:3]} plain {plain[:3]} max abs diff {np.max(np.abs(got - ref)):.3e} "
          f"max diff/tolerance {np.max(np.abs(got - ref) / (1e-9 * np.abs(ref) + 1e-6)):.2e}")
    assert np.array_equal(st.cpu().numpy(), st_ref)
    assert np.all(np.abs(got - ref) <= 1e-9 * np.abs(ref) + 1e-6)
    assert got[1] == base[1]                               # G = 1 exactly when the series vanish
    assert np.all(np.abs(got[[0, 2]] - base[[0, 2]]) > 1e-2)    # and it does act otherwise (logL is noise-dominated)
    plan.set_chunk(4)                                      # chunking picks the right coefficient rows
    got2 = plan.loglike_fdep(dev(P), dev(fc), fstar, dev(D))
    torch.cuda.synchronize()
    assert np.array_equal(got2.cpu().numpy(), got)
    plan.close()
