"""The data-selected paths of stage (b) and the boundary's corner cases that no seeded config is known to reach:
forced base-series fallback and cube-root amplitude (emri_plan_set_synth_debug) checked element-wise against the oracle
with the path counters (emri_plan_synth_report) asserted non-zero; a natural input that takes both; degenerate geometry
(reading R16); the stretch move on a plan with K_max = K/2; small strides at full length; no allocation in the hot call."""
import numpy as np
import pytest

from paper_2311_17174_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
H_TOL = 1e-9


@pytest.fixture(scope="module")
def emri():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2311_17174_b200 import emri as m
    m.load()
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def h_err(got, ref):
    return np.max(np.abs(got - ref), axis=-1) / np.max(np.abs(ref), axis=-1)


@pytest.mark.parametrize("force_base,force_cbrt", [(True, False), (False, True), (True, True)])
def test_forced_slow_paths_match_oracle(emri, oracle, force_base, force_cbrt):
    """every unit on the base series in e^2 and / or every sample on the cube-root amplitude: same waveform"""
    cfg = W.scaled(W.CONFIGS[3], K=6, N=3 * 4096 + 300)          # several units and a ragged tail, n_max = 30
    P = W.draw_params(cfg)
    P[:, W.P_E0] = np.linspace(0.05, 0.5, cfg.K)
    for k in range(cfg.K):
        P[k, W.P_NU0] = W.nu0_for_plunge_after(P[k, W.P_M], P[k, W.P_MU], P[k, W.P_E0], 1000.0 * cfg.T_obs)
    h_ref, st_ref = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    assert not st_ref.any()
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    hI0, hII0 = plan.waveform(dev(P))
    rep0 = plan.synth_report()
    plan.set_synth_debug(force_base=force_base, force_cbrt=force_cbrt)
    hI, hII = plan.waveform(dev(P))
    rep = plan.synth_report()
    torch.cuda.synchronize()
    print("default paths", rep0, "forced", rep)
    assert rep0["base_units"] == 0 and rep0["cbrt_samples"] == 0          # the defaults take neither here
    if force_base:
        assert rep["base_units"] == rep["units"] > 0 and sum(rep["by_order"].values()) == 0
    if force_cbrt:
        assert rep["cbrt_samples"] == cfg.K * cfg.N
    for got, got0, ch in ((hI, hI0, 0), (hII, hII0, 1)):
        e = h_err(got.cpu().numpy(), h_ref[:, ch])
        assert np.all(e <= H_TOL), e
        assert np.all(h_err(got.cpu().numpy(), got0.cpu().numpy()) <= 1e-11)    # and the fast paths agree with them
    plan.close()


def test_natural_input_reaches_both_slow_paths(emri, oracle):
    """a stride of 4096 samples makes nu move by more than 4e-3 of the node value inside an interval (cube-root branch),
    and e = 0.6 chirping hard over 16-tile units makes order 8 of the local series significant (base-series fallback):
    the counters prove the paths ran, the oracle (same stride) that they are right"""
    N, S = 1 << 15, 4096
    cfg = W.scaled(W.CONFIGS[3], K=4, N=N, n_max=30)
    P = W.draw_params(cfg)
    P[:, W.P_M], P[:, W.P_MU], P[:, W.P_E0] = 2e5, 50.0, np.array([0.6, 0.55, 0.5, 0.3])
    for k in range(cfg.K):        # two days from plunge by the closed-form estimate
        P[k, W.P_NU0] = W.nu0_for_plunge_after(P[k, W.P_M], P[k, W.P_MU], P[k, W.P_E0], 2.5 * N * cfg.dt)
    h_ref, st_ref = oracle.waveform_batch(P, N, cfg.dt, cfg.n_max, S=S)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K)
    plan.set_unit_tiles(16)
    plan.set_coarse_stride(S)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    rep = plan.synth_report()
    torch.cuda.synchronize()
    print("paths", rep, "status", st.cpu().numpy(), st_ref)
    assert np.array_equal(st.cpu().numpy(), st_ref)
    assert rep["cbrt_samples"] > 0 and rep["base_units"] > 0
    live = np.max(np.abs(h_ref[:, 0]), axis=1) > 0
    assert live.any()
    for got, ch in ((hI, 0), (hII, 1)):
        g = got.cpu().numpy()
        assert np.all(h_err(g[live], h_ref[live, ch]) <= H_TOL)
    plan.close()


def test_degenerate_geometry_is_finite(emri, oracle):
    """reading R16: lambda = 0 (beta's atan2 arguments vanish identically: beta = 0) and theta_K = 0 (the literal
    (S.n cos thK - cos thS)/sin thK is 0/0; the library uses its expanded form) must give finite waveforms with status 0.
    The oracle's literal formulas are NaN exactly there, so: theta_K = 0 is compared with the oracle at theta_K = 1e-7
    (continuous), and lambda = 0 by what beta = 0 implies: L^ = S^ does not precess, so alpha0 must not matter."""
    cfg = W.scaled(W.CONFIGS[1], K=4, N=1 << 12)
    P = W.draw_params(cfg)
    P[1] = P[0]; P[1, W.P_LAM] = 0.0
    P[2] = P[1]; P[2, W.P_ALP0] += 1.234
    P[3] = P[0]; P[3, W.P_THK] = 0.0
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    D = plan.data_fft(hI[0].contiguous(), hII[0].contiguous())
    logL = plan.loglike(dev(P), D).cpu().numpy()
    hI, hII = hI.cpu().numpy(), hII.cpu().numpy()
    assert not st.cpu().numpy().any()
    assert np.all(np.isfinite(hI)) and np.all(np.isfinite(hII)) and np.all(np.isfinite(logL))
    assert np.max(np.abs(hI[1])) > 0 and np.max(np.abs(hI[3])) > 0
    assert np.max(np.abs(hI[1] - hI[2])) <= 1e-11 * np.max(np.abs(hI[1]))
    assert np.max(np.abs(hII[1] - hII[2])) <= 1e-11 * np.max(np.abs(hII[1]))
    q = P[3].copy(); q[W.P_THK] = 1e-7
    a, b, s3 = oracle.waveform(q, cfg.N, cfg.dt, cfg.n_max)
    assert s3 == 0
    assert np.max(np.abs(hI[3] - a)) <= 1e-5 * np.max(np.abs(a)) and np.max(np.abs(hII[3] - b)) <= 1e-5 * np.max(np.abs(b))
    plan.close()


def test_stretch_step_on_a_plan_of_half_the_ensemble(emri):
    """include/emri.h: K/2 <= K_max.  A plan created for K/2 walkers must give the same chain as one created for K"""
    cfg = W.scaled(W.CONFIGS[4], K=16, N=1 << 12, n_max=5)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    lo, hi = (dev(v) for v in W.prior_box(cfg))
    out = []
    for K_max in (cfg.K, cfg.K // 2):
        plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, K_max, psd)
        D = plan.waveform_fft(dev(P[:1]))[0].clone()
        X = dev(P)
        logL = torch.empty(cfg.K, dtype=torch.float64, device="cuda")
        for h in (0, 1):      # logL of the start ensemble, half by half (K > K_max for the small plan)
            sl = slice(h * cfg.K // 2, (h + 1) * cfg.K // 2)
            logL[sl] = plan.loglike(X[sl].contiguous(), D)
        acc = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
        for step in range(3):
            for half in (0, 1):
                plan.stretch_step(X, logL, D, lo, hi, 2.0, 99, step, half, accepted=acc)
        torch.cuda.synchronize()
        out.append((X.cpu().numpy(), logL.cpu().numpy()))
        plan.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert not np.array_equal(out[0][0], P)            # something was accepted


def test_small_stride_at_full_length(emri):
    """N = 2^21 with S = 16: 513 shooting segments (49 KB of shared memory in orbit_correct_kernel, above the default
    limit) -- both schedules run and agree"""
    cfg = W.scaled(W.CONFIGS[2], K=2, N=1 << 21)
    P = dev(W.draw_params(cfg))
    res = []
    for schedule in (1, 0):
        plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
        plan.set_coarse_stride(16)
        plan.set_orbit_schedule(schedule)
        st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
        nodes = plan.orbit(P, status=st)
        torch.cuda.synchronize()
        assert not st.cpu().numpy().any()
        res.append(nodes.cpu().numpy())
        plan.close()
    np.testing.assert_allclose(res[0][:, :, 1], res[1][:, :, 1], rtol=1e-14)      # nu
    np.testing.assert_allclose(res[0][:, :, 3], res[1][:, :, 3], rtol=1e-13, atol=1e-18)      # e
    d = (res[0][:, :, 0] - res[1][:, :, 0]) % 1.0
    assert np.max(np.minimum(d, 1.0 - d)) < 1e-10


def test_hot_call_does_not_allocate(emri):
    """include/emri.h: calls only enqueue.  After plan creation neither device memory nor the plan's workspace moves
    across emri_loglike calls -- full ensemble, a ragged one (its cuFFT plan object is built on first use, inside the
    work area that already exists) and a single walker"""
    cfg = W.scaled(W.CONFIGS[1], K=40, N=1 << 14)
    P = dev(W.draw_params(cfg))
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    plan.set_chunk(16)                                   # chunks of 16: 40 = 16 + 16 + 8
    D = plan.waveform_fft(P[:1].contiguous())[0].clone()
    logL = torch.empty(cfg.K, dtype=torch.float64, device="cuda")
    plan.loglike(P, D, logL)                             # warm-up: every kernel's module is loaded
    torch.cuda.synchronize()
    free0, ws0 = torch.cuda.mem_get_info()[0], plan.workspace_bytes()
    for K in (cfg.K, 37, 1, cfg.K):
        plan.loglike(P[:K].contiguous() if K < cfg.K else P, D, logL[:K])
    torch.cuda.synchronize()
    assert plan.workspace_bytes() == ws0
    assert torch.cuda.mem_get_info()[0] >= free0 - (2 << 20)      # cuFFT plan objects only (no work area, no buffers)
    plan.close()


@pytest.mark.parametrize("lgN,K,chunk", [(16, 5, 4), (17, 6, 6), (18, 9, 4), (19, 3, 2), (20, 5, 3), (21, 3, 2), (22, 3, 3)])
def test_fused_transform_and_likelihood_match_the_cufft_path_and_the_oracle(emri, oracle, lgN, K, chunk):
    """stages (c)+(d) fused (both transform passes and Eq. 8 in one kernel of the library) against the full cuFFT transform
    + streaming reduction, for every split N = N1 N2 (N1 = 256 .. 1024, N2 = 256 .. 4096), ragged chunks, noisy data, a
    plunging walker and an invalid one; and against the oracle's whole path at N = 2^16"""
    N = 1 << lgN
    cfg = W.scaled(W.CONFIGS[2], K=K, N=N, n_max=8)
    P = W.draw_params(cfg)
    P[1, W.P_NU0] = 0.9995 * W.nu_lso_hz(P[1, W.P_M], P[1, W.P_E0])      # about to plunge: truncated waveform
    P[2, W.P_DL] = -1.0                                                  # invalid: logL = -inf
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, K, psd)
    plan.set_chunk(chunk)
    assert plan.transform_is_fused()
    D = plan.waveform_fft(dev(P[:1]))[0].clone() + dev(W.noise_fft(N, cfg.dt, psd, 3))
    st = torch.zeros(K, dtype=torch.int32, device="cuda")
    fused = plan.loglike(dev(P), D, status=st).cpu().numpy()
    again = plan.loglike(dev(P), D).cpu().numpy()
    plan.set_chunk(K)
    whole = plan.loglike(dev(P), D).cpu().numpy()
    plan.set_transform(False)
    assert not plan.transform_is_fused()
    plain = plan.loglike(dev(P), D).cpu().numpy()
    st = st.cpu().numpy()
    print("fused", fused, "plain", plain, "status", st)
    assert st[2] == 1 and fused[2] == -np.inf and plain[2] == -np.inf
    ok = np.isfinite(plain)
    assert np.array_equal(fused, again) and np.array_equal(fused[ok], whole[ok])           # reproducible, chunk-invariant
    assert np.all(np.abs(fused[ok] - plain[ok]) <= 1e-9 * np.abs(plain[ok]) + 1e-6)
    # noise-less data = walker 0's own waveform: logL[0] = 0 within the absolute floor of the tolerance
    plan.set_transform(True)
    D0 = plan.waveform_fft(dev(P[:1]))[0].clone()
    z = plan.loglike(dev(P), D0).cpu().numpy()
    hh = 2.0 * np.max(np.abs(z[np.isfinite(z)]))                  # the scale of <h|h>
    assert z[0] <= 0.0 and abs(z[0]) <= 1e-12 * hh                # a sum of squared residuals: no cancellation (D16)
    if lgN == 16:
        ref, _ = oracle.loglike_batch(P, N, cfg.dt, cfg.n_max, D.cpu().numpy(), psd)
        assert np.all(np.abs(fused[ok] - ref[ok]) <= 1e-9 * np.abs(ref[ok]) + 1e-6)
    plan.close()


@pytest.mark.parametrize("lgN", [16, 20])
def test_loud_noise_free_injection_on_the_fused_path(emri, oracle, lgN):
    """the mock data are the noise-less fiducial waveform, so the residual vanishes at the injection.
    A loud source (D_L = 0.01 Gpc: <h|h> ~ 1e7 and more) is where a likelihood assembled from <d|d> - 2<d|h> + <h|h>
    would lose the north-star tolerance 1e-9 |logL_ref| + 1e-6 at walker 0 (logL_ref = 0); the fused path sums squared
    residuals (reading D16) and must hold it, for the injection and for the walkers away from it, against the oracle"""
    N = 1 << lgN
    cfg = W.scaled(W.CONFIGS[1], K=4, N=N, n_max=10 if lgN == 16 else 6)
    P = W.draw_params(cfg)
    P[:, W.P_DL] = 0.01
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    h_ref, st_ref = oracle.waveform_batch(P[:1], N, cfg.dt, cfg.n_max)
    assert not st_ref.any()
    D = np.stack([oracle.rfft(h_ref[0, 0]), oracle.rfft(h_ref[0, 1])])
    ref, _ = oracle.loglike_batch(P, N, cfg.dt, cfg.n_max, D, psd)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K, psd)
    assert plan.transform_is_fused()
    got = plan.loglike(dev(P), dev(D)).cpu().numpy()
    plan.set_transform(False)
    plain = plan.loglike(dev(P), dev(D)).cpu().numpy()
    print("N", N, "fused", got, "plain", plain, "oracle", ref)
    assert ref[0] == 0.0 and np.min(np.abs(ref[1:])) > 1e6        # loud indeed
    for a in (got, plain):
        assert a[0] <= 0.0 and abs(a[0]) <= 1e-6
        assert np.all(np.abs(a - ref) <= 1e-9 * np.abs(ref) + 1e-6)
    plan.close()


def test_graph_replay_gives_the_same_bits_and_follows_its_inputs(emri):
    """emri_loglike through a captured CUDA graph: same bits as plain enqueueing; a replay reads the CURRENT contents of
    the parameter and data buffers; a new argument set captures a new graph; settings drop the graphs"""
    cfg = W.scaled(W.CONFIGS[1], K=12, N=1 << 16)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    plan.set_chunk(8)
    D = plan.waveform_fft(dev(P[:1]))[0].clone() + dev(W.noise_fft(cfg.N, cfg.dt, psd, 5))
    p_d = dev(P)
    logL = torch.empty(cfg.K, dtype=torch.float64, device="cuda")
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    plan.set_graphs(False)
    ref = plan.loglike(p_d, D, logL, st).cpu().numpy().copy()
    n_plain = plan.launch_count()
    plan.set_graphs(True)
    c0 = plan.graph_stats()
    a = plan.loglike(p_d, D, logL, st).cpu().numpy().copy()          # captures
    b = plan.loglike(p_d, D, logL, st).cpu().numpy().copy()          # replays
    c1 = plan.graph_stats()
    assert np.array_equal(a, ref) and np.array_equal(b, ref)
    assert c1[0] == c0[0] + 1 and c1[1] == c0[1] + 1 and plan.launch_count() == n_plain
    # the graph reads the buffers it was captured with: change their contents, replay, compare with plain enqueueing
    P2 = P[::-1].copy()
    p_d.copy_(dev(P2))
    g = plan.loglike(p_d, D, logL, st).cpu().numpy().copy()
    assert plan.graph_stats()[1] == c1[1] + 1
    plan.set_graphs(False)
    assert np.array_equal(g, plan.loglike(p_d, D, logL, st).cpu().numpy())
    assert np.array_equal(g, ref[::-1])
    # another K, another graph; a setting drops them all
    plan.set_graphs(True)
    plan.loglike(p_d[:5].contiguous(), D)
    plan.loglike(p_d, D, logL, st)
    caps = plan.graph_stats()[0]
    plan.set_chunk(4)
    plan.loglike(p_d, D, logL, st)
    assert plan.graph_stats()[0] == caps + 1
    assert np.array_equal(logL.cpu().numpy(), ref[::-1])
    # with the data in the default stream's order: a legacy-stream caller and a side stream give the same result
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        out = plan.loglike(p_d, D).cpu().numpy()
    assert np.array_equal(out, ref[::-1])
    plan.close()


def test_second_noise_model_matches_oracle(emri, oracle):
    """the paper's second noise curve (refs [51, 52]: Robson-Cornish-Liu with the galactic confusion fit,
    a PSD with a sharp knee and 1e10 of dynamic range) through Eq. 8, both transform paths, against the oracle's whole path"""
    cfg = W.scaled(W.CONFIGS[1], K=6, N=1 << 16)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_robson(cfg.N, cfg.dt)
    assert np.all(psd[1:-1] > 0) and np.isinf(psd[0]) and np.isinf(psd[-1])
    h_ref, _ = oracle.waveform_batch(P[:1], cfg.N, cfg.dt, cfg.n_max)
    D = np.stack([oracle.rfft(h_ref[0, 0]), oracle.rfft(h_ref[0, 1])]) + W.noise_fft(cfg.N, cfg.dt, psd, 11)
    ref, st_ref = oracle.loglike_batch(P, cfg.N, cfg.dt, cfg.n_max, D, psd)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    for fused in (True, False):
        plan.set_transform(fused)
        got = plan.loglike(dev(P), dev(D)).cpu().numpy()
        print("Robson PSD, fused" if fused else "Robson PSD, plain", np.abs(got - ref) / np.abs(ref))
        assert np.all(np.abs(got - ref) <= 1e-9 * np.abs(ref) + 1e-6)
    # and it is a different likelihood from the Barack-Cutler one
    plan_bc = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, W.lisa_psd_barack_cutler(cfg.N, cfg.dt))
    other = plan_bc.loglike(dev(P), dev(D)).cpu().numpy()
    assert np.all(np.abs(other - ref) > 1e-3 * np.abs(ref))
    plan.close(); plan_bc.close()


def test_series_tolerance_bounds_the_truncation(emri, oracle):
    """emri_plan_set_series_tolerance: the error of the truncated harmonic series stays below ~n_max tol of max |h|
    (readings D8, D13), the default (1e-14) is indistinguishable from 1e-16 against the oracle, fewer orders and overtones are evaluated as tol grows, and even
    the loosest setting accepted is inside the parity tolerance"""
    cfg = W.scaled(W.CONFIGS[3], K=6, N=5 * 4096 + 78)
    P = W.draw_params(cfg)
    P[:, W.P_E0] = np.linspace(0.1, 0.5, cfg.K)
    for k in range(cfg.K):
        P[k, W.P_NU0] = W.nu0_for_plunge_after(P[k, W.P_M], P[k, W.P_MU], P[k, W.P_E0], 1000.0 * cfg.T_obs)
    h_ref, st_ref = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    assert not st_ref.any()
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    hI_def, hII_def = (t.clone() for t in plan.waveform(dev(P)))          # the default is 1e-14
    plan.set_series_tolerance(1e-14)
    hI_14, hII_14 = plan.waveform(dev(P))
    assert torch.equal(hI_def, hI_14) and torch.equal(hII_def, hII_14)
    work, errs = [], []
    for tol in (1e-16, 1e-14, 1e-10):
        plan.set_series_tolerance(tol)
        hI, hII = plan.waveform(dev(P))
        rep = plan.synth_report()
        e = max(h_err(hI.cpu().numpy(), h_ref[:, 0]).max(), h_err(hII.cpu().numpy(), h_ref[:, 1]).max())
        orders = sum(int(m) * n for m, n in rep["by_order"].items())
        print("tol", tol, "max error / max|h|", e, "harmonics", rep["harmonics_evaluated"], "order sum", orders)
        assert e <= max(2e-12, 2.0 * cfg.n_max * tol) and e <= H_TOL
        work.append((rep["harmonics_evaluated"], orders))
        errs.append(e)
    assert errs[1] <= 1.5 * errs[0] + 1e-14           # default vs the tightest setting: the same error against the oracle
    assert work[2][0] < work[0][0] and work[2][1] < work[0][1]
    for bad in (0.0, 1e-18, 1e-9, float("nan")):
        with pytest.raises(Exception):
            plan.set_series_tolerance(bad)
    plan.close()
