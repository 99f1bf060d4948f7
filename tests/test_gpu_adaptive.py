"""Stage (a) with the paper's own kind of integrator on the device (next row f-3, reading D14): Dormand-Prince 5(4) with
per-walker step control and dense output, against the oracle's S3' -- the step sequence itself, the coarse node table, the
waveform and the likelihood; plunge truncation; the LSO convention (backward integration)."""
import numpy as np
import pytest

from paper_2311_17174_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
ATOL = np.array([1e-9, 1e-18, 1e-9, 1e-14, 1e-9])


@pytest.fixture(scope="module")
def emri():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2311_17174_b200 import emri as m
    m.load()
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def circ_diff(a, b):
    d = (a - b) % 1.0
    return d - (d >= 0.5)


def forced_oracle(plan, k, rtol, atol, anchor=False):
    """the oracle re-integrating with the step sizes walker k's device integration took (teacher-forced, D14)"""
    from oracle.oracle import Oracle
    f, b = plan.orbit_steps(k, 0), plan.orbit_steps(k, 1)
    o = Oracle(anchor=anchor)
    o.set_adaptive((rtol, atol), forced_fwd=f["h"], forced_bwd=b["h"])
    return o, f, b


@pytest.mark.parametrize("ci,N,rtol", [(1, 1 << 16, 1e-8), (2, 1 << 20, 1e-11), (3, 1 << 18, 1e-13)])
def test_adaptive_steps_and_nodes_match_oracle(emri, oracle, ci, N, rtol):
    """(A) the controller: at a tolerance where the error estimate is above rounding noise the device takes the oracle's
    steps (same count, same times); at tolerances near rounding two correct implementations choose different steps, so
    only the step count is compared.  (B) teacher-forced: the oracle re-integrates with the DEVICE's step sizes and the
    coarse node table must then agree as tightly as the fixed-step scheme's does."""
    cfg = W.scaled(W.CONFIGS[ci], K=6, N=N)
    P = W.draw_params(cfg)
    atol = ATOL * (rtol / 1e-9)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K)
    plan.set_integrator((rtol, atol))
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    nodes = plan.orbit(dev(P), status=st)
    torch.cuda.synchronize()
    nodes, st = nodes.cpu().numpy(), st.cpu().numpy()
    Nc = -(-N // 256)
    for k in range(cfg.K):
        ref = oracle.dp5_steps(P[k], (Nc + 1) * 256 * cfg.dt, rtol, atol, stop_at_plunge=True)
        ada, got, _ = forced_oracle(plan, k, rtol, atol)
        assert got["stop"] == ref["stop"] == 0
        if rtol >= 1e-9:
            assert got["n"] == len(ref["t"])
            np.testing.assert_allclose(got["t"], ref["t"], rtol=1e-4, atol=1e-9)
            np.testing.assert_allclose(got["t"][:5], ref["t"][:5], rtol=1e-12)          # the first-step rule
        else:
            assert abs(got["n"] - len(ref["t"])) <= 0.25 * len(ref["t"])
        assert got["t"][-1] + got["h"][-1] == (Nc + 1) * 256 * cfg.dt                   # lands on the bound exactly
        # (C) validity: teacher-forcing alone would also pass a controller that accepts steps it should reject, so the
        # oracle judges every step the DEVICE accepted by its own error norm (must be < 1), and the step the device chose
        # next by the rule h min(10, 0.9 norm^-1/5) (smaller after a rejection; the last step is cut to the bound),
        # wherever the norm is above rounding (> 1e-3).  Measured on B200: the rule holds to 4e-8 at rtol 1e-8 and to
        # 7e-4 at rtol 1e-13, where the two norms of one step differ by rounding noise; slack 1e-3 and 1e-2.
        err = oracle.dp5_forced_errors(P[k], rtol, atol, got["h"])
        assert len(err) == got["n"]
        ratio, fac, elig = got["h"][1:-1] / got["h"][:-2], np.minimum(10.0, 0.9 * err[:-2] ** -0.2), err[:-2] > 1e-3
        elig[0] = True                                                                       # (never empty: keeps the prints simple)
        dev_ = np.abs(ratio[elig] / fac[elig] - 1)
        print(f"rtol {rtol} walker {k}: {got['n']} steps, norm max {err.max():.3f}, above 1: {np.sum(err >= 1)}, "
              f"rule: {elig.sum()} eligible, max excess {np.max(ratio[elig] / fac[elig]) - 1:.2e}, median dev {np.median(dev_):.2e}")
        slack = 1e-3 if rtol >= 1e-9 else 1e-2
        assert np.all(err < 1.0)
        assert np.all(ratio[elig] <= fac[elig] * (1 + slack)) and np.mean(dev_ < slack) >= 0.9
        orb = ada.orbit(P[k], N, cfg.dt, 256)
        assert st[k] == orb["status"] == 0 and nodes.shape[1] == orb["Nn"]
        val, slope, inc = nodes[k, :, 0:5].T, nodes[k, :, 5:10].T, nodes[k, :, 10:15].T
        for q in (0, 2, 4):
            assert np.max(np.abs(circ_diff(val[q], orb["val"][q]))) < 2e-11
            np.testing.assert_allclose(inc[q], orb["inc"][q], rtol=1e-12, atol=2e-13)
        for q in (1, 3):
            np.testing.assert_allclose(val[q], orb["val"][q], rtol=2e-14, atol=1e-300)
            np.testing.assert_allclose(inc[q], orb["inc"][q], rtol=1e-9, atol=1e-24)
        np.testing.assert_allclose(slope, orb["slope"], rtol=1e-12, atol=1e-30)
    plan.close()


def test_adaptive_waveform_and_loglike_match_oracle(emri, oracle):
    cfg = W.scaled(W.CONFIGS[2], K=6, N=1 << 16)
    P = W.draw_params(cfg)
    P[4, W.P_NU0] = 0.9997 * oracle.nu_lso(P[4, W.P_M], P[4, W.P_E0])         # plunges inside the window
    P[5, W.P_MU] = -3.0                                                       # invalid
    rtol, atol = 1e-12, ATOL * 1e-3
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    plan.set_integrator((rtol, atol))
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    torch.cuda.synchronize()
    # teacher-forced oracle, walker by walker
    h_ref, st_ref = np.zeros((cfg.K, 2, cfg.N)), np.zeros(cfg.K, dtype=np.int32)
    for k in range(cfg.K):
        ada, f, b = forced_oracle(plan, k, rtol, atol)
        h_ref[k, 0], h_ref[k, 1], st_ref[k] = ada.waveform(P[k], cfg.N, cfg.dt, cfg.n_max)
    D = np.stack([oracle.rfft(h_ref[0, 0]), oracle.rfft(h_ref[0, 1])]) + W.noise_fft(cfg.N, cfg.dt, psd, 21)
    L_ref = np.array([oracle.loglike(np.stack([oracle.rfft(h_ref[k, 0]), oracle.rfft(h_ref[k, 1])]), D, psd, cfg.N, cfg.dt)
                      for k in range(cfg.K)])
    logL = plan.loglike(dev(P), dev(D)).cpu().numpy()
    st = st.cpu().numpy()
    print("status", st, st_ref, "steps", [plan.orbit_steps(k, 0)["n"] for k in range(cfg.K)])
    assert np.array_equal(st, st_ref) and st[4] == 2 and st[5] == 1
    for ch, got in ((0, hI.cpu().numpy()), (1, hII.cpu().numpy())):
        for k in range(5):
            err = np.max(np.abs(got[k] - h_ref[k, ch])) / np.max(np.abs(h_ref[k, ch]))
            assert err <= 1e-9, (k, ch, err)
        assert not got[5].any()
    assert np.any(hI.cpu().numpy()[4] == 0.0) and np.any(hI.cpu().numpy()[4] != 0.0)        # truncated at plunge
    assert logL[5] == -np.inf and np.all(np.abs(logL[:5] - L_ref[:5]) <= 1e-9 * np.abs(L_ref[:5]) + 1e-6)
    # the free-running oracle (its own steps) is the same physics to the accuracy the tolerance buys
    from oracle.oracle import Oracle
    free = Oracle(adaptive=(rtol, atol)).waveform(P[0], cfg.N, cfg.dt, cfg.n_max)[0]
    assert np.max(np.abs(free - h_ref[0, 0])) <= 1e-6 * np.max(np.abs(free))
    # back to the fixed-step scheme on the same plan: the two integrators give the same physics (1e-6 of the amplitude)
    plan.set_integrator(None)
    h4, _ = plan.waveform(dev(P))
    assert np.max(np.abs(h4.cpu().numpy()[0] - h_ref[0, 0])) <= 1e-6 * np.max(np.abs(h_ref[0, 0]))
    plan.close()


def test_adaptive_orbit_from_the_lso_matches_oracle(emri):
    """the paper's own set-up end to end: state given at the LSO, adaptive integrator, backwards"""
    cfg = W.scaled(W.CONFIGS[2], K=5, N=1 << 18)
    P = W.draw_params(cfg)
    P[:, W.P_E0] = np.linspace(0.05, 0.4, cfg.K)
    rtol, atol = 1e-12, ATOL * 1e-3
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    plan.set_anchor(True)
    plan.set_integrator((rtol, atol))
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    nodes = plan.orbit(dev(P), status=st).cpu().numpy()
    st = st.cpu().numpy()
    hI, hII = plan.waveform(dev(P))
    hI = hI.cpu().numpy()
    idx = np.unique(np.concatenate([np.arange(0, 300), np.arange(cfg.N - 400, cfg.N), np.arange(0, cfg.N, 1013)]))
    for k in range(cfg.K):
        ada, f, b = forced_oracle(plan, k, rtol, atol, anchor=True)
        orb = ada.orbit(P[k], cfg.N, cfg.dt, 256)
        assert st[k] == orb["status"] == 0
        np.testing.assert_allclose(nodes[k, :, 1], orb["val"][1], rtol=2e-14)
        np.testing.assert_allclose(nodes[k, :, 3], orb["val"][3], rtol=1e-13)
        for q in (0, 2, 4):
            assert np.max(np.abs(circ_diff(nodes[k, :, q], orb["val"][q]))) < 2e-11
        a, bb, s_ref = ada.waveform(P[k], cfg.N, cfg.dt, cfg.n_max, idx=idx)
        assert s_ref == 0 and np.max(np.abs(hI[k, idx] - a)) <= 1e-9 * np.max(np.abs(hI[k]))
        assert b["n"] > 10 and b["h"][0] < 0 and b["stop"] == 0 and f["n"] >= 1         # the long branch runs backwards
    plan.close()


def test_reports_refuse_leftovers_of_another_integrator(emri):
    """emri_plan_orbit_report belongs to the parallel-in-time RK4 schedule and emri_plan_orbit_steps to the adaptive pair:
    each returns EMRI_EINVAL when the plan is configured for the other, or before stage (a) has run in that configuration,
    instead of handing out whatever an earlier call left in the buffers"""
    cfg = W.scaled(W.CONFIGS[0], K=4, N=1 << 14)
    P = dev(W.draw_params(cfg))
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    with pytest.raises(emri.EmriError):
        plan.orbit_report(cfg.K)                        # nothing has run yet
    plan.orbit(P)
    assert set(plan.orbit_report(cfg.K).tolist()) <= {1, 2}
    plan.set_integrator((1e-9, ATOL))
    with pytest.raises(emri.EmriError):
        plan.orbit_report(cfg.K)                        # modes of the RK4 call would be leftovers now
    with pytest.raises(emri.EmriError):
        plan.orbit_steps(0, 0)                          # the adaptive integrator has not run yet
    plan.orbit(P)
    assert plan.orbit_steps(0, 0)["n"] > 0
    with pytest.raises(emri.EmriError):
        plan.orbit_report(cfg.K)
    plan.set_integrator(None)
    with pytest.raises(emri.EmriError):
        plan.orbit_steps(0, 0)
    plan.set_orbit_schedule(0)
    plan.orbit(P)
    with pytest.raises(emri.EmriError):
        plan.orbit_report(cfg.K)                        # the sequential schedule writes no modes
    plan.close()
