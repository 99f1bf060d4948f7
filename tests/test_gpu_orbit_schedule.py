"""Stage (a) on the GPU: the parallel-in-time schedule (multiple shooting) must
reproduce the sequential RK4 recursion of S3 -- checked against the library's own sequential schedule
(tight) and against the oracle (the parity gate), including walkers that plunge inside the window."""
import numpy as np
import pytest

from paper_2311_17174_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


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


def run_orbit(emri, P, N, dt, n_max, schedule, S=256):
    K = P.shape[0]
    plan = emri.Plan(N, dt, n_max, K)
    if S != 256:
        plan.set_coarse_stride(S)
    plan.set_orbit_schedule(schedule)
    st = torch.zeros(K, dtype=torch.int32, device="cuda")
    nodes = plan.orbit(dev(P), status=st)
    torch.cuda.synchronize()
    modes = plan.orbit_report(K) if schedule == 1 else None
    out = nodes.cpu().numpy(), st.cpu().numpy(), modes
    plan.close()
    return out


def plunging_params(cfg, K, fracs):
    """config-`cfg` draws whose nu0 is moved up so that the 0PN estimate of the plunge time is
    fracs[k] * T_obs (inside the window for fracs < 1)"""
    P = W.draw_params(cfg, K=K)
    for k in range(K):
        P[k, W.P_NU0] = W.nu0_for_plunge_after(P[k, W.P_M], P[k, W.P_MU], P[k, W.P_E0], fracs[k] * cfg.T_obs)
    return P


@pytest.mark.parametrize("ci,N,S", [(1, 1 << 18, 256), (2, 1 << 20, 256), (3, 1 << 17, 64), (0, 1 << 12, 256)])
def test_shooting_reproduces_the_sequential_recursion(emri, ci, N, S):
    cfg = W.scaled(W.CONFIGS[ci], K=24, N=N)
    P = W.draw_params(cfg)
    n1, s1, modes = run_orbit(emri, P, N, cfg.dt, cfg.n_max, 1, S)
    n0, s0, _ = run_orbit(emri, P, N, cfg.dt, cfg.n_max, 0, S)
    assert np.array_equal(s0, s1) and not s0.any()
    assert np.all(modes == 1), f"shooting did not verify: modes {modes}"
    for q in (0, 2, 4):
        assert np.max(np.abs(circ_diff(n1[:, :, q], n0[:, :, q]))) < 2e-12
        np.testing.assert_allclose(n1[:, :, 10 + q], n0[:, :, 10 + q], rtol=2e-14, atol=1e-16)
    for q in (1, 3):
        np.testing.assert_allclose(n1[:, :, q], n0[:, :, q], rtol=4e-16, atol=1e-300)
        np.testing.assert_allclose(n1[:, :, 10 + q], n0[:, :, 10 + q], rtol=1e-12, atol=1e-30)
    np.testing.assert_allclose(n1[:, :, 5:10], n0[:, :, 5:10], rtol=1e-13, atol=1e-30)


def test_plunging_walkers_match_sequential_and_oracle(emri, oracle):
    cfg = W.scaled(W.CONFIGS[1], K=12, N=1 << 17)
    fracs = np.array([0.05, 0.2, 0.35, 0.5, 0.62, 0.75, 0.85, 0.93, 0.99, 1.05, 1.3, 3.0])
    P = plunging_params(cfg, cfg.K, fracs)
    n1, s1, modes = run_orbit(emri, P, cfg.N, cfg.dt, cfg.n_max, 1)
    n0, s0, _ = run_orbit(emri, P, cfg.N, cfg.dt, cfg.n_max, 0)
    print("status", s1, "modes", modes)
    assert np.array_equal(s0, s1)
    assert (s1 == 2).sum() >= 4 and (s1 == 0).sum() >= 1          # the set exercises both outcomes
    for k in range(cfg.K):
        ref = oracle.orbit(P[k], cfg.N, cfg.dt, 256)
        assert s1[k] == ref["status"]
        # nodes from j_pl on are copies of node j_pl - 1 with zero increments in both schedules
        np.testing.assert_allclose(n1[k, :, 1], n0[k, :, 1], rtol=1e-15)
        np.testing.assert_allclose(n1[k, :, 3], n0[k, :, 3], rtol=1e-15, atol=1e-300)
        np.testing.assert_allclose(n1[k, :, 1], ref["val"][1], rtol=2e-14)
        np.testing.assert_allclose(n1[k, :, 3], ref["val"][3], rtol=2e-14, atol=1e-300)
        for q in (0, 2, 4):
            assert np.max(np.abs(circ_diff(n1[k, :, q], n0[k, :, q]))) < 2e-12
            assert np.max(np.abs(circ_diff(n1[k, :, q], ref["val"][q]))) < 2e-11
            np.testing.assert_allclose(n1[k, :, 10 + q], ref["inc"][q], rtol=1e-13, atol=1e-15)


def test_waveform_of_plunging_walkers_matches_oracle(emri, oracle):
    cfg = W.scaled(W.CONFIGS[1], K=4, N=1 << 14)
    P = plunging_params(cfg, cfg.K, np.array([0.3, 0.6, 0.9, 2.0]))
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    torch.cuda.synchronize()
    h_ref, st_ref = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    assert np.array_equal(st.cpu().numpy(), st_ref) and (st_ref == 2).any()
    for ch, got in ((0, hI.cpu().numpy()), (1, hII.cpu().numpy())):
        err = np.max(np.abs(got - h_ref[:, ch]), axis=1) / np.max(np.abs(h_ref[:, ch]), axis=1)
        assert np.all(err <= 1e-9), err
        # zero after the plunge, as the oracle
        assert np.array_equal(got == 0.0, h_ref[:, ch] == 0.0)
    plan.close()


def test_invalid_and_immediately_plunged_walkers(emri):
    cfg = W.scaled(W.CONFIGS[0], K=4, N=1 << 12)
    P = W.draw_params(cfg)
    P[1, W.P_M] = -1.0                                            # bad parameter
    P[2, W.P_NU0] = 2.0 * W.nu_lso_hz(P[2, W.P_M], P[2, W.P_E0])  # already beyond the LSO
    P[3, W.P_E0] = float("nan")
    for schedule in (0, 1):
        nodes, st, modes = run_orbit(emri, P, cfg.N, cfg.dt, cfg.n_max, schedule)
        assert list(st) == [0, 1, 2, 1]
        assert not nodes[1:].any() and nodes[0].any()


# ------------------------------------------------------------------ next row f-3: the paper's IC convention (anchored at the LSO)
def lso_params(cfg, K, e_hi=0.5):
    P = W.draw_params(cfg, K=K)
    P[:, W.P_E0] = np.linspace(0.0, e_hi, K)          # e at plunge, including the circular case
    return P


@pytest.mark.parametrize("ci,N,S", [(1, 1 << 18, 256), (3, 1 << 16, 64), (2, 1 << 20, 256)])
def test_lso_anchored_orbit_matches_oracle_and_sequential(emri, oracle, oracle_lso, ci, N, S):
    cfg = W.scaled(W.CONFIGS[ci], K=10, N=N)
    P = lso_params(cfg, cfg.K)
    out = {}
    for schedule in (1, 0):
        plan = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K)
        if S != 256:
            plan.set_coarse_stride(S)
        plan.set_orbit_schedule(schedule)
        plan.set_anchor(True)
        st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
        nodes = plan.orbit(dev(P), status=st)
        torch.cuda.synchronize()
        out[schedule] = (nodes.cpu().numpy(), st.cpu().numpy(), plan.orbit_report(cfg.K) if schedule else None)
        plan.close()
    n1, s1, modes = out[1]
    n0, s0, _ = out[0]
    print("status", s1, "modes", modes)
    assert np.array_equal(s0, s1)
    if True:
        for k in range(cfg.K):
            ref = oracle_lso.orbit(P[k], N, cfg.dt, S)
            assert s1[k] == ref["status"]
            if ref["status"]:
                assert not n1[k].any() and not n0[k].any()
                continue
            val, slope, inc = n1[k, :, 0:5].T, n1[k, :, 5:10].T, n1[k, :, 10:15].T
            for q in (0, 2, 4):
                assert np.max(np.abs(circ_diff(val[q], ref["val"][q]))) < 2e-11
                assert np.max(np.abs(circ_diff(val[q], n0[k, :, q]))) < 2e-12
                np.testing.assert_allclose(inc[q], ref["inc"][q], rtol=1e-13, atol=1e-15)
            for q in (1, 3):
                np.testing.assert_allclose(val[q], ref["val"][q], rtol=2e-14, atol=1e-300)
                np.testing.assert_allclose(val[q], n0[k, :, q], rtol=4e-16, atol=1e-300)
                np.testing.assert_allclose(inc[q], ref["inc"][q], rtol=1e-11, atol=1e-25)
            np.testing.assert_allclose(slope, ref["slope"], rtol=1e-12, atol=1e-30)
    assert (s1 == 0).sum() >= 5


def test_lso_anchored_waveform_and_loglike_match_oracle(emri, oracle, oracle_lso):
    cfg = W.scaled(W.CONFIGS[2], K=6, N=1 << 13)
    P = lso_params(cfg, cfg.K, e_hi=0.4)
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    h_ref, st_ref = oracle_lso.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    D = np.stack([oracle.rfft(h_ref[1, 0]), oracle.rfft(h_ref[1, 1])]) + W.noise_fft(cfg.N, cfg.dt, psd, 9)
    L_ref, _ = oracle_lso.loglike_batch(P, cfg.N, cfg.dt, cfg.n_max, D, psd)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    plan.set_anchor(True)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    logL = plan.loglike(dev(P), dev(D))
    torch.cuda.synchronize()
    assert np.array_equal(st.cpu().numpy(), st_ref) and not st_ref.any()
    for ch, got in ((0, hI.cpu().numpy()), (1, hII.cpu().numpy())):
        err = np.max(np.abs(got - h_ref[:, ch]), axis=1) / np.max(np.abs(h_ref[:, ch]), axis=1)
        print("LSO-anchored waveform err", err)
        assert np.all(err <= 1e-9)
        assert np.all(got[:, -1] != 0.0)                      # live up to the last sample: the window ends at plunge
    got = logL.cpu().numpy()
    assert np.all(np.abs(got - L_ref) <= 1e-9 * np.abs(L_ref) + 1e-6)
    # back to the default convention on the same plan
    plan.set_anchor(False)
    h2, _ = plan.waveform(dev(P))
    torch.cuda.synchronize()
    ref2, _ = oracle.waveform_batch(P[:1], cfg.N, cfg.dt, cfg.n_max)
    assert np.max(np.abs(h2.cpu().numpy()[0] - ref2[0, 0])) <= 1e-9 * np.max(np.abs(ref2[0, 0]))
    plan.close()


def test_paper_fig1_grid_matches_oracle(emri, oracle, oracle_lso):
    """the paper's own illustration (Figure 1): M = 1e6, mu = 10, spins 0 / 0.4 / 0.8, e_LSO = 0 / 0.3 / 0.6,
    the last hour before the LSO, and the same nine systems over the last year (N = 2^21, sampled)"""
    import os
    P = W.paper_fig1_params(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_fig1_parameters.txt"))
    if True:
        for N, n_max, idx in ((256, 20, None), (1 << 21, 30, "sampled")):
            dt = 15.0
            plan = emri.Plan(N, dt, n_max, 9)
            plan.set_anchor(True)
            st = torch.zeros(9, dtype=torch.int32, device="cuda")
            hI, hII = plan.waveform(dev(P), status=st)
            torch.cuda.synchronize()
            hI, hII, st = hI.cpu().numpy(), hII.cpu().numpy(), st.cpu().numpy()
            if idx is not None:
                rng = np.random.default_rng(1)
                idx = np.unique(np.concatenate([np.arange(0, 300), np.arange(N - 600, N), rng.integers(0, N, 1200)]))
            for k in range(9):
                a, b, s_ref = oracle_lso.waveform(P[k], N, dt, n_max, idx=idx)
                assert st[k] == s_ref
                if s_ref:
                    assert not hI[k].any()          # e grew past 1 on the way back: invalid on both sides
                    continue
                sel = slice(None) if idx is None else idx
                eI = np.max(np.abs(hI[k][sel] - a)) / np.max(np.abs(hI[k]))
                eII = np.max(np.abs(hII[k][sel] - b)) / np.max(np.abs(hII[k]))
                assert eI <= 1e-9 and eII <= 1e-9, (N, k, eI, eII)
            print(f"Fig. 1 grid, N = {N}: status {st}, modes {plan.orbit_report(9)}")
            plan.close()
