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
