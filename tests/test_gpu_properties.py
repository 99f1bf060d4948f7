"""Properties of the CUDA path that hold at any size (layer 4): exact scalings, angle periodicities,
walker-permutation equivariance, run-to-run bitwise reproducibility."""
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


@pytest.fixture(scope="module")
def case(emri):
    cfg = W.scaled(W.CONFIGS[2], K=8, N=1 << 14)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    hI, hII = plan.waveform(dev(P))
    D = plan.data_fft(hI[0].contiguous(), hII[0].contiguous()) + dev(W.noise_fft(cfg.N, cfg.dt, psd, 5))
    logL = plan.loglike(dev(P), D)
    torch.cuda.synchronize()
    yield cfg, P, plan, hI.cpu().numpy(), hII.cpu().numpy(), D, logL.cpu().numpy()
    plan.close()


def wave(plan, P):
    hI, hII = plan.waveform(dev(P))
    torch.cuda.synchronize()
    return hI.cpu().numpy(), hII.cpu().numpy()


def test_strain_scales_as_one_over_distance_in_gr(emri):
    """h ~ 1/d_GW; in GR (Xi0 = 1) doubling D_L halves the strain up to the rounding of 1/D"""
    cfg = W.scaled(W.CONFIGS[1], K=4, N=1 << 13)
    P = W.draw_params(cfg)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    a, _ = wave(plan, P)
    P2 = P.copy()
    P2[:, W.P_DL] *= 2.0
    b, _ = wave(plan, P2)
    assert np.max(np.abs(a - 2.0 * b)) <= 4e-16 * np.max(np.abs(a))
    plan.close()


@pytest.mark.parametrize("col,shift", [(W.P_PHI0, 2 * np.pi), (W.P_GAM0, np.pi), (W.P_ALP0, 2 * np.pi),
                                       (W.P_PHS, 2 * np.pi), (W.P_PHK, 2 * np.pi)])
def test_angle_periodicities(case, col, shift):
    """only n Phi, 2 gamma and alpha enter (integers n): the waveform is periodic in the initial angles and azimuths"""
    cfg, P, plan, hI, hII, D, logL = case
    P2 = P.copy()
    P2[:, col] += shift
    a, b = wave(plan, P2)
    tol = 3e-12 * cfg.n_max          # rounding of (angle + period)/2pi, times the harmonic number
    assert np.max(np.abs(a - hI)) <= tol * np.max(np.abs(hI)) and np.max(np.abs(b - hII)) <= tol * np.max(np.abs(hII))


def test_walker_permutation_equivariance_is_bitwise(case):
    cfg, P, plan, hI, hII, D, logL = case
    perm = np.array([5, 2, 7, 0, 1, 6, 3, 4])
    a, b = wave(plan, P[perm])
    assert np.array_equal(a, hI[perm]) and np.array_equal(b, hII[perm])
    L2 = plan.loglike(dev(P[perm]), D)
    torch.cuda.synchronize()
    assert np.array_equal(L2.cpu().numpy(), logL[perm])


def test_repeated_calls_are_bitwise_identical(case):
    cfg, P, plan, hI, hII, D, logL = case
    for _ in range(3):
        L2 = plan.loglike(dev(P), D)
        torch.cuda.synchronize()
        assert np.array_equal(L2.cpu().numpy(), logL)
    a, b = wave(plan, P)
    assert np.array_equal(a, hI) and np.array_equal(b, hII)


def test_quadratic_identity_of_the_likelihood(case):
    """logL(d, h) = -1/2 (<d|d> - 2<d|h> + <h|h>): with d -> 0 and d -> 2h the cross term cancels"""
    cfg, P, plan, hI, hII, D, logL = case
    p0 = dev(P[:1])
    H = plan.waveform_fft(p0)[0]
    zero = torch.zeros_like(H)
    hh = -2.0 * plan.loglike(p0, zero).cpu().numpy()[0]            # <h|h>
    assert abs(plan.loglike(p0, 2.0 * H).cpu().numpy()[0] + 0.5 * hh) <= 1e-12 * hh      # <2h-h|2h-h> = <h|h>
    assert abs(plan.loglike(p0, H).cpu().numpy()[0]) <= 1e-14 * hh
