"""BASELINE.json configs at FULL size, in the launch configuration bench.py times (whole ensemble in one
emri_loglike call), compared with the oracle on a seeded subset of walkers and on sampled outputs;
plus the edge cases of the boundary (non-power-of-two N, one walker, the n_max cap, masked bins)."""
import numpy as np
import pytest

from paper_2311_17174_b200 import workloads as W
from survey_recipe import with_plunging_walkers

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


def logl_ok(got, ref):
    return np.all(np.abs(got - ref) <= 1e-9 * np.abs(ref) + 1e-6)


def subset_with_plungers(oracle, cfg, n=16):
    """SURVEY 8(d)-3's 16 walkers: argmax e0, argmin M, argmax mu/M, indices 0-3, seeded draws -- three of the draws
    replaced by the ensemble's last three rows, re-placed by the survey's nu0 rule (8(d)-1) so that they plunge
    1.25, 1.35 and 1.5 observation lengths after the window starts (the strongly chirping regime of PAPER.md:120)"""
    P = W.draw_params(cfg)
    rows = [cfg.K - 1, cfg.K - 2, cfg.K - 3]
    P = with_plunging_walkers(oracle, P, cfg, rows)
    if cfg.K <= n:
        return P, np.arange(cfg.K), rows
    # parity_walker_subset keeps the extremes and 0-3 whatever n is; ask for n - 3 and add the plungers
    P_rest = P.copy()
    sub = [int(k) for k in W.parity_walker_subset(P_rest, n=n - 3)]
    extra = [r for r in rows if r not in sub]
    sub = sub + extra
    rng = np.random.default_rng(7)
    while len(sub) < n:                      # a plunger row was already picked: top up with seeded draws
        k = int(rng.integers(0, cfg.K))
        if k not in sub:
            sub.append(k)
    return P, np.array(sorted(sub)), rows


@pytest.mark.parametrize("ci", [0, 1, 2, 3])
def test_full_size_loglike_on_walker_subset(emri, oracle, ci):
    cfg = W.CONFIGS[ci]
    P, sub, plungers = subset_with_plungers(oracle, cfg)
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    if cfg.K > 16:
        assert len(sub) == 16 and {int(np.argmax(P[:, W.P_E0])), int(np.argmin(P[:, W.P_M])),
                                   int(np.argmax(P[:, W.P_MU] / P[:, W.P_M]))} <= set(sub.tolist())
    hI, hII, st0 = oracle.waveform(P[0], cfg.N, cfg.dt, cfg.n_max)
    D = np.stack([oracle.rfft(hI), oracle.rfft(hII)])
    if cfg.noise_seed:
        D = D + W.noise_fft(cfg.N, cfg.dt, psd, cfg.noise_seed)
    ref, st_ref = oracle.loglike_batch(P[sub], cfg.N, cfg.dt, cfg.n_max, D, psd)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    got = plan.loglike(dev(P), dev(D), status=st)
    torch.cuda.synchronize()
    got, st = got.cpu().numpy(), st.cpu().numpy()
    diff = np.abs(got[sub] - ref)
    print(f"cfg{ci} K={cfg.K} N={cfg.N} n_max={cfg.n_max}: {len(sub)} walkers, max |logL| {np.max(np.abs(ref)):.4e}, "
          f"max |dlogL| {np.max(diff):.2e}, max |dlogL| / tolerance {np.max(diff / (1e-9 * np.abs(ref) + 1e-6)):.2e}")
    assert not st.any() and not st_ref.any()
    assert np.all(np.isfinite(got)) and logl_ok(got[sub], ref)
    if not cfg.noise_seed:
        assert abs(got[0]) <= 1e-6          # noise-less data = walker 0's own waveform
    modes = plan.orbit_report(cfg.K)
    assert np.all(modes == 1)              # every walker's parallel-in-time orbit verified
    rep = plan.synth_report()
    print(f"cfg{ci} stage (b) paths: {rep}")
    assert rep["units"] >= cfg.K * -(-cfg.N // 4096) and rep["skipped_units"] == 0     # units of <= 16 tiles
    assert sum(rep["by_order"].values()) + rep["base_units"] == rep["units"]
    plan.close()


@pytest.mark.parametrize("ci", [1, 2, 3])
def test_full_size_waveform_sampled(emri, oracle, ci):
    cfg = W.CONFIGS[ci]
    P, sub, plungers = subset_with_plungers(oracle, cfg)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, len(sub))
    hI, hII = plan.waveform(dev(P[sub]))
    torch.cuda.synchronize()
    hI, hII = hI.cpu().numpy(), hII.cpu().numpy()
    rng = np.random.default_rng(100 + ci)
    idx = np.unique(np.concatenate([np.arange(0, 520), np.arange(cfg.N - 520, cfg.N), rng.integers(0, cfg.N, 3000)]))
    worst = 0.0
    for r, k in enumerate(sub):
        a, b, st = oracle.waveform(P[k], cfg.N, cfg.dt, cfg.n_max, idx=idx)
        eI = np.max(np.abs(hI[r, idx] - a)) / np.max(np.abs(hI[r]))
        eII = np.max(np.abs(hII[r, idx] - b)) / np.max(np.abs(hII[r]))
        assert st == 0 and eI <= H_TOL and eII <= H_TOL, (k, eI, eII)
        worst = max(worst, eI, eII)
    print(f"cfg{ci}: {len(sub)} walkers x {len(idx)} sampled outputs, max |dh| / max |h| = {worst:.2e}")
    plan.close()


def test_non_power_of_two_length_and_single_walker(emri, oracle):
    """N = 1000 (cuFFT takes any even N); the oracle's transform here is its naive O(N^2) DFT"""
    cfg = W.scaled(W.CONFIGS[1], K=3, N=1000)
    P = W.draw_params(cfg)
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    h_ref, _ = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    D = np.stack([oracle.dft_naive(h_ref[0, 0]), oracle.dft_naive(h_ref[0, 1])]) + W.noise_fft(cfg.N, cfg.dt, psd, 7)
    ref = np.array([oracle.loglike(np.stack([oracle.dft_naive(h_ref[k, 0]), oracle.dft_naive(h_ref[k, 1])]), D, psd,
                                   cfg.N, cfg.dt) for k in range(cfg.K)])
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    got = plan.loglike(dev(P), dev(D))
    one = plan.loglike(dev(P[1:2]), dev(D))
    sp = plan.waveform_fft(dev(P[:1]))
    torch.cuda.synchronize()
    assert logl_ok(got.cpu().numpy(), ref)
    assert one.cpu().numpy()[0] == got.cpu().numpy()[1]                 # K = 1 gives the same bits
    H0 = oracle.dft_naive(h_ref[0, 0])
    assert np.max(np.abs(sp.cpu().numpy()[0, 0] - H0)) <= 1e-9 * np.max(np.abs(H0))
    plan.close()


def test_harmonic_cap_and_eccentric_walkers(emri, oracle):
    """n_max = 48 (EMRI_NMAX_CAP) with e0 up to 0.5: long base series, high local orders"""
    cfg = W.scaled(W.CONFIGS[3], K=6, N=1 << 12, n_max=48)
    P = W.draw_params(cfg)
    P[:, W.P_E0] = np.linspace(0.0, 0.5, cfg.K)
    for k in range(cfg.K):
        P[k, W.P_NU0] = W.nu0_for_plunge_after(P[k, W.P_M], P[k, W.P_MU], P[k, W.P_E0], 4.0 * cfg.T_obs)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    hI, hII = plan.waveform(dev(P))
    torch.cuda.synchronize()
    h_ref, st = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    assert not st.any()
    for ch, got in ((0, hI.cpu().numpy()), (1, hII.cpu().numpy())):
        err = np.max(np.abs(got - h_ref[:, ch]), axis=1) / np.max(np.abs(h_ref[:, ch]), axis=1)
        print("n_max=48 err", err)
        assert np.all(err <= H_TOL)
    plan.close()


@pytest.mark.parametrize("n_max,e_hi,N", [(96, 0.6, 3 * 4096 + 2), (128, 0.7, 1 << 12), (64, 0.3, 1 << 13)])
def test_many_harmonics_by_the_bessel_path(emri, oracle, n_max, e_hi, N):
    """n_max beyond 48 (the overtone loop; SURVEY f-4): the local series come from Bessel recurrences instead of
    the base series in e^2, whose terms would cancel by e^{n e}.  Element-wise against the oracle (power-series Bessel
    functions of order > argument), eccentricities up to e_hi, including e = 0 and a walker close to plunge whose units
    overflow the local orders and take the per-sample recurrence fallback"""
    cfg = W.scaled(W.CONFIGS[3], K=6, N=N, n_max=n_max)
    P = W.draw_params(cfg)
    P[:, W.P_E0] = np.linspace(0.0, e_hi, cfg.K)
    for k in range(cfg.K):
        P[k, W.P_NU0] = W.nu0_for_plunge_after(P[k, W.P_M], P[k, W.P_MU], P[k, W.P_E0], 4.0 * 2 ** 21 * cfg.dt)
    P[4, W.P_M], P[4, W.P_MU] = 2e5, 80.0
    P[4, W.P_NU0] = 0.97 * W.nu_lso_hz(P[4, W.P_M], P[4, W.P_E0])            # hours from plunge: e^2 moves fast
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    rep = plan.synth_report()
    torch.cuda.synchronize()
    h_ref, st_ref = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    print(f"n_max={n_max}: paths {rep} status {st.cpu().numpy()} {st_ref}")
    assert np.array_equal(st.cpu().numpy(), st_ref)
    for ch, got in ((0, hI.cpu().numpy()), (1, hII.cpu().numpy())):
        live = np.max(np.abs(h_ref[:, ch]), axis=1) > 0
        err = np.max(np.abs(got[live] - h_ref[live, ch]), axis=1) / np.max(np.abs(h_ref[live, ch]), axis=1)
        print("  err", err)
        assert np.all(err <= H_TOL)
    # the forced fallback (every unit evaluates the recurrences per sample) gives the same waveform
    plan.set_synth_debug(force_base=True)
    hI2, _ = plan.waveform(dev(P))
    rep2 = plan.synth_report()
    assert rep2["base_units"] == rep2["units"] > 0
    g, g2 = hI.cpu().numpy(), hI2.cpu().numpy()
    assert np.max(np.abs(g - g2)) <= 1e-11 * np.max(np.abs(g))
    plan.close()


def test_circular_orbit_has_only_the_quadrupole(emri, oracle):
    """e = 0 exactly (reading R18): e' = 0 keeps it there and only n = 2 survives: n_max = 2 and 30 agree"""
    cfg = W.scaled(W.CONFIGS[1], K=2, N=1 << 12)
    P = W.draw_params(cfg)
    P[:, W.P_E0] = 0.0
    out = []
    for n_max in (2, 30):
        plan = emri.Plan(cfg.N, cfg.dt, n_max, cfg.K)
        hI, hII = plan.waveform(dev(P))
        torch.cuda.synchronize()
        out.append((hI.cpu().numpy(), hII.cpu().numpy()))
        plan.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    h_ref, _ = oracle.waveform_batch(P, cfg.N, cfg.dt, 30)
    assert np.max(np.abs(out[1][0] - h_ref[:, 0])) <= H_TOL * np.max(np.abs(h_ref[:, 0]))


def test_fully_masked_psd_gives_zero_and_invalid_walker_minus_inf(emri):
    cfg = W.scaled(W.CONFIGS[0], K=3, N=1 << 10)
    P = W.draw_params(cfg)
    P[2, W.P_DL] = -1.0
    psd = np.full(cfg.N // 2 + 1, np.inf)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    D = torch.ones((2, cfg.N // 2 + 1), dtype=torch.complex128, device="cuda")
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    got = plan.loglike(dev(P), D, status=st).cpu().numpy()
    assert got[0] == 0.0 and got[1] == 0.0 and got[2] == -np.inf
    assert list(st.cpu().numpy()) == [0, 0, 1]
    plan.close()


def test_status_bits_delay_and_cosmology_setting(emri, oracle):
    """bit 4: |Delta T| beyond the one-interval guard (reading R20) => zero rows, logL = -inf, as the oracle;
    emri_plan_set_cosmology reaches the amplitude through z(D_L) and Xi(z)"""
    cfg = W.scaled(W.CONFIGS[2], K=4, N=1 << 12)
    P = W.draw_params(cfg)
    P[1, W.P_DELT] = 1e-12            # |Delta T| ~ 1e5 s > Delta = 3840 s
    P[2, W.P_DELT] = -3e-14           # ~ 3e3 s: inside the guard
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt)
    h_ref, st_ref = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max)
    assert list(st_ref) == [0, 4, 0, 0]
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K, psd)
    st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
    hI, hII = plan.waveform(dev(P), status=st)
    D = plan.data_fft(hI[0].contiguous(), hII[0].contiguous())
    logL = plan.loglike(dev(P), D)
    torch.cuda.synchronize()
    assert list(st.cpu().numpy()) == [0, 4, 0, 0]
    hI = hI.cpu().numpy()
    assert not hI[1].any() and logL.cpu().numpy()[1] == -np.inf
    for k in (0, 2, 3):
        assert np.max(np.abs(hI[k] - h_ref[k, 0])) <= H_TOL * np.max(np.abs(h_ref[k, 0]))
    # another cosmology: both sides move together
    plan.set_cosmology(73.0, 0.27)
    hI2, _ = plan.waveform(dev(P))
    torch.cuda.synchronize()
    h2, _ = oracle.waveform_batch(P, cfg.N, cfg.dt, cfg.n_max, H0=73.0, Om=0.27)
    hI2 = hI2.cpu().numpy()
    assert np.max(np.abs(hI2[0] - h2[0, 0])) <= H_TOL * np.max(np.abs(h2[0, 0]))
    assert np.max(np.abs(hI2[0] - hI[0])) > 1e-4 * np.max(np.abs(hI[0]))       # Xi(z) differs (Xi0 != 1 in this config)
    plan.close()


def test_argument_errors_on_the_device(emri):
    cfg = W.scaled(W.CONFIGS[0], K=2, N=1 << 10)
    plan = emri.Plan(cfg.N, cfg.dt, cfg.n_max, cfg.K)
    P3 = dev(W.draw_params(cfg, K=3))
    with pytest.raises(emri.EmriError, match="invalid argument"):
        plan.waveform(P3)                                   # K > K_max
    with pytest.raises(emri.EmriError, match="invalid argument"):
        plan.set_coarse_stride(100)                         # not a power of two
    with pytest.raises(emri.EmriError, match="invalid argument"):
        plan.set_cosmology(-1.0, 0.3)
    plan.close()


@pytest.mark.parametrize("N,S", [(4, 256), (16, 2), (258, 256), (514, 64), (2050, 256)])
def test_tiny_and_ragged_lengths(emri, oracle, N, S):
    """the smallest plans: one coarse interval, one shooting segment, a single ragged tile; stride 2 with 4 samples per
    tile row; waveform parity and both orbit schedules"""
    cfg = W.scaled(W.CONFIGS[1], K=3, N=N)
    P = W.draw_params(W.scaled(W.CONFIGS[1], K=3, N=1 << 16))      # nu0 placed for an 11-day window: nothing plunges here
    out = []
    for schedule in (1, 0):
        plan = emri.Plan(N, cfg.dt, cfg.n_max, cfg.K)
        plan.set_coarse_stride(S)
        plan.set_orbit_schedule(schedule)
        st = torch.zeros(cfg.K, dtype=torch.int32, device="cuda")
        hI, hII = plan.waveform(dev(P), status=st)
        torch.cuda.synchronize()
        out.append((hI.cpu().numpy(), hII.cpu().numpy(), st.cpu().numpy()))
        plan.close()
    h_ref, st_ref = oracle.waveform_batch(P, N, cfg.dt, cfg.n_max, S=S)
    for hI, hII, st in out:
        assert np.array_equal(st, st_ref) and not st.any()
        assert np.max(np.abs(hI - h_ref[:, 0])) <= H_TOL * np.max(np.abs(h_ref[:, 0]))
        assert np.max(np.abs(hII - h_ref[:, 1])) <= H_TOL * np.max(np.abs(h_ref[:, 1]))
    assert np.max(np.abs(out[0][0] - out[1][0])) <= 1e-12 * np.max(np.abs(out[1][0]))
