"""Pins of the stretch-move oracle (oracle/stretch.py): the counter-based generator against the
known-answer vectors of the Random123 distribution (Salmon et al., SC'11), the stretch density
g(z) ~ 1/sqrt(z) on [1/a, a] (Goodman & Weare 2010), and the invariant distribution of the whole
move on a target whose moments are known in closed form."""
import numpy as np

from oracle import stretch


def test_philox4x32_10_known_answers():
    # Random123 kat_vectors, philox4x32 with 10 rounds
    assert stretch.philox4x32_10((0, 0, 0, 0), (0, 0)) == (0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8)
    f = 0xFFFFFFFF
    assert stretch.philox4x32_10((f, f, f, f), (f, f)) == (0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD)
    assert stretch.philox4x32_10((0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344), (0xA4093822, 0x299F31D0)) == \
        (0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1)


def test_uniforms_are_in_the_open_interval_and_well_spread():
    u = np.array([stretch.draws(7, s, s & 1, i) for s in range(40) for i in range(50)])
    assert u.min() > 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.02 and abs(u.var() - 1.0 / 12.0) < 0.01
    assert stretch.u53(0, 0) == 0.5 / 2 ** 53 and stretch.u53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 0.5 / 2 ** 53
    # distinct counters give distinct streams
    assert stretch.draws(1, 0, 0, 0) != stretch.draws(1, 0, 1, 0) != stretch.draws(1, 1, 0, 0) != stretch.draws(2, 0, 0, 0)


def test_stretch_factor_has_the_goodman_weare_density():
    a = 2.0
    z = np.array([((a - 1.0) * stretch.draws(3, s, 0, i)[1] + 1.0) ** 2 / a for s in range(100) for i in range(100)])
    assert z.min() >= 1.0 / a and z.max() <= a
    # CDF of g(z) ~ 1/sqrt(z) on [1/a, a]: (sqrt(z) - 1/sqrt(a)) / (sqrt(a) - 1/sqrt(a))
    zs = np.sort(z)
    cdf = (np.sqrt(zs) - a ** -0.5) / (a ** 0.5 - a ** -0.5)
    emp = (np.arange(zs.size) + 0.5) / zs.size
    assert np.max(np.abs(cdf - emp)) < 0.02          # Kolmogorov distance, n = 1e4
    # symmetry g(1/z) = z g(z) that makes the move reversible: E[z^-1/2] = E[z^1/2]/... check one moment
    assert abs(np.mean(1.0 / np.sqrt(z)) * (a ** 0.5 - a ** -0.5) - np.log(a)) < 0.02


def test_proposals_lie_on_the_line_through_the_partner_and_respect_fixed_columns():
    rng = np.random.default_rng(0)
    K, P = 8, 5
    X = rng.normal(size=(K, P))
    lo, hi = np.full(P, -10.0), np.full(P, 10.0)
    lo[2] = hi[2] = 0.0                                  # fixed column
    prop = stretch.propose(X, lo, hi, 2.0, seed=11, step=3, half=1)
    for i in range(K // 2):
        k, j, z = K // 2 + i, prop["partner"][i], prop["z"][i]
        assert 0 <= j < K // 2
        free = [0, 1, 3, 4]
        np.testing.assert_allclose(prop["Y"][i, free] - X[j, free], z * (X[k, free] - X[j, free]), rtol=1e-14)
        assert prop["Y"][i, 2] == X[k, 2]
    assert prop["inbox"].all()
    prop2 = stretch.propose(X * 100.0, lo, hi, 2.0, seed=11, step=3, half=1)
    assert not prop2["inbox"].all()


def test_chain_samples_a_gaussian_with_the_right_moments():
    """the move leaves the target invariant: 3-d correlated Gaussian, 64 walkers, 1500 steps"""
    rng = np.random.default_rng(5)
    P, K = 3, 64
    A = rng.normal(size=(P, P))
    cov = A @ A.T + np.eye(P)
    icov = np.linalg.inv(cov)
    mu = np.array([1.0, -2.0, 0.5])

    def logl(Y):
        d = Y - mu
        return -0.5 * np.einsum("ij,jk,ik->i", d, icov, d)

    X = mu + rng.normal(size=(K, P))
    L = logl(X)
    lo, hi = np.full(P, -1e3), np.full(P, 1e3)
    keep, nacc = [], 0
    for step in range(1500):
        for half in (0, 1):
            acc, _, _ = stretch.half_step(X, L, lo, hi, 2.0, seed=99, step=step, half=half, loglike_fn=logl)
            nacc += acc.sum()
        if step >= 300:
            keep.append(X.copy())
    S = np.concatenate(keep)
    assert 0.3 < nacc / (1500 * K) < 0.9
    np.testing.assert_allclose(S.mean(axis=0), mu, atol=0.08)
    np.testing.assert_allclose(np.cov(S.T), cov, rtol=0.12, atol=0.08)
    np.testing.assert_allclose(L, logl(X), rtol=1e-12)      # the cached logL follows the walkers
