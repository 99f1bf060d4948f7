"""Affine-invariant stretch move (Goodman & Weare 2010; emcee's default, PAPER.md:57, :122 and refs [37], [38])
-- CPU oracle of the config-4 driver, TEST INFRASTRUCTURE.

Plain Python / numpy, written from the published algorithm and the reading R19 of DESIGN.md:
fixed halves [0, K/2) and [K/2, K); for walker k of the active half: partner j uniform in the other
half, z = ((a-1) u + 1)^2 / a  (density g(z) ~ 1/sqrt(z) on [1/a, a]), proposal Y = X_j + z (X_k - X_j),
accepted iff  ln u' < (P_free - 1) ln z + lnp(Y) - lnp(X_k),  lnp = logL + uniform box prior.

Random numbers are a counter-based generator so that device and oracle can draw the same stream
without sharing code: Philox4x32-10 (Salmon et al., SC'11), key = (seed lo, seed hi), counter =
(step lo, step hi, 2 i + half, draw) with i the index inside the active half; draw 0 gives (u_partner,
u_z) from words (0,1) and (2,3), draw 1 gives u' from words (0,1).  A uniform in (0,1) is
((hi << 32 | lo) >> 11 + 1/2) / 2^53.  This file shares nothing with paper_2311_17174_b200/csrc/stretch.cuh.
"""
import math

import numpy as np

M0, M1 = 0xD2511F53, 0xCD9E8D57          # Philox4x32 multipliers
W0, W1 = 0x9E3779B9, 0xBB67AE85          # Weyl key increments
MASK = 0xFFFFFFFF


def philox4x32_10(counter, key):
    """counter: 4 uint32, key: 2 uint32 -> 4 uint32 (ten rounds)"""
    c0, c1, c2, c3 = (int(v) & MASK for v in counter)
    k0, k1 = (int(v) & MASK for v in key)
    for _ in range(10):
        p0, p1 = M0 * c0, M1 * c2
        hi0, lo0, hi1, lo1 = p0 >> 32, p0 & MASK, p1 >> 32, p1 & MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & MASK, lo1, (hi0 ^ c3 ^ k1) & MASK, lo0
        k0, k1 = (k0 + W0) & MASK, (k1 + W1) & MASK
    return c0, c1, c2, c3


def u53(hi, lo):
    return ((((hi << 32) | lo) >> 11) + 0.5) / 9007199254740992.0


def draws(seed, step, half, i):
    """-> (u_partner, u_z, u_accept) of walker i of the active half"""
    key = (seed & MASK, (seed >> 32) & MASK)
    ctr = (step & MASK, (step >> 32) & MASK, (2 * i + half) & MASK)
    a = philox4x32_10(ctr + (0,), key)
    b = philox4x32_10(ctr + (1,), key)
    return u53(a[0], a[1]), u53(a[2], a[3]), u53(b[0], b[1])


def propose(X, lo, hi, a, seed, step, half):
    """Proposals of the active half.  X: [K][P].  -> dict(Y[H][P], z[H], lnu[H], inbox[H], partner[H])"""
    X = np.asarray(X, dtype=np.float64)
    K, P = X.shape
    H = K // 2
    free = lo < hi
    Y = np.empty((H, P))
    z = np.empty(H)
    lnu = np.empty(H)
    inbox = np.empty(H, dtype=bool)
    partner = np.empty(H, dtype=np.int64)
    for i in range(H):
        k = half * H + i
        u1, u2, u3 = draws(seed, step, half, i)
        j = (1 - half) * H + min(int(u1 * H), H - 1)
        zi = ((a - 1.0) * u2 + 1.0) ** 2 / a
        y = np.where(free, X[j] + zi * (X[k] - X[j]), X[k])
        Y[i], z[i], lnu[i], partner[i] = y, zi, math.log(u3), j
        inbox[i] = bool(np.all(~free | ((y >= lo) & (y <= hi))))
    return dict(Y=Y, z=z, lnu=lnu, inbox=inbox, partner=partner)


def accept(logL_X, logL_Y, prop, n_free):
    """accept flags of the active half given logL of the current walkers (active half) and of the proposals"""
    lY = np.where(prop["inbox"], logL_Y, -np.inf)
    lnq = (n_free - 1) * np.log(prop["z"]) + lY - logL_X
    return np.isfinite(lY) & (prop["lnu"] < lnq), lnq


def half_step(X, logL, lo, hi, a, seed, step, half, loglike_fn):
    """one update of half `half` in place; loglike_fn(Y[H][P]) -> logL[H].  -> (accepted[H], prop, logL_Y)"""
    K = X.shape[0]
    H = K // 2
    prop = propose(X, lo, hi, a, seed, step, half)
    lY = loglike_fn(prop["Y"])
    act = slice(half * H, half * H + H)
    acc, _ = accept(logL[act], lY, prop, int(np.sum(lo < hi)))
    Xa, La = X[act], logL[act]
    Xa[acc] = prop["Y"][acc]
    La[acc] = np.where(prop["inbox"], lY, -np.inf)[acc]
    return acc, prop, lY
