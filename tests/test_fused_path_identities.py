"""The two identities the fused transform + likelihood kernel (csrc/fftlike.cuh, reading D16) rests on,
checked with numpy on the CPU -- the mathematics of the readings, not the CUDA code (the `-m gpu` tests compare that with the
plain path and with the oracle):
  1. the two-pass split of the DFT, N = N1 N2, with the index conventions and the inter-pass twiddle the kernel uses;
  2. Eq. 8 as a sum over single elements of Z = DFT(h_I + i h_II), without pairing bins m and N - m."""
import numpy as np
import pytest


@pytest.mark.parametrize("N1,N2", [(4, 8), (16, 4), (8, 8)])
def test_two_pass_split_of_the_dft(N1, N2):
    """Z[m1 + N1 m2] = sum_{i2} W_N^{i2 m1} W_N2^{i2 m2} [ sum_{i1} z[N2 i1 + i2] W_N1^{i1 m1} ]"""
    rng = np.random.default_rng(N1 * 100 + N2)
    N = N1 * N2
    z = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    zz = z.reshape(N1, N2)                                        # [i1][i2]
    Y = np.fft.fft(zz, axis=0)                                    # pass A: N1-point transforms down the columns -> [m1][i2]
    m1 = np.arange(N1)[:, None]
    i2 = np.arange(N2)[None, :]
    Y = Y * np.exp(-2j * np.pi * i2 * m1 / N)                     # inter-pass twiddle W_N^{i2 m1}
    Zrows = np.fft.fft(Y, axis=1)                                 # pass B: N2-point transforms along the rows -> [m1][m2]
    Z = np.empty(N, dtype=complex)
    for a in range(N1):
        for b in range(N2):
            Z[a + N1 * b] = Zrows[a, b]
    assert np.allclose(Z, np.fft.fft(z), rtol=0, atol=1e-12 * np.max(np.abs(Z)))


def test_eq8_without_pairing():
    """-(2 dt/N) sum_m w_m (|D_I - H_I|^2 + |D_II - H_II|^2) = -(2 dt/N) [ C_self + sum_j alpha_j |Z_j - ZD_j|^2 ]
    with Z = DFT(h_I + i h_II), ZD[m] = D_I[m] + i D_II[m], ZD[N-m] = conj D_I[m] + i conj D_II[m], alpha = w/2; the
    self-paired bins m = 0, N/2 carry alpha = w, ZD = Re D_I + i Re D_II and C_self = w (Im D_I^2 + Im D_II^2)"""
    rng = np.random.default_rng(8)
    N, dt = 64, 15.0
    Nf = N // 2 + 1
    hI, hII = rng.standard_normal(N), rng.standard_normal(N)
    D = rng.standard_normal((2, Nf)) + 1j * rng.standard_normal((2, Nf))       # DC / Nyquist deliberately not real
    w = rng.uniform(0.5, 2.0, Nf)
    w[3] = 0.0                                                    # a masked bin
    # the definition, bin by bin (what the plain path and the oracle evaluate)
    HI, HII = np.fft.rfft(hI), np.fft.rfft(hII)
    direct = -(2 * dt / N) * np.sum(w * (np.abs(D[0] - HI) ** 2 + np.abs(D[1] - HII) ** 2))
    # the pairing-free form on Z = DFT(h_I + i h_II)
    Z = np.fft.fft(hI + 1j * hII)
    m = np.arange(Nf)
    assert np.allclose((Z[m] + np.conj(Z[(N - m) % N])) / 2, HI) and np.allclose((Z[m] - np.conj(Z[(N - m) % N])) / 2j, HII)
    alpha = np.zeros(N)
    ZD = np.zeros(N, dtype=complex)
    c_self = 0.0
    for k in range(Nf):
        j = (N - k) % N
        if j == k:
            alpha[k] = w[k]
            ZD[k] = D[0, k].real + 1j * D[1, k].real
            c_self += w[k] * (D[0, k].imag ** 2 + D[1, k].imag ** 2)
        else:
            alpha[k] = alpha[j] = 0.5 * w[k]
            ZD[k] = D[0, k] + 1j * D[1, k]
            ZD[j] = np.conj(D[0, k]) + 1j * np.conj(D[1, k])
    fused = -(2 * dt / N) * (c_self + np.sum(alpha * np.abs(Z - ZD) ** 2))
    assert fused == pytest.approx(direct, rel=1e-13)
    # and no cancellation: data = the model itself gives exactly 0
    D0 = np.stack([HI, HII])
    ZD0 = np.zeros(N, dtype=complex)
    for k in range(Nf):
        j = (N - k) % N
        ZD0[k] = D0[0, k] + 1j * D0[1, k] if j != k else D0[0, k].real + 1j * D0[1, k].real
        if j != k:
            ZD0[j] = np.conj(D0[0, k]) + 1j * np.conj(D0[1, k])
    assert np.sum(alpha * np.abs(Z - ZD0) ** 2) <= 1e-24 * np.sum(alpha * np.abs(Z) ** 2)
