"""Host-side check of the index algebra behind csrc/inject_whiten_long.cu: the four-step split
n = R L (sample L a + b, two-sided bin c + R e) with only the rows c <= R/2 formed, the pointwise stage applied on the
one-sided bin behind each two-sided index, and the Hermitian extension in the last pass reproduce
irfft((rfft(x) + H) f) exactly.  numpy only: no library, no oracle."""
import numpy as np
import pytest


@pytest.mark.parametrize("R,L", [(4, 32), (8, 64), (16, 16)])
def test_four_step_rows_reproduce_the_direct_transform(R, L):
    rng = np.random.default_rng(R * 1000 + L)
    n = R * L
    x = rng.standard_normal(n)
    filt = rng.random(n // 2 + 1)
    H = rng.standard_normal(n // 2 + 1) + 1j * rng.standard_normal(n // 2 + 1)
    H[0], H[-1] = H[0].real, H[-1].real
    ref = np.fft.irfft((np.fft.rfft(x) + H) * filt, n)

    def wn(e):
        return np.exp(-2j * np.pi * e / n)

    nr = R // 2 + 1
    b = np.arange(L)
    xa = x.reshape(R, L)                                       # xa[a][b] = x[L a + b]
    # pass 1: A[c][b] = w_n^(b c) sum_a x[L a + b] w_R^(a c), c <= R/2
    A = np.stack([wn(b * c) * sum(xa[a] * np.exp(-2j * np.pi * a * c / R) for a in range(R)) for c in range(nr)])
    # rows: Z[e] = X[c + R e]; pointwise on the one-sided bin behind it; unnormalised inverse
    B = np.zeros((nr, L), complex)
    for c in range(nr):
        Z = np.fft.fft(A[c])
        Y = np.zeros(L, complex)
        for e in range(L):
            k2 = c + R * e
            direct = k2 <= n // 2
            k = k2 if direct else n - k2
            v = Z[e] if direct else np.conj(Z[e])
            y = (v + H[k]) * filt[k]
            if k == 0 or k == n // 2:
                y = y.real
            Y[e] = y if direct else np.conj(y)
        B[c] = np.fft.ifft(Y) * L
    # pass 3: D[c][b] = w_n^(-b c) B[c][b], D[R - c] = conj D[c], y[L a + b] = Re sum_c D[c][b] w_R^(-a c)
    D = np.zeros((R, L), complex)
    for c in range(nr):
        D[c] = np.conj(wn(b * c)) * B[c]
    for c in range(nr, R):
        D[c] = np.conj(D[R - c])
    out = np.stack([sum(D[c] * np.exp(2j * np.pi * a * c / R) for c in range(R)).real for a in range(R)])
    assert np.abs(out.reshape(n) / n - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())
