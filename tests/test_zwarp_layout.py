"""CPU restatement (numpy) of the data flow of the warp-owned z passes for N >= 256 (csrc/zwarp_pass.cuh, zwarp_inv.cuh):
stage 0 (radix R0, stride 16, twiddles w_H^(r q)), stage 1 (16-point DFT of 16 consecutive values), the Hermitian split
over the mirrored block pairs (k0, R0 - k0) with halved twiddles, the stored order p = 16 k0 + k1 <-> k = k0 + R0 k1,
the column swizzle pz ^ (y & 15), and the inverse in the opposite order.  Checked against numpy's rfft / irfft, so a
wrong partner slot, twiddle index or mirror offset in that index logic shows up without a GPU.  (Not the oracle; it
shares nothing with oracle/.)"""
import numpy as np
import pytest


def _forward_line(x, R0, y):
    """real line x[N] -> (row[H] in stored, swizzled order, Nyquist value), following k_zw_fwd step by step"""
    N = x.size
    H = N // 2
    assert H == R0 * 16
    z = x[0::2] + 1j * x[1::2]                       # z = 2 m + parity: complex element m
    wH = np.exp(-2j * np.pi * np.arange(H) / H)
    wN = np.exp(-2j * np.pi * np.arange(N) / N)
    # stage 0: task q = 0..15 takes elements q + 16 r, DFT over r, twiddle w_H^(r q), stores back in place
    s = np.empty(H, complex)
    for q in range(16):
        v = np.fft.fft(z[q + 16 * np.arange(R0)])
        v *= wH[(np.arange(R0) * q) % H]
        s[q + 16 * np.arange(R0)] = v
    # stage 1: block k0 = 16 consecutive values, plain 16-point DFT: slot 16 k0 + k1 holds Z[k0 + R0 k1]
    for k0 in range(R0):
        s[16 * k0:16 * k0 + 16] = np.fft.fft(s[16 * k0:16 * k0 + 16])
    row = np.empty(H, complex)
    sw = y & 15

    def pair(za, zb, k):                             # zw_r2c_pair with wh = w_N^k / 2
        wh = 0.5 * wN[k]
        t, u = za + np.conj(zb), za - np.conj(zb)
        g = u * wh
        return 0.5 * t - 1j * g, np.conj(0.5 * t + 1j * g)

    for k0 in range(1, R0 // 2):                     # block pairs (k0, R0 - k0), lane j = k1
        for j in range(16):
            xa, xb = pair(s[16 * k0 + j], s[16 * (R0 - k0) + 15 - j], k0 + R0 * j)
            row[16 * k0 + (j ^ sw)] = xa
            row[16 * (R0 - k0) + ((15 - j) ^ sw)] = xb
    KB = R0 // 2
    nyq = None
    for j in range(16):                              # the self-mirrored blocks 0 and KB share a half-warp
        if j == 0:
            z0, zh = s[0], s[8]
            row[0 ^ sw] = z0.real + z0.imag
            nyq = z0.real - z0.imag
            row[8 ^ sw] = np.conj(zh)
        elif j < 8:
            xa, xb = pair(s[j], s[16 - j], R0 * j)
            row[j ^ sw] = xa
            row[(16 - j) ^ sw] = xb
        else:
            jj = j - 8
            xa, xb = pair(s[16 * KB + jj], s[16 * KB + 15 - jj], KB + R0 * jj)
            row[16 * KB + (jj ^ sw)] = xa
            row[16 * KB + ((15 - jj) ^ sw)] = xb
    return row, nyq


def _inverse_line(row, nyq, R0, y):
    """(row, Nyquist value) -> real line, following k_zw_inv; unnormalised like the kernel (a factor N/2... = H)"""
    H = row.size
    N = 2 * H
    wH = np.exp(-2j * np.pi * np.arange(H) / H)
    wN = np.exp(-2j * np.pi * np.arange(N) / N)
    sw = y & 15
    s = np.empty(H, complex)

    def pair(xa, xb, k):                             # zw_c2r_pair
        wh = 0.5 * wN[k]
        t, u = xa + np.conj(xb), xa - np.conj(xb)
        o = u * np.conj(wh)
        return 0.5 * t + 1j * o, np.conj(0.5 * t - 1j * o)

    for k0 in range(1, R0 // 2):
        for j in range(16):
            za, zb = pair(row[16 * k0 + (j ^ sw)], row[16 * (R0 - k0) + ((15 - j) ^ sw)], k0 + R0 * j)
            s[16 * k0 + j] = za
            s[16 * (R0 - k0) + 15 - j] = zb
    KB = R0 // 2
    for j in range(16):
        if j == 0:
            x0, xh = row[0 ^ sw].real, nyq
            s[0] = 0.5 * (x0 + xh) + 0.5j * (x0 - xh)
            s[8] = np.conj(row[8 ^ sw])
        elif j < 8:
            s[j], s[16 - j] = pair(row[j ^ sw], row[(16 - j) ^ sw], R0 * j)
        else:
            jj = j - 8
            s[16 * KB + jj], s[16 * KB + 15 - jj] = pair(row[16 * KB + (jj ^ sw)], row[16 * KB + ((15 - jj) ^ sw)], KB + R0 * jj)
    for k0 in range(R0):                             # inverse of the last plan stage
        s[16 * k0:16 * k0 + 16] = np.fft.ifft(s[16 * k0:16 * k0 + 16]) * 16
    z = np.empty(H, complex)
    for q in range(16):                              # inverse stage 0: conjugate twiddle, inverse DFT over r
        v = s[q + 16 * np.arange(R0)] * np.conj(wH[(np.arange(R0) * q) % H])
        z[q + 16 * np.arange(R0)] = np.fft.ifft(v) * R0
    x = np.empty(N)
    x[0::2], x[1::2] = z.real, z.imag
    return x


@pytest.mark.parametrize("N,R0", [(256, 8), (512, 16)])
def test_warp_owned_z_pass_index_logic_matches_rfft(N, R0):
    rng = np.random.default_rng(N)
    H = N // 2
    for y in (0, 5, 15, 37):
        x = rng.normal(size=N)
        row, nyq = _forward_line(x, R0, y)
        X = np.fft.rfft(x)
        sw = y & 15
        for p in range(H):                           # stored slot p = 16 k0 + k1 holds frequency k0 + R0 k1, in column p ^ sw
            k0, k1 = divmod(p, 16)
            k = k0 + R0 * k1
            assert abs(row[p ^ sw] - X[k]) <= 1e-9 * np.abs(X).max(), (N, y, p)
        assert abs(nyq - X[H].real) <= 1e-9 * np.abs(X).max()
        back = _inverse_line(row, nyq, R0, y)
        assert np.abs(back - H * x).max() <= 1e-9 * H * np.abs(x).max()   # unnormalised half-length transforms: factor H
