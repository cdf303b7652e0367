"""Choice of sampled wavenumbers for the full-size parity tests (host logic only, no arithmetic of the method)."""
import numpy as np


def stratified_modes(N, n, seed):
    """Stored indices (ix, iy, iz) covering every residue class the kernels tile by: along the strided axes the first and
    the last column tile of each half (rows n and n + L of every register-stage class, positive and negative
    wavenumbers), along z every lane 0..15 and the last 16 stored entries; half systematic (each listed coordinate is
    hit), half uniform random; plus the box corners, the axes, the Nyquist planes and k = 0."""
    L, H = N // 2, N // 2
    t = min(16, L // 2)
    strided = np.unique(np.concatenate([np.arange(0, t), np.arange(L - t, L), np.arange(L + 1, L + 1 + t), np.arange(N - t, N)]))
    zs = np.unique(np.concatenate([np.arange(0, t), np.arange(H - t, H)]))
    ns_ = n // 2
    i = np.arange(ns_)
    sys_ = np.stack([strided[(7 * i) % len(strided)], strided[(13 * i + 5) % len(strided)], zs[(3 * i + 1) % len(zs)]], axis=1)
    rng = np.random.default_rng(seed)
    nr = n - ns_
    rnd = np.stack([rng.integers(0, N, nr), rng.integers(0, N, nr), rng.integers(0, H, nr)], axis=1)
    K = N // 2 - 1
    fixed = np.array([(1, 0, 0), (0, 1, 0), (0, 0, 1), (K, K, K), (N - K, N - K, K), (N - K, 3, K), (5, N - K, 0), (K, 0, 0),
                      (N // 2, 2, 2), (2, N // 2, 2), (2, 2, N // 2), (0, 0, 0)])
    return np.concatenate([sys_, rnd, fixed]).astype(np.int32)


def spectral_state(u):
    """The initial state u(0) = P_N u_0 (eq. 2.1, third line; readings A3, A8, A11) of a physical field u[3][N][N][N], written with
    numpy only: analysis transform with 1/N^3, Nyquist planes zeroed, Leray projector for k != 0, mean kept.  Used to hand the
    SAME spectral input to the CUDA path (ns_set_spectral) and to the oracle where the oracle's own orc_set_initial would take
    minutes (>= 192^3); orc_set_initial is pinned against exactly this restatement in tests/test_oracle_pins.py (P0)."""
    N = u.shape[-1]
    uh = np.fft.rfftn(u, axes=(1, 2, 3)) / float(N) ** 3
    uh[:, N // 2] = 0
    uh[:, :, N // 2] = 0
    uh[:, :, :, N // 2] = 0
    k = np.fft.fftfreq(N, 1.0 / N)
    kx, ky, kz = k[:, None, None], k[None, :, None], np.arange(N // 2 + 1.0)[None, None, :]
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    ku = (kx * uh[0] + ky * uh[1] + kz * uh[2]) / k2
    ku[0, 0, 0] = 0
    uh[0] -= kx * ku
    uh[1] -= ky * ku
    uh[2] -= kz * ku
    return np.ascontiguousarray(uh)
