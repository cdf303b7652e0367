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
