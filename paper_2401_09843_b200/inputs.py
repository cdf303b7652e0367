"""Seeded synthetic input generators shared by the CUDA path's tests/bench and the CPU oracle's tests.

This module holds NONE of the method's arithmetic (no padding, no RHS, no projection, no RK): it only
makes physical-space velocity samples u[3][N][N][N] (fp64, C order, index [comp][ix][iy][iz],
x_j = 2*pi*j/N) that are handed unchanged to both `ns_set_initial` (CUDA) and `orc_set_initial`
(oracle).  Random numbers come from a counter-based SplitMix64 stream written out here, so arrays do
not depend on library versions.  numpy.fft is used only to shape the spectrum of the random fields.

Workload recipes (they stand in for the paper's workloads):
  config 1  taylor_green_perturbed   N=32   z-independent Taylor-Green + 1e-3 band-limited noise
  config 2  gaussian_field k^4 exp   N=128  E(k) ~ k^4 exp(-2 (k/4)^2), E_tot = 0.5
  config 3  shear_layer              N=256  doubly periodic perturbed shear layer
  config 4  shear_layer ensemble     32 x N=128, seed 1000+i per sample
  config 5  gaussian_field k^-5/3    N=512  E(k) ~ k^-5/3 on 1 <= k <= N/3, E_tot = 0.5
The paper's own experiments (NEXT-2 of SURVEY.md 8(f), hyperviscosity order s = 1.5):
  tg3d      taylor_green_3d_perturbed   eq. (6.1)-(6.3)
  cyl       cylindrical_shear           eq. (6.4)-(6.6)
"""
from __future__ import annotations

import hashlib

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_MIX1 = np.uint64(0xBF58476D1CE4E5B9)
_MIX2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """Counter-based SplitMix64: 64 random bits for every (seed, stream, index)."""
    with np.errstate(over="ignore"):
        idx = np.asarray(index, dtype=np.uint64)
        z = (np.uint64(seed & 0xFFFFFFFFFFFFFFFF) * _MIX2
             + np.uint64(stream & 0xFFFFFFFFFFFFFFFF) * _MIX1
             + (idx + np.uint64(1)) * _GOLDEN)
        z = (z ^ (z >> np.uint64(30))) * _MIX1
        z = (z ^ (z >> np.uint64(27))) * _MIX2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """n doubles uniform in [0,1)."""
    idx = np.arange(offset, offset + n, dtype=np.uint64)
    return (splitmix64(seed, stream, idx) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(seed: int, stream: int, n: int) -> np.ndarray:
    """n standard normals by Box-Muller on two uniform streams."""
    out = np.empty(n, dtype=np.float64)
    chunk = 1 << 24
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        u1 = uniform01(seed, 2 * stream, m, s)
        u2 = uniform01(seed, 2 * stream + 1, m, s)
        out[s:s + m] = np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)
    return out


def grid(N: int):
    x = 2.0 * np.pi * np.arange(N) / N
    return np.meshgrid(x, x, x, indexing="ij")


def taylor_green_2d(N: int) -> np.ndarray:
    """z-independent Taylor-Green vortex u = (sin x cos y, -cos x sin y, 0)."""
    X, Y, _ = grid(N)
    u = np.zeros((3, N, N, N))
    u[0] = np.sin(X) * np.cos(Y)
    u[1] = -np.cos(X) * np.sin(Y)
    return u


def abc_flow(N: int, A: float = 1.0, B: float = 0.7, C: float = 0.4) -> np.ndarray:
    """Beltrami (ABC) flow: curl u = u."""
    X, Y, Z = grid(N)
    u = np.empty((3, N, N, N))
    u[0] = A * np.sin(Z) + C * np.cos(Y)
    u[1] = B * np.sin(X) + A * np.cos(Z)
    u[2] = C * np.sin(Y) + B * np.cos(X)
    return u


def _wavenumbers(N: int):
    k = np.fft.fftfreq(N, 1.0 / N)
    kz = np.fft.rfftfreq(N, 1.0 / N)
    return np.meshgrid(k, k, kz, indexing="ij")


def gaussian_field(N: int, seed: int, spectrum, e_tot: float | None = None, rms: float | None = None) -> np.ndarray:
    """Band-limited Gaussian random solenoidal field with shell spectrum E(|k|) ~ spectrum(|k|).

    Built as the curl of a white-noise vector potential whose Fourier amplitude is shaped by
    sqrt(E(|k|))/|k|^2 (so |u_hat| ~ sqrt(E)/|k|, i.e. shell energy ~ E); solenoidal by
    construction.  Rescaled so that 1/2 <|u|^2> = e_tot, or so that the RMS of |u| is `rms`."""
    KX, KY, KZ = _wavenumbers(N)
    kabs = np.sqrt(KX * KX + KY * KY + KZ * KZ)
    with np.errstate(divide="ignore", invalid="ignore"):
        shape = np.where(kabs > 0, np.sqrt(np.maximum(spectrum(kabs), 0.0)) / (kabs * kabs), 0.0)
    nyq = (np.abs(KX) == N // 2) | (np.abs(KY) == N // 2) | (np.abs(KZ) == N // 2)
    shape[nyq] = 0.0
    shape[0, 0, 0] = 0.0
    A = []
    for c in range(3):
        w = normal01(seed, c, N * N * N).reshape(N, N, N)
        A.append(np.fft.rfftn(w) * shape)
        del w
    u = np.empty((3, N, N, N))
    u[0] = np.fft.irfftn(1j * (KY * A[2] - KZ * A[1]), s=(N, N, N), axes=(0, 1, 2))
    u[1] = np.fft.irfftn(1j * (KZ * A[0] - KX * A[2]), s=(N, N, N), axes=(0, 1, 2))
    u[2] = np.fft.irfftn(1j * (KX * A[1] - KY * A[0]), s=(N, N, N), axes=(0, 1, 2))
    e = 0.5 * float(np.mean(np.sum(u * u, axis=0)))
    if e_tot is not None:
        u *= np.sqrt(e_tot / e)
    elif rms is not None:
        u *= rms / np.sqrt(2.0 * e)
    return u


def taylor_green_perturbed(N: int = 32, seed: int = 1, amplitude: float = 1e-3) -> np.ndarray:
    """Config 1: Taylor-Green + band-limited (0 < |k| <= 4, flat amplitude) solenoidal noise of RMS `amplitude`."""
    flat = lambda k: np.where(k <= 4.0, k * k, 0.0)  # flat |u_hat| <=> shell energy ~ k^2
    return taylor_green_2d(N) + gaussian_field(N, seed, flat, rms=amplitude)


def gaussian_k4(N: int = 128, seed: int = 2) -> np.ndarray:
    """Config 2: E(k) ~ k^4 exp(-2 (k/4)^2), total energy 0.5."""
    return gaussian_field(N, seed, lambda k: k ** 4 * np.exp(-2.0 * (k / 4.0) ** 2), e_tot=0.5)


def gaussian_k53(N: int = 512, seed: int = 5) -> np.ndarray:
    """Config 5: E(k) ~ k^(-5/3) on 1 <= k <= N/3, zero elsewhere, total energy 0.5."""
    def spec(k):
        with np.errstate(divide="ignore"):
            return np.where((k >= 1.0) & (k <= N / 3.0), np.power(np.maximum(k, 1.0), -5.0 / 3.0), 0.0)
    return gaussian_field(N, seed, spec, e_tot=0.5)


def _shear_layer_plane(N: int, seed: int, rho: float, delta: float, nmodes: int):
    """(u1, u2)(x, y) of the perturbed doubly periodic shear layer, each [N][N]."""
    x = 2.0 * np.pi * np.arange(N) / N
    a = uniform01(seed, 100, 2 * nmodes) * delta
    b = uniform01(seed, 101, 2 * nmodes) * 2.0 * np.pi
    k = np.arange(1, nmodes + 1)
    s1 = np.sum(a[:nmodes, None] * np.sin(k[:, None] * x[None, :] + b[:nmodes, None]), axis=0)
    s2 = np.sum(a[nmodes:, None] * np.sin(k[:, None] * x[None, :] + b[nmodes:, None]), axis=0)
    X = x[:, None]
    Y = x[None, :]
    lower = np.tanh((Y - 0.5 * np.pi - s1[:, None]) / rho)
    upper = np.tanh((1.5 * np.pi + s2[:, None] - Y) / rho)
    return np.where(Y <= np.pi, lower, upper), 0.05 * np.sin(X) * np.ones_like(Y)


def shear_layer(N: int, seed: int, rho: float = 0.05, delta: float = 0.025, nmodes: int = 10) -> np.ndarray:
    """Configs 3/4: doubly periodic perturbed shear layer (BASELINE.json configs[2]).

    u1 = tanh((y - pi/2 - s1(x))/rho) for y <= pi, tanh((3pi/2 + s2(x) - y)/rho) for y > pi;
    u2 = 0.05 sin x; u3 = 0;  s_j(x) = sum_{k=1..10} a_jk sin(k x + b_jk), a ~ U[0,delta], b ~ U[0,2pi].
    Not solenoidal as written; `set_initial` projects it."""
    u1, u2 = _shear_layer_plane(N, seed, rho, delta, nmodes)
    u = np.zeros((3, N, N, N))
    u[0] = u1[:, :, None]
    u[1] = u2[:, :, None]
    return u


def shear_layer_ensemble(N: int = 128, batch: int = 32, seed0: int = 1000) -> np.ndarray:
    """Config 4: `batch` shear-layer samples, sample i uses seed seed0 + i.  [batch][3][N][N][N]."""
    return np.stack([shear_layer(N, seed0 + i) for i in range(batch)])


def taylor_green_3d_perturbed(N: int, seed: int, delta: float = 0.025) -> np.ndarray:
    """The paper's perturbed 3-D Taylor-Green vortex, eq. (6.1)-(6.3) with A = 1, B = -1, C = 0,
    on [0,2pi)^3 (the paper's 2 pi x is our x):
      u = cos x sin y sin z + e_0,  v = -sin x cos y sin z + e_1,  w = e_2,
      e_d = (1/8) sum_{(i,j,k) in {0,1}^3} d_{d,i,j,k} a_i(2x) a_j(2y) a_k(2z),  a_0 = sin, a_1 = cos,
      d_{d,i,j,k} ~ U[-delta, delta] i.i.d. (24 numbers per sample).  The perturbation is not solenoidal as written;
    `set_initial` projects it."""
    X, Y, Z = grid(N)
    d = (2.0 * uniform01(seed, 200, 24) - 1.0) * delta
    u = np.zeros((3, N, N, N))
    u[0] = np.cos(X) * np.sin(Y) * np.sin(Z)
    u[1] = -np.sin(X) * np.cos(Y) * np.sin(Z)
    a = lambda i, t: np.sin(t) if i == 0 else np.cos(t)
    for c in range(3):
        for i in range(2):
            for j in range(2):
                for k in range(2):
                    u[c] += 0.125 * d[((c * 2 + i) * 2 + j) * 2 + k] * a(i, 2 * X) * a(j, 2 * Y) * a(k, 2 * Z)
    return u


def cylindrical_shear(N: int, seed: int, rho: float = 0.05, delta: float = 0.025, nmodes: int = 10) -> np.ndarray:
    """The paper's cylindrical shear flow, eq. (6.4)-(6.6), in unit coordinates X = x/2pi etc.:
      u = tanh(2 pi (r - 0.25)/rho)  (rho = 0: the sign function of eq. 6.6),  v = w = 0,
      r^2 = (Y - 0.5 + s_y(X))^2 + (Z - 0.5 + s_z(X))^2,  s(X) = delta sum_{k=1..p} a_k sin(2 pi k X - b_k),
      a_k ~ U[0,1], b_k ~ U[0,2pi] i.i.d., p = 10, delta = 0.025."""
    xs = np.arange(N) / N
    a = uniform01(seed, 210, 2 * nmodes)
    b = uniform01(seed, 211, 2 * nmodes) * 2.0 * np.pi
    k = np.arange(1, nmodes + 1)
    sy = delta * np.sum(a[:nmodes, None] * np.sin(2.0 * np.pi * k[:, None] * xs[None, :] - b[:nmodes, None]), axis=0)
    sz = delta * np.sum(a[nmodes:, None] * np.sin(2.0 * np.pi * k[:, None] * xs[None, :] - b[nmodes:, None]), axis=0)
    Y = xs[None, :, None]
    Z = xs[None, None, :]
    r = np.sqrt((Y - 0.5 + sy[:, None, None]) ** 2 + (Z - 0.5 + sz[:, None, None]) ** 2)
    u = np.zeros((3, N, N, N))
    u[0] = np.where(r <= 0.25, -1.0, 1.0) if rho == 0 else np.tanh(2.0 * np.pi * (r - 0.25) / rho)
    return u


def checksum(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:16]


# ------------------------------------------------------------------------------------------------ two-dimensional inputs
# (the paper validates its 2-D solver on the Taylor-Green vortex and the vortex patch)
def grid2(N: int):
    x = 2.0 * np.pi * np.arange(N) / N
    return np.meshgrid(x, x, indexing="ij")


def taylor_green_2d_plane(N: int) -> np.ndarray:
    """2-D Taylor-Green vortex u = (sin x cos y, -cos x sin y) on [0,2pi)^2: u[2][N][N]."""
    X, Y = grid2(N)
    return np.stack([np.sin(X) * np.cos(Y), -np.cos(X) * np.sin(Y)])


def gaussian_field_2d(N: int, seed: int, spectrum, e_tot: float = 0.5) -> np.ndarray:
    """Band-limited Gaussian random solenoidal 2-D field with ring spectrum E(|k|) ~ spectrum(|k|): the curl of a white-noise
    stream function shaped by sqrt(E)/|k|^(3/2) (so |u_hat| ~ sqrt(E/|k|), ring energy ~ E); rescaled to 1/2 <|u|^2> = e_tot."""
    k = np.fft.fftfreq(N, 1.0 / N)
    KX, KY = np.meshgrid(k, np.fft.rfftfreq(N, 1.0 / N), indexing="ij")
    kabs = np.sqrt(KX * KX + KY * KY)
    with np.errstate(divide="ignore", invalid="ignore"):
        shape = np.where(kabs > 0, np.sqrt(np.maximum(spectrum(kabs), 0.0)) / kabs ** 1.5, 0.0)
    shape[(np.abs(KX) == N // 2) | (np.abs(KY) == N // 2)] = 0.0
    psi = np.fft.rfft2(normal01(seed, 0, N * N).reshape(N, N)) * shape
    u = np.stack([np.fft.irfft2(1j * KY * psi, s=(N, N)), np.fft.irfft2(-1j * KX * psi, s=(N, N))])
    return u * np.sqrt(e_tot / (0.5 * float(np.mean(np.sum(u * u, axis=0)))))


def vortex_patch(N: int, seed: int = 0, radius: float = 1.0, delta: float = 0.0) -> np.ndarray:
    """Vortex patch ([19]): vorticity 1 inside a disc of the given radius centred at (pi, pi) (optionally
    displaced by a seeded offset of size delta), minus its mean so that it is the curl of a periodic velocity; the velocity
    is obtained from the stream function -Laplace psi = omega with numpy.fft.  u[2][N][N]."""
    X, Y = grid2(N)
    off = (2.0 * uniform01(seed, 300, 2) - 1.0) * delta
    om = ((X - np.pi - off[0]) ** 2 + (Y - np.pi - off[1]) ** 2 <= radius ** 2).astype(np.float64)
    om -= om.mean()
    k = np.fft.fftfreq(N, 1.0 / N)
    KX, KY = np.meshgrid(k, np.fft.rfftfreq(N, 1.0 / N), indexing="ij")
    k2 = KX * KX + KY * KY
    k2[0, 0] = 1.0
    psi = np.fft.rfft2(om) / k2
    psi[0, 0] = 0.0
    return np.stack([np.fft.irfft2(1j * KY * psi, s=(N, N)), np.fft.irfft2(-1j * KX * psi, s=(N, N))])


def shear_layer_2d(N: int, seed: int, rho: float = 0.05, delta: float = 0.025, nmodes: int = 10) -> np.ndarray:
    """The doubly periodic perturbed shear layer of configs 3/4 as a genuinely two-dimensional field: u[2][N][N]."""
    return np.stack(_shear_layer_plane(N, seed, rho, delta, nmodes))
