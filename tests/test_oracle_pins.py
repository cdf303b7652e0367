"""Pins P0-P11 for the CPU oracle: every check compares the oracle with
something OTHER than itself -- an O(n^2)/O(N^6) brute force written here in numpy, numpy.fft as a
library special case, closed forms, invariants of the equations, or values fixed by the paper.
All of them run on CPU:  python -m pytest tests -m "not gpu".
"""
import os

import numpy as np
import pytest

from paper_2401_09843_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def read_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            parts = line.split()
            out[parts[0]] = [float(v) for v in parts[1:]]
    return out


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def wavenumbers(N):
    k = np.fft.fftfreq(N, 1.0 / N)
    kz = np.arange(N // 2 + 1, dtype=float)
    return np.meshgrid(k, k, kz, indexing="ij")


def half_weights(N):
    w = np.full(N // 2 + 1, 2.0)
    w[0] = 1.0
    return w[None, None, :]


def random_state(oracle, N, seed, kmax=None):
    kmax = N / 3.0 if kmax is None else kmax
    u = inputs.gaussian_field(N, seed, lambda k: np.where(k <= kmax, k ** 2 * np.exp(-(k / 3.0) ** 2), 0.0), e_tot=0.5)
    return oracle.set_initial(N, u)


def full_state(oracle, N, seed):
    """Random solenoidal state exciting EVERY active mode (up to |k_i| = N/2-1), for aliasing-sensitive pins."""
    u = inputs.gaussian_field(N, seed, lambda k: 1.0 / (1.0 + k), e_tot=0.5)
    return oracle.set_initial(N, u)


# ------------------------------------------------------------------------------------------- P0
@pytest.mark.parametrize("n", [2, 3, 4, 6, 8, 12, 16, 24, 48, 96, 192])
@pytest.mark.parametrize("sign", [-1, 1])
def test_p0_fft_vs_direct_dft(oracle, n, sign):
    x = inputs.normal01(7, n, 2 * n).view(np.complex128)
    j = np.arange(n)
    W = np.exp(sign * 2j * np.pi * (np.outer(j, j) % n) / n)   # the definition, written out here (argument reduced)
    want = W @ x
    assert rel(oracle.fft1d(x, sign), want) < 1e-14
    assert rel(oracle.dft1d(x, sign), want) < 1e-14
    lib = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n  # library routine as a special case
    assert rel(oracle.fft1d(x, sign), lib) < 1e-14


@pytest.mark.parametrize("n", [4, 6, 8])
def test_p0_fft3d_vs_bruteforce(oracle, n):
    a = inputs.normal01(11, n, 2 * n ** 3).view(np.complex128).reshape(n, n, n)
    j = np.arange(n)
    W = np.exp(-2j * np.pi * (np.outer(j, j) % n) / n)
    want = np.einsum("ai,bj,ck,ijk->abc", W, W, W, a)        # O(N^6)-equivalent direct 3-D DFT
    assert rel(oracle.fft3d(a, -1), want) < 1e-14
    assert rel(oracle.fft3d(oracle.fft3d(a, -1), +1) / n ** 3, a) < 1e-14


def test_p0_set_initial_get_fields_roundtrip(oracle):
    N = 12
    u = inputs.gaussian_field(N, 3, lambda k: np.where(k <= 4, 1.0, 0.0), e_tot=0.5)
    uh = oracle.set_initial(N, u)
    # a band-limited solenoidal field is reproduced exactly; coefficients are the normalised DFT
    assert rel(oracle.get_fields(N, uh), u) < 1e-13
    want = np.fft.rfftn(u, axes=(1, 2, 3)) / N ** 3
    want[:, N // 2, :, :] = 0
    want[:, :, N // 2, :] = 0
    want[:, :, :, N // 2] = 0
    assert rel(uh, want) < 1e-13


def test_p0_set_initial_projects(oracle):
    N = 8
    u = inputs.normal01(5, 0, 3 * N ** 3).reshape(3, N, N, N)   # NOT solenoidal
    uh = oracle.set_initial(N, u)
    KX, KY, KZ = wavenumbers(N)
    div = KX * uh[0] + KY * uh[1] + KZ * uh[2]
    assert np.abs(div).max() < 1e-14
    # mean kept, Nyquist zero
    assert abs(uh[0, 0, 0, 0] - u[0].mean()) < 1e-15
    assert np.all(uh[:, N // 2] == 0) and np.all(uh[:, :, N // 2] == 0) and np.all(uh[:, :, :, N // 2] == 0)
    # projector written out: u - k (k.u)/k^2 of the plain normalised transform
    raw = np.fft.rfftn(u, axes=(1, 2, 3)) / N ** 3
    k2 = KX ** 2 + KY ** 2 + KZ ** 2
    k2[0, 0, 0] = 1.0
    ku = (KX * raw[0] + KY * raw[1] + KZ * raw[2]) / k2
    want = np.stack([raw[0] - KX * ku, raw[1] - KY * ku, raw[2] - KZ * ku])
    want[:, N // 2] = 0
    want[:, :, N // 2] = 0
    want[:, :, :, N // 2] = 0
    # (projection and Nyquist-zeroing commute only if zeroing is done first: do the same here)
    raw[:, N // 2] = 0
    raw[:, :, N // 2] = 0
    raw[:, :, :, N // 2] = 0
    ku = (KX * raw[0] + KY * raw[1] + KZ * raw[2]) / k2
    want = np.stack([raw[0] - KX * ku, raw[1] - KY * ku, raw[2] - KZ * ku])
    assert rel(uh, want) < 1e-13


# ------------------------------------------------------------------------------------------- P1
def direct_convolution_rhs(N, uh):
    """N_hat_k = P_k[ -i sum_j k_j sum_{p+q=k; p,q in K_N} u_i(p) u_j(q) ]  -- O(N^6), no FFT, no padding."""
    K = N // 2 - 1
    n = 2 * K + 1
    F = np.zeros((3, n, n, n), dtype=np.complex128)          # full spectrum, index k + K
    for ix in range(N):
        kx = ix if ix < N // 2 else ix - N
        if ix == N // 2:
            continue
        for iy in range(N):
            ky = iy if iy < N // 2 else iy - N
            if iy == N // 2:
                continue
            for kz in range(0, N // 2):
                v = uh[:, ix, iy, kz]
                F[:, kx + K, ky + K, kz + K] = v
                if kz > 0:
                    F[:, -kx + K, -ky + K, -kz + K] = np.conj(v)
    conv = np.zeros((3, 3, n, n, n), dtype=np.complex128)     # sum_{p+q=k} u_i(p) u_j(q), k in K_N only
    for px in range(-K, K + 1):
        for py in range(-K, K + 1):
            for pz in range(-K, K + 1):
                up = F[:, px + K, py + K, pz + K]
                if not np.any(up):
                    continue
                # q = k - p must lie in [-K, K]: k in [max(-K, p-K), min(K, p+K)]
                lo = [max(-K, p - K) for p in (px, py, pz)]
                hi = [min(K, p + K) for p in (px, py, pz)]
                ks = tuple(slice(l + K, h + K + 1) for l, h in zip(lo, hi))
                qs = tuple(slice(l - p + K, h - p + K + 1) for l, h, p in zip(lo, hi, (px, py, pz)))
                conv[(slice(None), slice(None)) + ks] += up[:, None, None, None, None] * F[(None, slice(None)) + qs]
    out = np.zeros((3, N, N, N // 2 + 1), dtype=np.complex128)
    for ix in range(N):
        if ix == N // 2:
            continue
        kx = ix if ix < N // 2 else ix - N
        for iy in range(N):
            if iy == N // 2:
                continue
            ky = iy if iy < N // 2 else iy - N
            for kz in range(N // 2):
                k = np.array([kx, ky, kz], dtype=float)
                k2 = k @ k
                if k2 == 0:
                    continue
                B = conv[:, :, kx + K, ky + K, kz + K]
                b = -1j * (B @ k)
                out[:, ix, iy, kz] = b - k * (k @ b) / k2
    return out


@pytest.mark.parametrize("N", [4, 6, 8])
def test_p1_rhs_vs_direct_convolution(oracle, N):
    uh = full_state(oracle, N, 20 + N)
    parts = oracle.rhs_parts(N, oracle.Params(), uh)
    want = direct_convolution_rhs(N, uh)
    assert np.linalg.norm(want) > 1e-3
    assert rel(parts["n"], want) < 1e-13
    assert rel(parts["r"], want) < 1e-13        # no dissipation -> R = N


# ------------------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("name", ["taylor_green", "abc"])
def test_p2_gradient_nonlinearity_projects_to_zero(oracle, name):
    N = 16
    u = inputs.taylor_green_2d(N) if name == "taylor_green" else inputs.abc_flow(N)
    uh = oracle.set_initial(N, u)
    parts = oracle.rhs_parts(N, oracle.Params(), uh)
    nb = np.linalg.norm(parts["b"])
    assert nb > 1e-2                                   # the unprojected term is NOT small ...
    assert np.linalg.norm(parts["n"]) / nb < 1e-14     # ... but it is a pure gradient
    # Taylor-Green coefficients are +-1/4 (reading A2: normalised coefficients)
    if name == "taylor_green":
        assert abs(abs(uh[0, 1, 1, 0]) - 0.25) < 1e-15


# ------------------------------------------------------------------------------------------- P3
def test_p3_rk3_decay_closed_form(oracle):
    g = read_golden("rk3_decay_taylor_green.txt")
    nu, dt, steps = g["nu"][0], g["dt"][0], int(g["steps"][0])
    z = -nu * g["k2"][0] * dt
    assert abs((1 + z + z * z / 2 + z ** 3 / 6) - g["g"][0]) < 2e-16       # the fixture is the polynomial
    N = 16
    uh0 = oracle.set_initial(N, inputs.taylor_green_2d(N))
    uh = uh0.copy()
    p = oracle.Params(nu=nu)
    for _ in range(steps):
        uh = oracle.step(N, p, uh, dt)
    assert rel(uh, g["g_pow_steps"][0] * uh0) < 1e-14
    one = oracle.step(N, p, uh0, dt)
    assert rel(one, g["g"][0] * uh0) < 1e-15
    # ABC flow: |k|^2 = 1, exercises the z axis
    a0 = oracle.set_initial(N, inputs.abc_flow(N))
    a = a0.copy()
    for _ in range(5):
        a = oracle.step(N, p, a, dt)
    z = -nu * dt
    assert rel(a, (1 + z + z * z / 2 + z ** 3 / 6) ** 5 * a0) < 1e-14


# ------------------------------------------------------------------------------------------- P4
@pytest.mark.parametrize("N", [16, 32])
def test_p4_energy_identity(oracle, N):
    uh = full_state(oracle, N, 40 + N)
    nh = oracle.rhs_parts(N, oracle.Params(), uh)["n"]
    w = half_weights(N)
    s = np.sum(w * np.real(np.conj(uh) * nh))
    scale = np.sum(w * np.abs(uh) * np.abs(nh))
    assert scale > 1e-6
    assert abs(s) < 1e-13 * scale


# ------------------------------------------------------------------------------------------- P5
def test_p5_rhs_is_solenoidal_and_masked(oracle):
    N = 16
    uh = full_state(oracle, N, 50)
    r = oracle.rhs(N, oracle.Params(nu=0.02, eps=0.05, s=1.0), uh)
    KX, KY, KZ = wavenumbers(N)
    div = KX * r[0] + KY * r[1] + KZ * r[2]
    kn = np.sqrt(KX ** 2 + KY ** 2 + KZ ** 2)
    assert np.abs(div).max() < 1e-14 * max(1.0, (kn * np.abs(r).sum(0)).max())
    assert np.all(r[:, N // 2] == 0) and np.all(r[:, :, N // 2] == 0) and np.all(r[:, :, :, N // 2] == 0)
    assert np.all(r[:, 0, 0, 0] == 0)


# ------------------------------------------------------------------------------------------- P6
def test_p6_galilean_shift(oracle):
    N = 16
    uh = full_state(oracle, N, 60)
    U = np.array([0.3, -0.7, 0.45])
    shifted = uh.copy()
    shifted[:, 0, 0, 0] += U
    n0 = oracle.rhs_parts(N, oracle.Params(), uh)["n"]
    n1 = oracle.rhs_parts(N, oracle.Params(), shifted)["n"]
    KX, KY, KZ = wavenumbers(N)
    want = -1j * (KX * U[0] + KY * U[1] + KZ * U[2])[None] * uh
    want[:, 0, 0, 0] = 0
    assert rel(n1 - n0, want) < 1e-13


# ------------------------------------------------------------------------------------------- P7
def test_p7_independent_of_padding(oracle):
    N = 12
    uh = full_state(oracle, N, 70)
    a = oracle.rhs_parts(N, oracle.Params(), uh, M=3 * N // 2)["n"]
    b = oracle.rhs_parts(N, oracle.Params(), uh, M=2 * N)["n"]
    assert rel(a, b) < 1e-13


# ------------------------------------------------------------------------------------------- P8
def test_p8_energy_spectrum(oracle):
    N = 16
    u = inputs.gaussian_field(N, 80, lambda k: np.where(k <= 5, k ** 2, 0.0), e_tot=0.37)
    uh = oracle.set_initial(N, u)
    E = oracle.energy_spectrum(N, uh, N)
    assert abs(E.sum() - 0.5 * np.mean(np.sum(u * u, axis=0))) < 1e-14
    assert abs(E.sum() - 0.37) < 1e-13
    assert np.all(E[7:] < 1e-30)                     # band limit |k| <= 5 (round-off only above)
    tg = oracle.set_initial(N, inputs.taylor_green_2d(N))
    E = oracle.energy_spectrum(N, tg, 8)
    want = np.zeros(8)
    want[1] = 0.25                                   # |k| = sqrt 2 -> bin 1;  1/2 <|u|^2> = 1/4
    assert np.abs(E - want).max() < 1e-15
    # single-shell input lands in exactly one bin
    one = inputs.gaussian_field(N, 81, lambda k: np.where((k >= 2.5) & (k < 3.5), 1.0, 0.0), e_tot=0.2)
    E = oracle.energy_spectrum(N, oracle.set_initial(N, one), N)
    assert abs(E[3] - 0.2) < 1e-14 and abs(E.sum() - E[3]) < 1e-15


def test_p8b_enstrophy_spectrum(oracle):
    """Reading A20 (PAPER.md:L163 names the writer only).  Pins: Taylor-Green has omega = (0, 0, 2 sin x sin y), so
    1/2 <|omega|^2> = 1/2 lands in bin 1; a Beltrami (ABC) field has curl u = u, so Z = E bin by bin; a gradient
    field has no vorticity (this separates |k x u|^2 from the solenoidal shortcut |k|^2 |u|^2); and sum_K Z equals
    1/2 <|curl u|^2> with the curl taken by centred spectral differences written here with numpy.fft."""
    N = 16
    tg = oracle.set_initial(N, inputs.taylor_green_2d(N))
    Z = oracle.enstrophy_spectrum(N, tg, 8)
    want = np.zeros(8)
    want[1] = 0.5
    assert np.abs(Z - want).max() < 1e-15
    x = 2 * np.pi * np.arange(N) / N
    X, Y, Zc = np.meshgrid(x, x, x, indexing="ij")
    A, B, C = 0.7, -0.4, 1.1
    abc = np.stack([A * np.sin(Zc) + C * np.cos(Y), B * np.sin(X) + A * np.cos(Zc), C * np.sin(Y) + B * np.cos(X)])
    ua = oracle.set_initial(N, abc)
    assert np.abs(oracle.enstrophy_spectrum(N, ua, N) - oracle.energy_spectrum(N, ua, N)).max() < 1e-14
    # gradient field: u = grad(phi), written straight into the spectral state (set_initial would project it away)
    rng = np.random.default_rng(82)
    phi = rng.standard_normal((N, N, N))
    ph = np.fft.rfftn(phi) / N ** 3
    k = np.fft.fftfreq(N, 1.0 / N)
    kz = np.arange(N // 2 + 1.0)
    g = np.stack([1j * k[:, None, None] * ph, 1j * k[None, :, None] * ph, 1j * kz[None, None, :] * ph])
    g[:, N // 2] = 0; g[:, :, N // 2] = 0; g[:, :, :, N // 2] = 0
    assert oracle.energy_spectrum(N, g, N).sum() > 1e-3
    assert oracle.enstrophy_spectrum(N, g, N).max() < 1e-28
    # Parseval against a curl evaluated with numpy.fft on the physical field
    u = inputs.gaussian_field(N, 83, lambda kk: np.where(kk <= 5, kk ** 2, 0.0), e_tot=0.37)
    uh = oracle.set_initial(N, u)
    U = np.fft.fftn(u, axes=(1, 2, 3))
    KX, KY, KZ = np.meshgrid(k, k, k, indexing="ij")
    for K in (KX, KY, KZ):
        K[np.abs(K) == N // 2] = 0.0   # the oracle state carries no Nyquist planes
    W = np.stack([KY * U[2] - KZ * U[1], KZ * U[0] - KX * U[2], KX * U[1] - KY * U[0]]) * 1j
    w = np.real(np.fft.ifftn(W, axes=(1, 2, 3)))
    assert abs(oracle.enstrophy_spectrum(N, uh, N).sum() - 0.5 * np.mean(np.sum(w * w, axis=0))) < 1e-12


# ------------------------------------------------------------------------------------------- P9
def test_p9_structure_function_identity(oracle):
    N = 12
    uh = full_state(oracle, N, 90)
    S = oracle.structure_function(N, uh)
    KX, KY, KZ = wavenumbers(N)
    e = np.sum(np.abs(uh) ** 2, axis=0) * half_weights(N)
    dx = 2 * np.pi / N
    want = np.array([np.sum(e * 2 * ((1 - np.cos(KX * l * dx)) + (1 - np.cos(KY * l * dx)) + (1 - np.cos(KZ * l * dx)))) / 3
                     for l in range(1, N // 2 + 1)])
    assert np.abs(S / want - 1).max() < 1e-12


def test_p9b_structure_function_order_p(oracle):
    """S_p (reading A15 extended to p != 2): p = 2 is S2; a single shear mode u = (0, a sin(kx), 0) has
    S_p(l) = (1/3) (2a |sin(k l dx / 2)|)^p <cos^p> with <cos^4> = 3/8, <cos^6> = 5/16 (exact on the grid);
    odd and fractional orders against increments taken with numpy.roll."""
    N = 16
    uh = full_state(oracle, N, 91)
    assert np.abs(oracle.structure_function_p(N, uh, 2.0) / oracle.structure_function(N, uh) - 1).max() < 1e-13
    a, k = 0.8, 2
    x = 2 * np.pi * np.arange(N) / N
    u = np.zeros((3, N, N, N))
    u[1] = a * np.sin(k * x)[:, None, None]
    um = oracle.set_initial(N, u)
    l = np.arange(1, N // 2 + 1)
    for p, c in ((4.0, 3.0 / 8.0), (6.0, 5.0 / 16.0)):
        want = (2 * a * np.abs(np.sin(k * l * (2 * np.pi / N) / 2))) ** p * c / 3.0
        assert np.abs(oracle.structure_function_p(N, um, p) - want).max() < 1e-13
    phys = oracle.get_fields(N, uh)
    for p in (1.0, 3.0, 2.5):
        want = np.array([sum(np.mean(np.sum((np.roll(phys, -ll, axis=d + 1) - phys) ** 2, axis=0) ** (p / 2)) for d in range(3)) / 3.0
                         for ll in l])
        assert np.abs(oracle.structure_function_p(N, uh, p) / want - 1).max() < 1e-12


# ------------------------------------------------------------------------------------------- P10
def test_p10_third_order_in_time(oracle):
    N = 8
    uh0 = random_state(oracle, N, 100, kmax=2.5)
    p = oracle.Params(nu=0.05)
    T = 0.4

    def run(nsteps):
        u = uh0.copy()
        for _ in range(nsteps):
            u = oracle.step(N, p, u, T / nsteps)
        return u

    ref = run(128)
    e1 = np.linalg.norm(run(4) - ref)
    e2 = np.linalg.norm(run(8) - ref)
    assert 7.0 < e1 / e2 < 9.0


# ------------------------------------------------------------------------------------------- P11
@pytest.mark.parametrize("s", [1.0, 1.5])
def test_p11_hyperviscous_single_mode(oracle, s):
    N, eps = 16, 0.05
    kk = 6                                      # |k| = 6 > m_N = sqrt(16) = 4
    x = 2 * np.pi * np.arange(N) / N
    u = np.zeros((3, N, N, N))
    u[1] = np.cos(kk * x)[:, None, None]         # u = (0, cos 6x, 0): u.grad u = 0, so N_hat = 0
    uh0 = oracle.set_initial(N, u)
    p = oracle.Params(eps=eps, s=s)
    # closed form written out (readings A5, A6): eps_N = eps/N^(2s-1), Q = 1 - (m/|k|)^((2s-1)/theta), theta = 1/2
    d = eps / N ** (2 * s - 1) * kk ** (2 * s) * (1 - (np.sqrt(N) / kk) ** ((2 * s - 1) / 0.5))
    if s == 1.0:
        assert abs(d - eps / N * (kk * kk - N)) < 1e-15
    assert abs(oracle.dissipation(N, p, float(kk * kk)) - d) < 1e-15
    dt, n = 0.01, 7
    uh = uh0.copy()
    for _ in range(n):
        uh = oracle.step(N, p, uh, dt)
    z = -d * dt
    assert rel(uh, (1 + z + z * z / 2 + z ** 3 / 6) ** n * uh0) < 1e-14
    # below the cutoff nothing is damped
    assert oracle.dissipation(N, p, 9.0) == 0.0
    assert oracle.dissipation(N, oracle.Params(eps=eps, s=s, q_sharp=1), 36.0) == pytest.approx(eps / N ** (2 * s - 1) * kk ** (2 * s), rel=1e-15)


# ------------------------------------------------------------------------------------------- P12
@pytest.mark.parametrize("N", [6, 8])
def test_p12_rhs_at_modes_vs_direct_convolution(oracle, N):
    """orc_rhs_at_modes (used for sampled parity at 256^3 / 512^3) against the test's own O(N^6) sum, every mode."""
    uh = full_state(oracle, N, 40 + N)
    modes = np.array([(ix, iy, iz) for ix in range(N) for iy in range(N) for iz in range(N // 2 + 1)], dtype=np.int32)
    got = oracle.rhs_at_modes(N, oracle.Params(), uh, modes)
    want = direct_convolution_rhs(N, uh)
    assert rel(got.T.reshape(want.shape), want) < 1e-13
    nyq = (modes[:, 0] == N // 2) | (modes[:, 1] == N // 2) | (modes[:, 2] == N // 2)
    assert np.all(got[nyq] == 0) and np.all(got[0] == 0)


@pytest.mark.parametrize("N,s", [(12, 1.0), (32, 1.0), (32, 1.5)])
def test_p12_rhs_at_modes_vs_stepwise_oracle(oracle, N, s):
    """... and against the step-by-step pseudo-spectral RHS with dissipation, on sampled modes incl. the box corners."""
    uh = full_state(oracle, N, 60 + N)
    p = oracle.Params(nu=0.01, eps=0.05, s=s)
    r = oracle.rhs(N, p, uh)
    rng = np.random.default_rng(N)
    K = N // 2 - 1
    modes = np.concatenate([
        np.stack([rng.integers(0, N, 40), rng.integers(0, N, 40), rng.integers(0, N // 2 + 1, 40)], axis=1),
        np.array([(K, K, K), (N - K, N - K, K), (K, N - K, 0), (0, 0, 1), (1, 0, 0), (0, 0, 0), (N // 2, 1, 1), (1, 1, N // 2)]),
    ]).astype(np.int32)
    got = oracle.rhs_at_modes(N, p, uh, modes)
    want = np.stack([r[:, ix, iy, iz] for ix, iy, iz in modes])
    assert np.abs(got - want).max() < 1e-13 * np.abs(r).max()
    assert np.linalg.norm(want) > 1e-3


def test_max_velocity_and_padding(oracle):
    N = 8
    uh = oracle.set_initial(N, inputs.taylor_green_2d(N))
    # |u|^2 = sin^2 x cos^2 y + cos^2 x sin^2 y <= 1, attained at x = pi/2, y = 0 (on the 12-point padded grid too)
    assert abs(oracle.max_velocity(N, uh) - 1.0) < 1e-14
    assert abs(oracle.rhs_parts(N, oracle.Params(), uh)["umax"] - 1.0) < 1e-14


def _both_umax(oracle, N, uh):
    a = oracle.max_velocity(N, uh)
    b = oracle.rhs_parts(N, oracle.Params(), uh)["umax"]
    assert a == b          # the two entry points evaluate the same definition
    return a


def test_p13_max_velocity_is_euclidean_norm_of_all_three_components(oracle):
    """Pin of reading A10 / SURVEY.md 8(c) item 10, part (i): a constant field U has umax = |U|_2 exactly.  Fails for a
    dropped component (0.3, -0.7 only -> 0.7616), for the max-component norm (0.7) and for the 1-norm (1.45)."""
    N = 8
    U = np.array([0.3, -0.7, 0.45])
    uh = np.zeros(oracle.spectral_shape(N), dtype=np.complex128)
    uh[:, 0, 0, 0] = U
    assert abs(_both_umax(oracle, N, uh) - np.sqrt(0.09 + 0.49 + 0.2025)) < 1e-15
    # and with the third component alone (a field whose u1 = u2 = 0)
    uh[:2] = 0
    assert abs(_both_umax(oracle, N, uh) - 0.45) < 1e-15


def test_p13_max_velocity_is_taken_on_the_padded_grid(oracle):
    """Part (ii): u = (0, 0, cos(x - 2 pi/12)) at N = 8.  Its maximum 1 is attained at x = 2 pi/12, a point of the 12-point
    padded grid that is NOT on the 8-point grid, where the maximum is cos(pi/12) = 0.96593 (at x = 0 and x = 2 pi/8).
    Fails when the maximum is taken over the N grid instead of the M = 3N/2 grid."""
    N = 8
    x = 2 * np.pi * np.arange(N) / N
    u = np.zeros((3, N, N, N))
    u[2] = np.cos(x - 2 * np.pi / 12)[:, None, None]
    assert abs(np.abs(u[2]).max() - np.cos(np.pi / 12)) < 1e-15
    uh = oracle.set_initial(N, u)               # a z-directed shear depending on x only is solenoidal: unchanged
    assert abs(_both_umax(oracle, N, uh) - 1.0) < 1e-14
    # the same along y and z (u1 depending on y, u2 depending on z) -- catches an axis handled on the wrong grid
    u = np.zeros((3, N, N, N))
    u[0] = np.cos(x - 2 * np.pi / 12)[None, :, None]
    assert abs(_both_umax(oracle, N, oracle.set_initial(N, u)) - 1.0) < 1e-14
    u = np.zeros((3, N, N, N))
    u[1] = np.cos(x - 2 * np.pi / 12)[None, None, :]
    assert abs(_both_umax(oracle, N, oracle.set_initial(N, u)) - 1.0) < 1e-14


@pytest.mark.parametrize("N", [8, 12, 16])
def test_p13_max_velocity_vs_zero_padded_numpy_irfftn(oracle, N):
    """Part (iii): a random solenoidal state exciting every active mode, evaluated on the M = 3N/2 grid by a zero-padded
    numpy.fft.irfftn written here (library routine as a second witness), Euclidean norm, maximum over the grid."""
    uh = full_state(oracle, N, 900 + N)
    M = 3 * N // 2
    pad = np.zeros((3, M, M, M // 2 + 1), dtype=np.complex128)
    K = N // 2 - 1
    for ix in range(N):
        kx = ix if ix < N // 2 else ix - N
        if abs(kx) > K:
            continue
        for iy in range(N):
            ky = iy if iy < N // 2 else iy - N
            if abs(ky) > K:
                continue
            pad[:, kx % M, ky % M, :K + 1] = uh[:, ix, iy, :K + 1]
    phys = np.fft.irfftn(pad, s=(M, M, M), axes=(1, 2, 3)) * M ** 3    # unnormalised synthesis sum_k u_hat e^{ikx}
    want = np.sqrt((phys ** 2).sum(axis=0)).max()
    got = _both_umax(oracle, N, uh)
    assert abs(got - want) < 1e-13 * want
    # the maximum over the N grid differs (so the pin discriminates) and so do the other norms
    coarse = np.sqrt((oracle.get_fields(N, uh) ** 2).sum(axis=0)).max()
    assert abs(coarse - want) > 1e-6 * want
    assert abs(np.abs(phys).max() - want) > 1e-6 * want
