"""Pins Q0-Q8 of the TWO-DIMENSIONAL CPU oracle (oracle/ns2d_oracle.cpp): every check compares it with
something other than itself -- numpy.fft, an O(N^4) direct convolution written here, closed forms, invariants of the 2-D
equations (energy AND enstrophy), and the independently pinned THREE-dimensional oracle run on z-independent data (the
paper's own validation idea).  CPU only:  python -m pytest tests -m "not gpu".
"""
import numpy as np
import pytest

from paper_2401_09843_b200 import inputs


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def wavenumbers(N):
    return np.meshgrid(np.fft.fftfreq(N, 1.0 / N), np.arange(N // 2 + 1, dtype=float), indexing="ij")


def half_weights(N):
    w = np.full(N // 2 + 1, 2.0)
    w[0] = 1.0
    return w[None, :]


def full_state(o2, N, seed):
    """Random solenoidal 2-D state exciting every active mode."""
    return o2.set_initial(N, inputs.gaussian_field_2d(N, seed, lambda k: 1.0 / (1.0 + k)))


def full_spectrum(uh, N):
    """[2][N][N] full complex spectrum indexed by (kx mod N, ky mod N) from the half spectrum (ky = 0 line: Hermitian part)."""
    F = np.zeros((2, N, N), dtype=np.complex128)
    K = N // 2 - 1
    for kx in range(-K, K + 1):
        for ky in range(-K, K + 1):
            if ky > 0:
                v = uh[:, kx % N, ky]
            elif ky < 0:
                v = np.conj(uh[:, (-kx) % N, -ky])
            else:
                v = 0.5 * (uh[:, kx % N, 0] + np.conj(uh[:, (-kx) % N, 0]))
            F[:, kx % N, ky % N] = v
    return F


# ------------------------------------------------------------------------------------------- Q0
@pytest.mark.parametrize("n", [4, 6, 12, 16, 24, 48])
def test_q0_fft2d_vs_numpy(oracle2d, n):
    a = inputs.normal01(3, n, 2 * n * n).view(np.complex128).reshape(n, n)
    assert rel(oracle2d.fft2d(a, -1), np.fft.fft2(a)) < 1e-14
    assert rel(oracle2d.fft2d(a, +1), np.fft.ifft2(a) * n * n) < 1e-14


@pytest.mark.parametrize("N", [8, 12, 16])
def test_q0_set_initial_and_get_fields(oracle2d, N):
    u = inputs.gaussian_field_2d(N, 5, lambda k: 1.0 / (1.0 + k)) + 0.3 * inputs.normal01(N, 9, 2 * N * N).reshape(2, N, N)
    uh = oracle2d.set_initial(N, u)
    KX, KY = wavenumbers(N)
    ref = np.fft.rfft2(u, axes=(1, 2)) / N ** 2
    ref[:, N // 2] = 0
    ref[:, :, N // 2] = 0
    k2 = KX ** 2 + KY ** 2
    k2[0, 0] = 1.0
    ku = (KX * ref[0] + KY * ref[1]) / k2
    ku[0, 0] = 0
    ref = ref - np.stack([KX * ku, KY * ku])
    assert rel(uh, ref) < 1e-14
    assert np.abs(KX * uh[0] + KY * uh[1]).max() < 1e-14
    # get_fields is the real part of the synthesis of the half spectrum
    back = np.fft.irfft2(uh, s=(N, N), axes=(1, 2)) * N ** 2
    assert rel(oracle2d.get_fields(N, uh), back) < 1e-13


# ------------------------------------------------------------------------------------------- Q1
@pytest.mark.parametrize("N", [4, 6, 8, 12, 16])
def test_q1_rhs_vs_direct_convolution(oracle2d, N):
    """N_hat(k) = P_k[-i sum_j k_j sum_{p+q=k; p,q in K_N} u_i(p) u_j(q)], O(N^4), written out here."""
    uh = full_state(oracle2d, N, 40 + N)
    F = full_spectrum(uh, N)
    K = N // 2 - 1
    got = oracle2d.rhs_parts(N, oracle2d.Params(), uh)
    want_b = np.zeros_like(uh)
    want_n = np.zeros_like(uh)
    for kx in range(-K, K + 1):
        for ky in range(0, K + 1):
            B = np.zeros((2, 2), dtype=np.complex128)
            for px in range(max(-K, kx - K), min(K, kx + K) + 1):
                for py in range(max(-K, ky - K), min(K, ky + K) + 1):
                    up, uq = F[:, px % N, py % N], F[:, (kx - px) % N, (ky - py) % N]
                    B += np.outer(up, uq)
            k = np.array([kx, ky], dtype=float)
            b = -1j * (B @ k)          # b_i = -i sum_j k_j B_ij (B symmetric after the full sum)
            want_b[:, kx % N, ky] = b
            if kx or ky:
                want_n[:, kx % N, ky] = b - k * (k @ b) / (k @ k)
    assert rel(got["b"], want_b) < 1e-13
    assert rel(got["n"], want_n) < 1e-13


# ------------------------------------------------------------------------------------------- Q2
def test_q2_taylor_green_projects_to_zero_and_decays_exactly(oracle2d):
    N, nu, dt = 16, 0.01, 1e-3
    uh = oracle2d.set_initial(N, inputs.taylor_green_2d_plane(N))
    parts = oracle2d.rhs_parts(N, oracle2d.Params(), uh)
    assert np.abs(parts["b"]).max() > 0.1 and np.abs(parts["n"]).max() < 1e-15      # a gradient: removed by the projection
    p = oracle2d.Params(nu=nu)
    u = uh.copy()
    for _ in range(20):
        u = oracle2d.step(N, p, u, dt)
    z = -nu * 2.0 * dt
    g = 1 + z + z * z / 2 + z ** 3 / 6
    assert abs(g ** 20 - 0.9996000799893343) < 1e-15      # the golden of tests/golden/rk3_decay_taylor_green.txt
    assert rel(u, g ** 20 * uh) < 1e-14


@pytest.mark.parametrize("s", [1.0, 1.5])
def test_q2_hyperviscous_single_mode(oracle2d, s):
    """One shear mode u = (0, cos(9 x)) with |k| = 9 > m_N = 4 (N = 16... m = sqrt(N)): N_hat = 0, decays by g(-d_k dt)^n."""
    N, n = 32, 5
    X, _ = inputs.grid2(N)
    u = np.stack([np.zeros((N, N)), np.cos(9 * X)])
    uh = oracle2d.set_initial(N, u)
    p = oracle2d.Params(eps=0.05, s=s)
    kabs, mN, q = 9.0, np.sqrt(N), (2 * s - 1) / 0.5
    d = 0.05 / N ** (2 * s - 1) * kabs ** (2 * s) * (1 - (mN / kabs) ** q)
    dt = 0.01
    z = -d * dt
    g = 1 + z + z * z / 2 + z ** 3 / 6
    v = uh.copy()
    for _ in range(n):
        v = oracle2d.step(N, p, v, dt)
    assert rel(v, g ** n * uh) < 1e-14 and g < 1


# ------------------------------------------------------------------------------------------- Q3
@pytest.mark.parametrize("N", [16, 24, 32])
def test_q3_energy_and_enstrophy_identities(oracle2d, N):
    """Exact dealiasing: the truncated nonlinear term conserves energy, and in two dimensions also enstrophy:
    Re sum_k w conj(u_k).N_k = 0 and Re sum_k w |k|^2 conj(u_k).N_k = 0."""
    uh = full_state(oracle2d, N, 70 + N)
    n = oracle2d.rhs_parts(N, oracle2d.Params(), uh)["n"]
    KX, KY = wavenumbers(N)
    w = half_weights(N)
    e = np.sum(w * np.real(np.conj(uh) * n))
    z = np.sum(w * (KX ** 2 + KY ** 2) * np.real(np.conj(uh) * n))
    assert abs(e) < 1e-13 * np.sum(w * np.abs(uh) * np.abs(n))
    assert abs(z) < 1e-13 * np.sum(w * (KX ** 2 + KY ** 2) * np.abs(uh) * np.abs(n))


# ------------------------------------------------------------------------------------------- Q4
def test_q4_solenoidal_masks_galilean_padding(oracle2d):
    N = 16
    uh = full_state(oracle2d, N, 11)
    p = oracle2d.Params(nu=0.01, eps=0.05)
    r = oracle2d.rhs(N, p, uh)
    KX, KY = wavenumbers(N)
    assert np.abs(KX * r[0] + KY * r[1]).max() < 1e-14 * np.abs(r).max() * N
    assert np.all(r[:, N // 2] == 0) and np.all(r[:, :, N // 2] == 0) and np.all(r[:, 0, 0] == 0)
    # Galilean shift: N[u + U] - N[u] = -i (k.U) u
    U = np.array([0.3, -0.7])
    sh = uh.copy()
    sh[:, 0, 0] += U
    n0 = oracle2d.rhs_parts(N, oracle2d.Params(), uh)["n"]
    n1 = oracle2d.rhs_parts(N, oracle2d.Params(), sh)["n"]
    want = -1j * (KX * U[0] + KY * U[1])[None] * uh
    want[:, 0, 0] = 0
    assert rel(n1 - n0, want) < 1e-13
    # independence of the padded size (readings A3 / A12)
    assert rel(oracle2d.rhs(N, p, uh, M=2 * N), r) < 1e-13


# ------------------------------------------------------------------------------------------- Q5
@pytest.mark.parametrize("N", [8, 16])
def test_q5_matches_the_3d_oracle_on_z_independent_data(oracle, oracle2d, N):
    """"The 3D solver is then checked by initializing the flow field with the previously checked 2D initial
    conditions while keeping the extra dimension constant".  Here the other way round: the (independently pinned) 3-D oracle on
    (u1, u2, 0)(x, y) must give, in its kz = 0 plane, what the 2-D oracle gives -- RHS, an RK3 step, max|u|, spectra."""
    u2 = inputs.gaussian_field_2d(N, 21, lambda k: 1.0 / (1.0 + k))
    u3 = np.zeros((3, N, N, N))
    u3[0] = u2[0][:, :, None]
    u3[1] = u2[1][:, :, None]
    uh2 = oracle2d.set_initial(N, u2)
    uh3 = oracle.set_initial(N, u3)
    assert rel(uh3[:2, :, :, 0][:, :, :N // 2 + 1], uh2) < 1e-14 and np.abs(uh3[2]).max() < 1e-15 and np.abs(uh3[:, :, :, 1:]).max() < 1e-15
    kw = dict(nu=0.01, eps=0.05, s=1.5)
    r2 = oracle2d.rhs_parts(N, oracle2d.Params(**kw), uh2)
    r3 = oracle.rhs_parts(N, oracle.Params(**kw), uh3)
    assert rel(r3["r"][:2, :, :N // 2 + 1, 0], r2["r"]) < 1e-13
    assert abs(r3["umax"] - r2["umax"]) < 1e-14 * r2["umax"]
    s2 = oracle2d.step(N, oracle2d.Params(**kw), uh2, 0.01)
    s3 = oracle.step(N, oracle.Params(**kw), uh3, 0.01)
    assert rel(s3[:2, :, :N // 2 + 1, 0], s2) < 1e-13
    assert np.abs(oracle.energy_spectrum(N, uh3, N) - oracle2d.energy_spectrum(N, uh2, N)).max() < 1e-14
    assert np.abs(oracle.enstrophy_spectrum(N, uh3, N) - oracle2d.enstrophy_spectrum(N, uh2, N)).max() < 1e-13


# ------------------------------------------------------------------------------------------- Q6
def test_q6_max_velocity(oracle2d):
    N = 8
    uh = np.zeros(oracle2d.spectral_shape(N), dtype=np.complex128)
    uh[:, 0, 0] = [0.3, -0.7]
    assert abs(oracle2d.max_velocity(N, uh) - np.sqrt(0.58)) < 1e-15          # Euclidean norm of both components
    assert oracle2d.rhs_parts(N, oracle2d.Params(), uh)["umax"] == oracle2d.max_velocity(N, uh)
    x = 2 * np.pi * np.arange(N) / N
    u = np.zeros((2, N, N))
    u[1] = np.cos(x - 2 * np.pi / 12)[:, None]                               # maximum 1 on the 12-point padded grid only
    assert abs(oracle2d.max_velocity(N, oracle2d.set_initial(N, u)) - 1.0) < 1e-14
    u = np.zeros((2, N, N))
    u[0] = np.cos(x - 2 * np.pi / 12)[None, :]
    assert abs(oracle2d.max_velocity(N, oracle2d.set_initial(N, u)) - 1.0) < 1e-14
    # random state on the padded grid by a zero-padded numpy irfft2
    N = 12
    M = 18
    uh = full_state(oracle2d, N, 33)
    pad = np.zeros((2, M, M // 2 + 1), dtype=np.complex128)
    K = N // 2 - 1
    for ix in range(N):
        kx = ix if ix < N // 2 else ix - N
        if abs(kx) <= K:
            pad[:, kx % M, :K + 1] = uh[:, ix, :K + 1]
    phys = np.fft.irfft2(pad, s=(M, M), axes=(1, 2)) * M ** 2
    want = np.sqrt((phys ** 2).sum(axis=0)).max()
    assert abs(oracle2d.max_velocity(N, uh) - want) < 1e-13 * want


# ------------------------------------------------------------------------------------------- Q7
def test_q7_spectra(oracle2d):
    N = 16
    u = inputs.gaussian_field_2d(N, 8, lambda k: k * np.exp(-k / 3.0))
    uh = oracle2d.set_initial(N, u)
    f = oracle2d.get_fields(N, uh)
    assert abs(oracle2d.energy_spectrum(N, uh, 2 * N).sum() - 0.5 * np.mean(np.sum(f * f, axis=0))) < 1e-14
    KX, KY = wavenumbers(N)
    om = np.fft.irfft2(1j * (KX * uh[1] - KY * uh[0]), s=(N, N)) * N ** 2
    assert abs(oracle2d.enstrophy_spectrum(N, uh, 2 * N).sum() - 0.5 * np.mean(om * om)) < 1e-13
    tg = oracle2d.set_initial(N, inputs.taylor_green_2d_plane(N))
    E = oracle2d.energy_spectrum(N, tg, N)
    assert abs(E[1] - 0.25) < 1e-15 and np.abs(np.delete(E, 1)).max() < 1e-30
    assert abs(oracle2d.enstrophy_spectrum(N, tg, N)[1] - 0.5) < 1e-15          # omega = 2 sin x sin y: 1/2 <omega^2> = 1/2


# ------------------------------------------------------------------------------------------- Q8
def test_q8_vortex_patch_conservation(oracle2d):
    """Vortex patch: under the inviscid truncated dynamics the mean flow never changes, the field stays
    solenoidal, and energy and enstrophy are conserved up to the time-stepping error of the third-order scheme: halving
    dt over the same horizon reduces both drifts by about 2^3."""
    N = 32
    uh = oracle2d.set_initial(N, inputs.vortex_patch(N, radius=1.0))
    p = oracle2d.Params()
    dt = 0.4 * (2 * np.pi / N) / oracle2d.max_velocity(N, uh)
    E0, Z0 = oracle2d.energy_spectrum(N, uh, N).sum(), oracle2d.enstrophy_spectrum(N, uh, N).sum()
    drift = []
    for nsteps, h in ((8, dt), (16, dt / 2)):
        v = uh.copy()
        for _ in range(nsteps):
            v = oracle2d.step(N, p, v, h)
        assert np.all(v[:, 0, 0] == uh[:, 0, 0]) and np.abs(uh[:, 0, 0]).max() < 1e-15     # R(0) = 0: the mean flow never changes
        drift.append((abs(oracle2d.energy_spectrum(N, v, N).sum() / E0 - 1), abs(oracle2d.enstrophy_spectrum(N, v, N).sum() / Z0 - 1)))
        KX, KY = wavenumbers(N)
        assert np.abs(KX * v[0] + KY * v[1]).max() < 1e-14
    assert drift[0][0] < 1e-4 and drift[0][1] < 1e-2
    assert 6.0 < drift[0][0] / drift[1][0] < 10.0 and 6.0 < drift[0][1] / drift[1][1] < 10.0
