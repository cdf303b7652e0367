"""Host checks of the seeded input generators for the paper's own experiments (eq. 6.1-6.6)
and of the oracle on them with the paper's hyperviscosity order s = 1.5 (no GPU)."""
import numpy as np
import pytest

from paper_2401_09843_b200 import inputs


@pytest.fixture(scope="module")
def oracle():
    from oracle import ns_oracle
    return ns_oracle


def test_taylor_green_3d_perturbed_recipe():
    N = 16
    u = inputs.taylor_green_3d_perturbed(N, seed=3)
    X, Y, Z = inputs.grid(N)
    base = np.stack([np.cos(X) * np.sin(Y) * np.sin(Z), -np.sin(X) * np.cos(Y) * np.sin(Z), np.zeros_like(X)])
    e = u - base
    # eq. (6.2): |e_d| <= (1/8) * 8 * 0.025, only the second harmonics, a different draw per component and per seed
    assert np.abs(e).max() <= 0.025 + 1e-15
    E = np.fft.fftn(e, axes=(1, 2, 3))
    k = np.abs(np.fft.fftfreq(N, 1.0 / N))
    mask = np.ones((N, N, N), bool)
    sel = np.isin(k, (0.0, 2.0))
    mask[np.ix_(sel, sel, sel)] = False
    assert np.abs(E[:, mask]).max() < 1e-10
    assert not np.allclose(e[0], e[1]) and not np.allclose(u, inputs.taylor_green_3d_perturbed(N, seed=4))
    # eq. (6.1) with A + B + C = 0 is solenoidal
    U = np.fft.fftn(base, axes=(1, 2, 3))
    kk = np.fft.fftfreq(N, 1.0 / N)
    div = kk[:, None, None] * U[0] + kk[None, :, None] * U[1] + kk[None, None, :] * U[2]
    assert np.abs(div).max() < 1e-9


def test_cylindrical_shear_recipe():
    N = 64
    u = inputs.cylindrical_shear(N, seed=5, rho=0.0)
    assert set(np.unique(u[0])) == {-1.0, 1.0} and not u[1].any() and not u[2].any()
    # eq. (6.6): u = -1 inside the perturbed cylinder of radius 1/4 (area pi/16 of every x-slice, to grid accuracy)
    frac = (u[0] < 0).mean(axis=(1, 2))
    assert np.abs(frac - np.pi / 16).max() < 0.02
    # the axis of the cylinder moves with x by at most delta * p = 0.25
    yc = np.array([np.argwhere(u[0, i] < 0)[:, 0].mean() for i in range(N)]) / N
    assert np.ptp(yc) > 1e-3 and np.abs(yc - 0.5).max() < 0.25
    s = inputs.cylindrical_shear(N, seed=5, rho=0.05)
    assert np.all(np.sign(s[0][np.abs(s[0]) > 0.9]) == u[0][np.abs(s[0]) > 0.9])
    assert not np.allclose(s, inputs.cylindrical_shear(N, seed=6, rho=0.05))


@pytest.mark.parametrize("name", ["tg3d", "cyl"])
def test_oracle_on_paper_experiments_is_dissipative(oracle, name):
    """s = 1.5 hyperviscosity: the discrete energy does not grow under SSP-RK3 at CFL 0.2, the
    state stays solenoidal, and with eps = 0 the nonlinear term alone conserves energy to O(dt^3) per step."""
    N = 16
    u = inputs.taylor_green_3d_perturbed(N, 1) if name == "tg3d" else inputs.cylindrical_shear(N, 1, rho=0.2)
    uh = oracle.set_initial(N, u)
    p = oracle.Params(eps=0.05, s=1.5)
    E = [oracle.energy_spectrum(N, uh, N).sum()]
    for _ in range(5):
        dt = 0.2 * (2 * np.pi / N) / oracle.max_velocity(N, uh)
        uh = oracle.step(N, p, uh, dt)
        E.append(oracle.energy_spectrum(N, uh, N).sum())
    assert all(b <= a * (1 + 1e-12) for a, b in zip(E, E[1:])) and E[-1] < E[0]
    k = np.fft.fftfreq(N, 1.0 / N)
    div = k[:, None, None] * uh[0] + k[None, :, None] * uh[1] + np.arange(N // 2 + 1.0)[None, None, :] * uh[2]
    assert np.abs(div).max() < 1e-13


def test_stratified_modes_cover_every_class():
    from _sampling import stratified_modes
    for N in (256, 512):
        m = stratified_modes(N, 512, 1)
        assert len(m) >= 512
        for ax in (0, 1):
            assert set(range(16)) <= set(m[:, ax] % 16)                       # every R2 class / column-tile lane
            assert {0, 7, N // 2 - 1, N // 2 + 1, N - 8, N - 1} <= set(m[:, ax])  # first / last tiles of both halves
            assert (m[:, ax] > N // 2).sum() > 100 and (m[:, ax] < N // 2).sum() > 100
        assert set(range(16)) <= set(m[:, 2]) and set(range(N // 2 - 16, N // 2)) <= set(m[:, 2])
