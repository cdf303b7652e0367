"""GPU parity tests of the TWO-DIMENSIONAL solver (include/ns2d.h): the CUDA path through the C ABI against
the 2-D CPU oracle (oracle/ns2d_oracle.cpp) element by element on the same seeded inputs, at every supported size, plus the
invariants of the 2-D equations run on the GPU path.  Tolerances as in three dimensions: relative L2 <= 1e-12 per RHS,
<= 1e-10 after 20 RK3 steps (fp64); 1e-5 / 1e-4 (fp32).   python -m pytest tests -m gpu
"""
import numpy as np
import pytest

from paper_2401_09843_b200 import inputs

pytestmark = pytest.mark.gpu
TOL_RHS_F64, TOL_STEPS_F64 = 1e-12, 1e-10


@pytest.fixture(scope="module")
def ns():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_09843_b200 import binding
    binding.lib()
    return binding


def rel(a, b):
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) else np.float64)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(np.asarray(b).ravel()), 1e-300))


def field2(N, seed):
    return inputs.gaussian_field_2d(N, seed, lambda k: 1.0 / (1.0 + k) ** 2)


@pytest.mark.parametrize("N", [128, 256, 512])
def test_2d_rhs_and_steps_fp64(ns, oracle2d, N):
    """set_initial (non-solenoidal input), get_fields, one RHS (every stored entry) and 12 / 3 / 1 CFL steps with the oracle
    replaying the GPU's dt, three samples of different recipes in one launch; spectra of the final state."""
    us = np.stack([field2(N, 100 + N) + 0.2 * inputs.normal01(N, 7, 2 * N * N).reshape(2, N, N),
                   inputs.shear_layer_2d(N, 3), inputs.vortex_patch(N, seed=5, radius=1.0, delta=0.3)])
    kw = dict(nu=0.001, eps=0.05, s=1.0)
    s = ns.Solver2D(N, batch=3, **kw)
    s.set_initial(us)
    p = oracle2d.Params(**kw)
    uh = [oracle2d.set_initial(N, u) for u in us]
    got = s.get_spectral()
    f = s.get_fields()
    for b in range(3):
        assert rel(got[b], uh[b]) < 1e-13
        assert np.all(got[b][:, N // 2] == 0) and np.all(got[b][:, :, N // 2] == 0)
        assert rel(f[b], oracle2d.get_fields(N, uh[b])) < 1e-13
    s.set_spectral(np.stack(uh))
    r = s.rhs()
    um = s.max_velocity()
    for b in range(3):
        want = oracle2d.rhs_parts(N, p, uh[b])
        assert rel(r[b], want["r"]) < TOL_RHS_F64
        # no single entry is off; round-off scales with the flux before the projection (for the shear layer and the vortex
        # patch most of it is a gradient that the projection removes), so the bound is relative to max|b|, not max|R|
        assert np.abs(r[b] - want["r"]).max() < 1e-13 * np.abs(want["b"]).max()
        assert np.all(r[b][:, N // 2] == 0) and np.all(r[b][:, :, N // 2] == 0) and np.all(r[b][:, 0, 0] == 0)
        assert abs(um[b] - want["umax"]) < 1e-13 * want["umax"]
    assert np.array_equal(s.get_spectral(), np.stack(uh))          # state unchanged by ns2d_rhs
    nsteps = {128: 12, 256: 3, 512: 1}[N]     # the single-threaded naive oracle needs 1.3 s per 512^2 step and sample
    worst = 0.0
    for i in range(nsteps):
        dts = s.step_cfl(0.2, 1e9)
        uh = [oracle2d.step(N, p, uh[b], dts[b]) for b in range(3)]
        worst = max(worst, max(rel(s.get_spectral()[b], uh[b]) for b in range(3)))
        assert worst < TOL_STEPS_F64, (i, worst)
    E, Z = s.energy_spectrum(N), s.enstrophy_spectrum(N)
    for b in range(3):
        assert np.abs(E[b] - oracle2d.energy_spectrum(N, uh[b], N)).max() < 1e-13
        Zo = oracle2d.enstrophy_spectrum(N, uh[b], N)
        assert np.abs(Z[b] - Zo).max() < 1e-12 * Zo.max()
    print(f"2-D N = {N}: worst rel-L2 over {nsteps} steps {worst:.2e}")


def test_2d_invariants_on_the_gpu_path(ns):
    N = 256
    KX, KY = np.meshgrid(np.fft.fftfreq(N, 1.0 / N), np.arange(N // 2 + 1.0), indexing="ij")
    w = np.full(N // 2 + 1, 2.0)
    w[0] = 1.0
    # Taylor-Green: the nonlinear term is a gradient; decay at the closed-form RK3 rate (tests/golden/rk3_decay_taylor_green.txt)
    s = ns.Solver2D(N)
    s.set_initial(inputs.taylor_green_2d_plane(N)[None])
    assert np.abs(s.rhs()).max() < 1e-14
    s = ns.Solver2D(N, nu=0.01)
    s.set_initial(inputs.taylor_green_2d_plane(N)[None])
    u0 = s.get_spectral()
    for _ in range(20):
        s.step(1e-3)
    assert rel(s.get_spectral(), 0.9996000799893343 * u0) < 1e-13
    assert abs(s.time(0) - 0.02) < 1e-15
    # energy and enstrophy identities, solenoidal RHS, Galilean shift (inviscid)
    s = ns.Solver2D(N)
    s.set_initial(field2(N, 77)[None])
    uh = s.get_spectral()[0]
    r = s.rhs()[0]
    assert abs(np.sum(w * np.real(np.conj(uh) * r))) < 1e-13 * np.sum(w * np.abs(uh) * np.abs(r))
    k2 = KX ** 2 + KY ** 2
    assert abs(np.sum(w * k2 * np.real(np.conj(uh) * r))) < 1e-13 * np.sum(w * k2 * np.abs(uh) * np.abs(r))
    assert np.abs(KX * r[0] + KY * r[1]).max() < 1e-13 * np.abs(r).max() * N
    U = np.array([0.3, -0.7])
    sh = uh.copy()
    sh[:, 0, 0] += U
    s.set_spectral(sh[None])
    want = -1j * (KX * U[0] + KY * U[1])[None] * uh
    want[:, 0, 0] = 0
    assert rel(s.rhs()[0] - r, want) < 1e-12


def test_2d_batch_is_bitwise_independent_and_t_end(ns):
    """Reading A18 in two dimensions with a large batch: every sample of a 96-sample launch equals its batch-of-1 result bit for
    bit; ns2d_advance brings every sample to t_end; the replay call reproduces a CFL step."""
    N, B = 128, 96
    us = np.stack([inputs.shear_layer_2d(N, 1000 + i) + 0.01 * field2(N, 50 + i) for i in range(B)])
    kw = dict(eps=0.05, s=1.5)
    sb = ns.Solver2D(N, batch=B, **kw)
    sb.set_initial(us)
    before = sb.get_spectral()
    dts = sb.step_cfl(0.2, 1e9)
    got = sb.get_spectral()
    for i in (0, 37, 95):
        s1 = ns.Solver2D(N, batch=1, **kw)
        s1.set_initial(us[i:i + 1])
        d1 = s1.step_cfl(0.2, 1e9)
        assert d1[0] == dts[i] and np.array_equal(s1.get_spectral()[0], got[i])
    s2 = ns.Solver2D(N, batch=B, **kw)
    s2.set_spectral(before)
    s2.step_dts(dts)
    assert np.array_equal(s2.get_spectral(), got)
    n = sb.advance(0.2, 0.05)
    assert n > 2 and all(abs(sb.time(b) - 0.05) < 1e-15 for b in (0, 50, 95))
    E = sb.energy_spectrum(N)
    assert np.isfinite(E).all() and len(set(np.round(dts, 12))) > 10


def test_2d_fp32_and_errors(ns, oracle2d):
    N = 256
    u = field2(N, 9)
    kw = dict(nu=0.001, eps=0.05)
    s = ns.Solver2D(N, dtype="f32", **kw)
    s.set_initial(u[None])
    uh = oracle2d.set_initial(N, u)
    assert rel(s.get_spectral()[0], uh) < 1e-6
    p = oracle2d.Params(**kw)
    assert rel(s.rhs()[0], oracle2d.rhs(N, p, uh)) < 1e-5
    for _ in range(20):
        s.step(1e-3)
        uh = oracle2d.step(N, p, uh, 1e-3)
    assert rel(s.get_spectral()[0], uh) < 1e-4
    assert rel(s.get_fields()[0], oracle2d.get_fields(N, uh)) < 1e-4
    # errors and the non-finite guard
    t = ns.Solver2D(N, batch=2)
    with pytest.raises(ns.NSError) as e:
        t.step(1e-3)
    assert e.value.code == ns.NS_ERR_STATE
    good = np.stack([oracle2d.set_initial(N, field2(N, 1)), oracle2d.set_initial(N, field2(N, 2))])
    bad = good.copy()
    bad[1, 0, 3, 2] = np.nan
    t.set_spectral(bad)
    with pytest.raises(ns.NSError) as e:
        t.step_cfl(0.2, 1e9)
    assert e.value.code == ns.NS_ERR_NONFINITE and "sample 1" in str(e.value)
    n0 = t.kernel_launches()
    t.set_spectral(good)
    t.step(1e-3)
    assert t.kernel_launches() - n0 == 1 + 3 * 4 + 1      # to_internal + 3 stages x (b1, b2, b3, b4) + dt setup
    assert t.device_bytes() > 0


@pytest.mark.parametrize("N", [48, 100, 200])
def test_2d_general_even_n_on_a_larger_transform_grid(ns, oracle2d, N):
    """An N that is not 128 / 256 / 512 runs on the next of those as transform grid (padded grid 3 Nt / 2 > 3N/2), the
    state truncated to the user's N: against the 2-D oracle at the user's N with the SAME padded size -- set_initial (mixed-radix or
    plain DFT on the N grid), get_fields, RHS (every entry; also against M = 3N/2), max|u|, CFL steps, spectra."""
    u = field2(N, 600 + N) + 0.2 * inputs.normal01(N, 9, 2 * N * N).reshape(2, N, N)
    kw = dict(nu=0.001, eps=0.05, s=1.5)
    s = ns.Solver2D(N, batch=1, **kw)
    Nt, M = s.transform_grid, s.padded_size
    assert Nt in (128, 256) and Nt > N and M > 3 * N // 2
    s.set_initial(u[None])
    uh = oracle2d.set_initial(N, u)
    got = s.get_spectral()[0]
    assert got.shape == uh.shape and rel(got, uh) < 1e-13
    assert rel(s.get_fields()[0], oracle2d.get_fields(N, uh)) < 1e-13
    s.set_spectral(uh[None])
    assert np.array_equal(s.get_spectral()[0], uh)
    p = oracle2d.Params(**kw)
    want = oracle2d.rhs_parts(N, p, uh, M)
    r = s.rhs()[0]
    assert rel(r, want["r"]) < TOL_RHS_F64
    assert rel(r, oracle2d.rhs(N, p, uh)) < TOL_RHS_F64
    assert np.all(r[:, N // 2] == 0) and np.all(r[:, :, N // 2] == 0)
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    worst = 0.0
    for i in range(4):
        dts = s.step_cfl(0.2, 1e9)
        assert abs(dts[0] - 0.2 * (2 * np.pi / N) / oracle2d.max_velocity(N, uh, M)) < 1e-12 * dts[0]
        uh = oracle2d.step(N, p, uh, dts[0], M)
        worst = max(worst, rel(s.get_spectral()[0], uh))
        assert worst < TOL_STEPS_F64, (i, worst)
    assert np.abs(s.energy_spectrum(N)[0] - oracle2d.energy_spectrum(N, uh, N)).max() < 1e-13
    print(f"2-D N = {N} on transform grid {Nt}: worst rel-L2 over 4 steps {worst:.2e}")
