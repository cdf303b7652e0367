"""GPU parity tests: the CUDA path (through the C ABI of include/ns.h, via the ctypes binding) against
the CPU oracle, element by element on the same seeded inputs.  Tolerances are BASELINE.json's
north_star: relative L2 error <= 1e-12 per RHS and <= 1e-10 after 20 RK steps in fp64, 1e-5 / 1e-4 in
fp32.  Run on the B200 box:  python -m pytest tests -m gpu
"""
import numpy as np
import pytest

from paper_2401_09843_b200 import inputs
from _sampling import spectral_state

pytestmark = pytest.mark.gpu

TOL_RHS_F64, TOL_STEPS_F64 = 1e-12, 1e-10
TOL_RHS_F32, TOL_STEPS_F32 = 1e-5, 1e-4


@pytest.fixture(scope="module")
def ns():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_09843_b200 import binding
    binding.lib()  # fails loudly if libns.so is missing
    return binding


def rel(a, b):
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) else np.float64)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(np.asarray(b).ravel()), 1e-300))


def field(N, seed, full=False):
    if full:
        return inputs.gaussian_field(N, seed, lambda k: 1.0 / (1.0 + k), e_tot=0.5)
    return inputs.gaussian_field(N, seed, lambda k: k ** 4 * np.exp(-2.0 * (k / 4.0) ** 2), e_tot=0.5)


# ------------------------------------------------------------------------------------------------
def test_spectral_roundtrip_bit_exact(ns):
    N = 32
    s = ns.Solver(N, batch=2)
    rng = np.random.default_rng(0)
    u = (rng.standard_normal(s.spectral_shape) + 1j * rng.standard_normal(s.spectral_shape))
    s.set_spectral(u)
    got = s.get_spectral()
    want = u.copy()
    want[:, :, N // 2] = 0
    want[:, :, :, N // 2] = 0
    want[:, :, :, :, N // 2] = 0
    assert np.array_equal(got, want)
    s.set_spectral(got)
    assert np.array_equal(s.get_spectral(), got)


@pytest.mark.parametrize("N", [16, 32, 64])
def test_set_initial_and_get_fields(ns, oracle, N):
    u = field(N, 10 + N, full=True) + 0.3 * inputs.normal01(N, 9, 3 * N ** 3).reshape(3, N, N, N)  # not solenoidal
    s = ns.Solver(N)
    s.set_initial(u[None])
    want = oracle.set_initial(N, u)
    got = s.get_spectral()[0]
    assert rel(got, want) < 1e-13
    assert np.all(got[:, N // 2] == 0) and np.all(got[:, :, N // 2] == 0) and np.all(got[:, :, :, N // 2] == 0)
    assert rel(s.get_fields()[0], oracle.get_fields(N, want)) < 1e-13


@pytest.mark.parametrize("N", [16, 32, 64, 128])
def test_rhs_parity_fp64(ns, oracle, N):
    u = field(N, 100 + N, full=(N <= 64))
    p = dict(nu=0.01, eps=0.05, s=1.0)
    s = ns.Solver(N, **p)
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    s.set_spectral(uh[None])            # identical starting state on both sides
    want = oracle.rhs_parts(N, oracle.Params(**p), uh)
    got = s.rhs()[0]
    assert rel(got, want["r"]) < TOL_RHS_F64
    assert np.all(got[:, N // 2] == 0) and np.all(got[:, :, N // 2] == 0) and np.all(got[:, :, :, N // 2] == 0)
    assert np.all(got[:, 0, 0, 0] == 0)
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    # state unchanged by ns_rhs
    assert np.array_equal(s.get_spectral()[0], uh)


def test_config1_20_steps_fp64(ns, oracle):
    """BASELINE.json configs[0]: N=32, Taylor-Green + 1e-3 perturbation, nu = 0.01, dt = 1e-3, 20 RK steps."""
    N, dt = 32, 1e-3
    u = inputs.taylor_green_perturbed(N, seed=1)
    s = ns.Solver(N, nu=0.01)
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    assert rel(s.get_spectral()[0], uh) < 1e-13
    s.set_spectral(uh[None])
    p = oracle.Params(nu=0.01)
    assert rel(s.rhs()[0], oracle.rhs(N, p, uh)) < TOL_RHS_F64
    worst = 0.0
    for _ in range(20):
        s.step(dt)
        uh = oracle.step(N, p, uh, dt)
        worst = max(worst, rel(s.get_spectral()[0], uh))
    assert worst < TOL_STEPS_F64
    assert abs(s.time(0) - 20 * dt) < 1e-15
    E = s.energy_spectrum(N)[0]
    assert np.abs(E - oracle.energy_spectrum(N, uh, N)).max() < 1e-14
    Z = s.enstrophy_spectrum(N)[0]
    Zo = oracle.enstrophy_spectrum(N, uh, N)
    assert np.abs(Z - Zo).max() < 1e-13 * Zo.max()
    S = s.structure_function()[0]
    assert np.abs(S / oracle.structure_function(N, uh) - 1).max() < 1e-11


@pytest.mark.parametrize("N", [32, 64])
def test_hyperviscous_steps_fp64(ns, oracle, N):
    """Config-2 style: Gaussian field, hyperviscosity eps = 0.05, s = 1, CFL 0.2; oracle replays the GPU's dt."""
    u = inputs.gaussian_field(N, 2, lambda k: k ** 4 * np.exp(-2.0 * (k / 4.0) ** 2), e_tot=0.5)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    uh = oracle.set_initial(N, u)
    s.set_spectral(uh[None])
    p = oracle.Params(**kw)
    nsteps = 10 if N == 32 else 4
    for _ in range(nsteps):
        umax = oracle.max_velocity(N, uh)
        dts = s.step_cfl(0.2, 1e9)
        assert abs(dts[0] - 0.2 * (2 * np.pi / N) / umax) < 1e-12 * dts[0]
        uh = oracle.step(N, p, uh, dts[0])
    assert rel(s.get_spectral()[0], uh) < TOL_STEPS_F64


def test_fractional_order(ns, oracle):
    N = 32
    u = field(N, 7, full=True)
    kw = dict(nu=0.002, eps=0.05, s=1.5)
    s = ns.Solver(N, **kw)
    uh = oracle.set_initial(N, u)
    s.set_spectral(uh[None])
    assert rel(s.rhs()[0], oracle.rhs(N, oracle.Params(**kw), uh)) < TOL_RHS_F64


@pytest.mark.parametrize("name,N", [("tg3d", 64), ("cyl", 64), ("tg3d", 128)])
def test_paper_experiments_s15(ns, oracle, name, N):
    """NEXT-2 of SURVEY.md 8(f): the paper's own workloads, perturbed 3-D Taylor-Green (eq. 6.1-6.3) and cylindrical
    shear flow (eq. 6.4-6.6), with its fractional hyperviscosity order s = 1.5: set_initial,
    one RHS and CFL-0.2 steps against the oracle, which replays the GPU's dt."""
    u = inputs.taylor_green_3d_perturbed(N, 11) if name == "tg3d" else inputs.cylindrical_shear(N, 12, rho=0.05)
    kw = dict(eps=0.05, s=1.5)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    assert rel(s.get_spectral()[0], uh) < 1e-13
    s.set_spectral(uh[None])
    p = oracle.Params(**kw)
    assert rel(s.rhs()[0], oracle.rhs(N, p, uh)) < TOL_RHS_F64
    for _ in range(4 if N == 64 else 1):
        dts = s.step_cfl(0.2, 1e9)
        assert abs(dts[0] - 0.2 * (2 * np.pi / N) / oracle.max_velocity(N, uh)) < 1e-12 * dts[0]
        uh = oracle.step(N, p, uh, dts[0])
    assert rel(s.get_spectral()[0], uh) < TOL_STEPS_F64
    Zo = oracle.enstrophy_spectrum(N, uh, N)
    assert np.abs(s.enstrophy_spectrum(N)[0] - Zo).max() < 1e-10 * Zo.max()


@pytest.mark.parametrize("N,dtype", [(32, "f64"), (64, "f64"), (32, "f32")])
def test_structure_function_order_p(ns, oracle, N, dtype):
    """ns_structure_function_p (physical-space kernel) against the oracle for p = 1, 3, 4 and, for p = 2, also against
    ns_structure_function (the spectral-identity path); two samples in one launch."""
    us = np.stack([field(N, 500 + N), inputs.taylor_green_3d_perturbed(N, 13)])
    s = ns.Solver(N, batch=2, dtype=dtype)
    s.set_initial(us)
    tol = 1e-11 if dtype == "f64" else 2e-5
    for b in range(2):
        uh = oracle.set_initial(N, us[b])
        for p in (1.0, 3.0, 4.0):
            assert np.abs(s.structure_function_p(p)[b] / oracle.structure_function_p(N, uh, p) - 1).max() < tol
    assert np.abs(s.structure_function_p(2.0, nl=5) / s.structure_function(nl=5) - 1).max() < tol
    with pytest.raises(ns.NSError):
        s.structure_function_p(0.0)


def test_ensemble_moments(ns, oracle):
    """Pointwise mean and variance of the empirical measure over the batch (Algorithm 1) against the
    same moments of the oracle's physical fields; a batch of identical samples has zero variance to round-off."""
    N, B = 32, 5
    us = np.stack([inputs.cylindrical_shear(N, 40 + i, rho=0.3) for i in range(B)])
    s = ns.Solver(N, batch=B)
    s.set_initial(us)
    mean, var = s.ensemble_moments()
    f = np.stack([oracle.get_fields(N, oracle.set_initial(N, u)) for u in us])
    assert np.abs(mean - f.mean(axis=0)).max() < 1e-13
    assert np.abs(var - f.var(axis=0)).max() < 1e-13 and var.max() > 1e-3
    s.set_initial(np.stack([us[0]] * B))
    mean, var = s.ensemble_moments()
    assert var.max() < 1e-28 and np.abs(mean - f[0]).max() < 1e-13


def test_two_handles_on_two_streams(ns):
    """Handles are independent (include/ns.h): two solvers stepping concurrently on two streams -- their tensor-memory
    kernels share the SMs' 512 TMEM columns -- give bit for bit what each gives alone."""
    import torch
    N = 256
    ua = inputs.taylor_green_3d_perturbed(N, 21)[None]
    ub = inputs.cylindrical_shear(N, 22, rho=0.1)[None]
    kw = dict(eps=0.05, s=1.0)
    ref = []
    for u in (ua, ub):
        s = ns.Solver(N, **kw)
        s.set_initial(u)
        for _ in range(3):
            s.step(1e-3)
        ref.append(s.get_spectral())
        del s
    st = [torch.cuda.Stream(), torch.cuda.Stream()]
    sol = [ns.Solver(N, stream=st[i].cuda_stream, **kw) for i in range(2)]
    sol[0].set_initial(ua)
    sol[1].set_initial(ub)
    for _ in range(3):
        for s in sol:
            s.step(1e-3)          # asynchronous launches on the handle's stream
    got = [s.get_spectral() for s in sol]
    assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1])


def test_advance_to_t_end(ns):
    """ns_advance == the host loop over ns_step_cfl it replaces, bit for bit, with every sample ending at t_end."""
    N, B, t_end = 32, 3, 0.05
    us = np.stack([field(N, 600 + i) * (1.0 + i) for i in range(B)])
    kw = dict(eps=0.05, s=1.5)
    a = ns.Solver(N, batch=B, **kw)
    a.set_initial(us)
    steps = 0
    while min(a.time(b) for b in range(B)) < t_end:
        a.step_cfl(0.2, t_end, return_dt=False)
        steps += 1
    b_ = ns.Solver(N, batch=B, **kw)
    b_.set_initial(us)
    n = b_.advance(0.2, t_end)
    assert steps <= n <= steps + 3 and steps > 5
    assert all(abs(b_.time(i) - t_end) < 1e-15 for i in range(B))
    assert np.array_equal(a.get_spectral(), b_.get_spectral())
    assert b_.advance(0.2, t_end) == 0                       # already there
    c = ns.Solver(N, batch=B, **kw)
    c.set_initial(us)
    assert c.advance(0.2, t_end, max_steps=2) == 2 and c.time(0) < t_end


def test_batch_is_bitwise_independent(ns):
    """Reading A18: a batched launch gives bit for bit the per-sample result of batch = 1."""
    N, B = 32, 5
    us = np.stack([inputs.shear_layer(N, 1000 + i) + 0.01 * field(N, 50 + i) for i in range(B)])
    sb = ns.Solver(N, batch=B, eps=0.05)
    sb.set_initial(us)
    for _ in range(3):
        sb.step(2e-3)
    got = sb.get_spectral()
    rb = sb.rhs()
    for i in (0, 3, 4):
        s1 = ns.Solver(N, batch=1, eps=0.05)
        s1.set_initial(us[i:i + 1])
        for _ in range(3):
            s1.step(2e-3)
        assert np.array_equal(s1.get_spectral()[0], got[i])
        assert np.array_equal(s1.rhs()[0], rb[i])


def test_step_cfl_per_sample_and_t_end(ns, oracle):
    N, B = 32, 3
    us = np.stack([(1.0 + i) * field(N, 60 + i) for i in range(B)])
    s = ns.Solver(N, batch=B, nu=0.01)
    s.set_initial(us)
    umax = s.max_velocity()
    for i in range(B):
        uh = oracle.set_initial(N, us[i])
        assert abs(umax[i] - oracle.max_velocity(N, uh)) < 1e-12 * umax[i]
    t_end = 0.9 * 0.2 * (2 * np.pi / N) / umax[0]       # sample 0 is limited by t_end, the faster ones by CFL
    before = s.get_spectral()
    dts = s.step_cfl(0.2, t_end)
    assert dts[0] == pytest.approx(t_end, rel=1e-15)
    for i in (1, 2):
        assert dts[i] == pytest.approx(min(0.2 * (2 * np.pi / N) / umax[i], t_end), rel=1e-12)
    # replay with ns_step_dts reproduces the step bit for bit
    s2 = ns.Solver(N, batch=B, nu=0.01)
    s2.set_spectral(before)
    s2.step_dts(dts)
    assert np.array_equal(s2.get_spectral(), s.get_spectral())
    # finished samples are untouched
    mid = s.get_spectral()
    dts2 = s.step_cfl(0.2, t_end)
    assert dts2[0] == 0.0
    after = s.get_spectral()
    assert np.array_equal(after[0], mid[0])
    assert s.time(0) == pytest.approx(t_end, rel=1e-15)
    assert np.isnan(s.time(B))


# ------------------------------------------------------------- full BASELINE sizes, sampled outputs
def _sample_modes(N, n, seed):
    rng = np.random.default_rng(seed)
    K = N // 2 - 1
    lowk = np.stack([rng.integers(-4, 5, n // 2) % N, rng.integers(-4, 5, n // 2) % N, rng.integers(0, 5, n // 2)], axis=1)
    anyk = np.stack([rng.integers(0, N, n - n // 2), rng.integers(0, N, n - n // 2), rng.integers(0, N // 2, n - n // 2)], axis=1)
    fixed = np.array([(1, 0, 0), (0, 0, 1), (K, K, K), (N - K, 3, K), (5, N - K, 0), (N // 2, 2, 2), (0, 0, 0)])
    return np.concatenate([lowk, anyk, fixed]).astype(np.int32)


def test_config4_ensemble_two_samples(ns, oracle):
    """BASELINE.json configs[3]: 32 x 128^3 shear-layer ensemble in one launch; the last sample (31) against the oracle
    (1 RHS + 1 CFL step, oracle replays the GPU's dt), spectra and structure functions of those samples."""
    N, B = 128, 32
    us = inputs.shear_layer_ensemble(N, B, seed0=1000)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, batch=B, **kw)
    s.set_initial(us)
    p = oracle.Params(**kw)
    u0 = s.get_spectral()
    r0 = s.rhs()
    dts = s.step_cfl(0.2, 1.0)
    got = s.get_spectral()
    E = s.energy_spectrum(N)
    Zs = s.enstrophy_spectrum(N)
    S = s.structure_function()
    for i in (31,):     # sample 1 is replayed for several steps in tests/test_gpu_schedule.py
        uh = oracle.set_initial(N, us[i])       # the oracle works on ITS OWN initial state (no input from the CUDA path)
        assert rel(u0[i], uh) < 1e-13
        assert rel(r0[i], oracle.rhs(N, p, uh)) < TOL_RHS_F64
        assert abs(dts[i] - 0.2 * (2 * np.pi / N) / oracle.max_velocity(N, uh)) < 1e-12 * dts[i]
        un = oracle.step(N, p, uh, dts[i])
        assert rel(got[i], un) < TOL_STEPS_F64
        assert np.abs(E[i] - oracle.energy_spectrum(N, un, N)).max() < 1e-13
        Zo = oracle.enstrophy_spectrum(N, un, N)
        assert np.abs(Zs[i] - Zo).max() < 1e-10 * Zo.max()
        assert np.abs(S[i] / oracle.structure_function(N, un) - 1).max() < 1e-10
    assert len(set(np.round(dts, 12))) > 1          # distinct seeds -> distinct steps


def test_config4_ensemble_to_t1(ns):
    """BASELINE.json configs[3] at full length: the 32 x 128^3 shear-layer ensemble integrated to t = 1 at CFL 0.2 in one
    batched run (ns_advance).  The oracle needs hours for this horizon (its parity over the first step is
    test_config4_ensemble_two_samples), so this checks what must hold at any length: every sample ends at t = 1,
    sample 7 of the batch equals bit for bit the same sample integrated alone (reading A18), the energy of every sample
    has not grown, the ensemble statistics are finite, and the two independent routes to S_2 (spectral identity and
    physical-space increments) agree."""
    N, B = 128, 32
    us = inputs.shear_layer_ensemble(N, B, seed0=1000)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, batch=B, **kw)
    s.set_initial(us)
    E0 = s.energy_spectrum(N).sum(axis=1)
    n = s.advance(0.2, 1.0)
    assert 20 < n < 2000 and all(abs(s.time(b) - 1.0) < 1e-14 for b in range(B))
    E = s.energy_spectrum(N)
    assert np.isfinite(E).all() and np.all(E.sum(axis=1) <= E0 * (1 + 1e-12)) and np.all(E.sum(axis=1) > 0.5 * E0)
    S2 = s.structure_function(nl=16)
    assert np.abs(s.structure_function_p(2.0, nl=16) / S2 - 1).max() < 1e-10
    mean, var = s.ensemble_moments()
    assert np.isfinite(mean).all() and var.max() > 1e-4          # distinct seeds decorrelate the samples
    Emean = E.mean(axis=0)                                       # the reported ensemble-mean spectrum
    assert Emean[1:4].sum() > 0.5 * Emean.sum()                  # the shear layer keeps its energy at the largest scales
    one = ns.Solver(N, batch=1, **kw)
    one.set_initial(us[7:8])
    one.advance(0.2, 1.0)
    assert np.array_equal(one.get_spectral()[0], s.get_spectral()[7])


# ---------------------------------------------------------------------- invariants run on the GPU path
def test_gpu_invariants(ns):
    N = 32
    KX, KY, KZ = np.meshgrid(np.fft.fftfreq(N, 1.0 / N), np.fft.fftfreq(N, 1.0 / N), np.arange(N // 2 + 1.0), indexing="ij")
    w = np.full(N // 2 + 1, 2.0)
    w[0] = 1.0
    # P2: Taylor-Green and ABC nonlinear terms are gradients -> RHS = 0 without viscosity
    for u in (inputs.taylor_green_2d(N), inputs.abc_flow(N)):
        s = ns.Solver(N)
        s.set_initial(u[None])
        assert np.abs(s.rhs()).max() < 1e-14
    # P3: decay at the closed-form RK3 rate
    s = ns.Solver(N, nu=0.01)
    s.set_initial(inputs.taylor_green_2d(N)[None])
    u0 = s.get_spectral()
    for _ in range(20):
        s.step(1e-3)
    assert rel(s.get_spectral(), 0.9996000799893343 * u0) < 1e-13
    # P4 energy identity, P5 solenoidal RHS, P6 Galilean shift
    s = ns.Solver(N)
    s.set_initial(field(N, 77, full=True)[None])
    uh = s.get_spectral()[0]
    r = s.rhs()[0]
    assert abs(np.sum(w * np.real(np.conj(uh) * r))) < 1e-13 * np.sum(w * np.abs(uh) * np.abs(r))
    div = KX * r[0] + KY * r[1] + KZ * r[2]
    assert np.abs(div).max() < 1e-13 * np.abs(r).max() * N
    U = np.array([0.3, -0.7, 0.45])
    sh = uh.copy()
    sh[:, 0, 0, 0] += U
    s.set_spectral(sh[None])
    want = -1j * (KX * U[0] + KY * U[1] + KZ * U[2])[None] * uh
    want[:, 0, 0, 0] = 0
    assert rel(s.rhs()[0] - r, want) < 1e-12


# ------------------------------------------------------------------------------------------- fp32
@pytest.mark.parametrize("N", [32, 64])
def test_fp32_parity(ns, oracle, N):
    u = field(N, 300 + N)
    kw = dict(nu=0.01, eps=0.05)
    s = ns.Solver(N, dtype="f32", **kw)
    uh = oracle.set_initial(N, u)
    s.set_initial(u[None])
    assert rel(s.get_spectral()[0], uh) < 1e-6
    p = oracle.Params(**kw)
    assert rel(s.rhs()[0], oracle.rhs(N, p, uh)) < TOL_RHS_F32
    for _ in range(20 if N == 32 else 8):
        s.step(1e-3)
        uh = oracle.step(N, p, uh, 1e-3)
    assert rel(s.get_spectral()[0], uh) < TOL_STEPS_F32
    assert rel(s.get_fields()[0], oracle.get_fields(N, uh)) < 1e-4


def test_fp32_rhs_parity_128(ns, oracle):
    """fp32 RHS at 128^3 (L = 64 kernels) against the full fp64 oracle."""
    N = 128
    u = field(N, 428)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, dtype="f32", **kw)
    uh = oracle.set_initial(N, u)
    s.set_spectral(uh[None].astype(np.complex64))
    assert rel(s.rhs()[0], oracle.rhs(N, oracle.Params(**kw), uh)) < TOL_RHS_F32


@pytest.mark.parametrize("N", [256, 512])
def test_fp32_full_size_sampled(ns, oracle, k53_512, k53_512_hat, N):
    """fp32 at the sizes that run the long-line kernels (L = 128, 256: 16 values per lane, tensor-memory parking):
    ns_rhs at sampled wavenumbers against the oracle's direct truncated convolution, the whole array against the
    fp64 CUDA result (itself checked against the oracle in test_full_size_sampled_rhs_and_step), and one RK3 step."""
    u = inputs.gaussian_field(N, 256, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5) if N == 256 else k53_512
    uh = spectral_state(u) if N == 256 else k53_512_hat        # numpy restatement of set_initial: the common input
    kw = dict(eps=0.05, s=1.0)
    s64 = ns.Solver(N, **kw)
    s64.set_spectral(uh[None])
    del u
    r64 = s64.rhs()[0]
    dt = 0.2 * (2 * np.pi / N) / s64.max_velocity()[0]
    s64.step(dt)
    u64 = s64.get_spectral()[0]
    del s64
    s = ns.Solver(N, dtype="f32", **kw)
    s.set_spectral(uh[None].astype(np.complex64))
    r = s.rhs()[0]
    assert rel(r, r64) < TOL_RHS_F32
    rmax = np.abs(r64).max()
    modes = _sample_modes(N, 10, N + 1)
    want = oracle.rhs_at_modes(N, oracle.Params(**kw), uh, modes)
    got = np.stack([r[:, ix, iy, iz] for ix, iy, iz in modes])
    assert np.abs(got - want).max() < 2e-5 * rmax, np.abs(got - want).max() / rmax
    assert abs(s.max_velocity()[0] * dt / (0.2 * (2 * np.pi / N)) - 1.0) < 1e-5
    s.step(dt)
    assert rel(s.get_spectral()[0], u64) < TOL_RHS_F32


def test_nonfinite_state_is_reported(ns):
    """A NaN / inf in the state is detected on the device by the max|u| reduction of stage 1 (which propagates
    non-finite values), the sample is frozen, and the next synchronising call returns NS_ERR_NONFINITE naming it;
    ns_advance stops instead of spinning to max_steps; the other samples of the batch are unaffected."""
    N, B = 32, 3
    us = np.stack([field(N, 700 + i) for i in range(B)])
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, batch=B, **kw)
    s.set_initial(us)
    good = s.get_spectral()
    ref = ns.Solver(N, batch=B, **kw)
    ref.set_spectral(good)
    dts_ref = ref.step_cfl(0.2, 1e9)
    for value, sample in ((np.nan, 1), (np.inf, 2), (-np.inf, 0)):
        bad = good.copy()
        bad[sample, 0, 3, 2, 1] = value
        s.set_spectral(bad)
        t0 = [s.time(i) for i in range(B)]          # ns_set_spectral keeps the sample times
        with pytest.raises(ns.NSError) as e:
            s.step_cfl(0.2, 1e9)
        assert e.value.code == ns.NS_ERR_NONFINITE and f"sample {sample}" in str(e.value)
        got = s.get_spectral()
        for i in range(B):
            if i == sample:     # frozen: bit for bit the state that was set (NaN != NaN, so compare the bytes)
                assert got[i].tobytes() == bad[i].tobytes()
            else:
                assert np.array_equal(got[i], ref.get_spectral()[i])
        other = (sample + 1) % B
        assert s.time(sample) == t0[sample] and s.time(other) == t0[other] + dts_ref[other]
        with pytest.raises(ns.NSError) as e:
            s.advance(0.2, 1.0)
        assert e.value.code == ns.NS_ERR_NONFINITE
        with pytest.raises(ns.NSError) as e:
            s.max_velocity()
        assert e.value.code == ns.NS_ERR_NONFINITE
        # fixed-dt steps are asynchronous; the mark is reported by the next synchronising call
        s.set_spectral(bad)
        s.step(1e-3)
        with pytest.raises(ns.NSError) as e:
            s.step_dts(np.full(B, 1e-3))
        assert e.value.code == ns.NS_ERR_NONFINITE and f"sample {sample}" in str(e.value)
    s.set_spectral(good)                                  # a new state clears the mark
    assert np.array_equal(s.step_cfl(0.2, 1e9), dts_ref)
    assert np.isfinite(s.max_velocity()).all()


# ---------------------------------------------------------------------------------- errors / device buffers
def test_errors_and_device_buffers(ns):
    import torch
    N = 32
    s = ns.Solver(N)
    with pytest.raises(ns.NSError) as e:
        s.step(1e-3)
    assert e.value.code == ns.NS_ERR_STATE
    with pytest.raises(ns.NSError):
        s.rhs()
    u = field(N, 5)
    s.set_initial(torch.from_numpy(u[None]).cuda())              # device input
    host = s.get_spectral()
    dev = torch.empty(s.spectral_shape, dtype=torch.complex128, device="cuda")
    s.get_spectral(dev)
    torch.cuda.synchronize()
    assert np.array_equal(dev.cpu().numpy(), host)
    rdev = torch.empty_like(dev)
    s.rhs(rdev)
    torch.cuda.synchronize()
    assert np.array_equal(rdev.cpu().numpy(), s.rhs())
    with pytest.raises(ns.NSError) as e:
        s.energy_spectrum(0)
    assert e.value.code == ns.NS_ERR_INVALID_ARG
    n0 = s.kernel_launches()
    s.step(1e-3)
    assert s.kernel_launches() - n0 == 3 * 6 + 1      # 3 stages x (a1, a2, fused a3+a4, a5, a6, a7) + dt setup
    assert s.device_bytes() > 0
    # a non-default stream
    st = torch.cuda.Stream()
    s2 = ns.Solver(N, stream=st.cuda_stream)
    s2.set_initial(u[None])
    s2.step(1e-3)
    s.set_initial(u[None])
    s.step(1e-3)
    assert np.array_equal(s2.get_spectral(), s.get_spectral())
