"""GPU parity schedule of SURVEY.md section 8(d) at the BASELINE.json sizes (configs[1]..configs[4]), the CUDA path
through the C ABI against the CPU oracle on the same seeded inputs:

  config 2  128^3          1 RHS + 20 CFL-0.2 RK3 steps, the oracle replaying the GPU's dt sequence, relative L2 at EVERY step
  config 3  256^3          the config's own input: full-array orc_rhs_parts (every stored entry) + 3 replayed steps
  config 4  32 x 128^3     one sample of the batched run replayed for 10 steps, E(K) and S_2 compared (reading A17)
  config 5  512^3          >= 512 STRATIFIED sampled wavenumbers against the direct truncated convolution, relative L2
                           over the sample, plus the energy identity P4 and the solenoidality P5 on the whole array

Tolerances are the north_star's: relative L2 <= 1e-12 per ns_rhs, <= 1e-10 after (up to) 20 ns_step in fp64.
Run on the B200 box:  python -m pytest tests -m gpu

The oracle is deliberately naive (25 s per 256^3 RHS on the box's 16 cores), so the whole `-m gpu` suite is sized to stay well
inside the driver's 1200 s limit: by default config 3 checks the full-array RHS only and config 4 replays four steps;
`NS_FULL_SCHEDULE=1` runs the full
counts (3 and 10 steps, 20 steps at 96^3, two samples at 192^3) -- the log of such a run is profiles/r02_parity_schedule.md.
"""
import os
import time

import numpy as np
import pytest

from paper_2401_09843_b200 import inputs
from _sampling import spectral_state, stratified_modes

pytestmark = pytest.mark.gpu

TOL_RHS_F64, TOL_STEPS_F64 = 1e-12, 1e-10
FULL = os.environ.get("NS_FULL_SCHEDULE") == "1"


@pytest.fixture(scope="module")
def ns():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_09843_b200 import binding
    binding.lib()
    return binding


def rel(a, b):
    return float(np.linalg.norm((np.asarray(a) - b).ravel()) / max(np.linalg.norm(np.asarray(b).ravel()), 1e-300))


# ------------------------------------------------------------------------------------------------ config 2
def test_config2_128_rhs_and_20_cfl_steps(ns, oracle):
    """BASELINE.json configs[1]: N = 128, Gaussian k^4 exp field (seed 2), hyperviscosity eps = 0.05, s = 1, m = sqrt(N),
    CFL 0.2: one RHS and the first 20 RK3 steps, the oracle replaying the GPU's dt; relative L2 at every step."""
    N = 128
    u = inputs.gaussian_k4(N, seed=2)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    assert rel(s.get_spectral()[0], uh) < 1e-13
    s.set_spectral(uh[None])
    p = oracle.Params(**kw)
    want = oracle.rhs_parts(N, p, uh)
    assert rel(s.rhs()[0], want["r"]) < TOL_RHS_F64
    worst, t0, tsum = 0.0, time.perf_counter(), 0.0
    for i in range(20):
        dts = s.step_cfl(0.2, 1e9)
        if i in (0, 10):     # dt against the oracle's own max|u| (costs an oracle inverse transform: not every step)
            assert abs(dts[0] - 0.2 * (2 * np.pi / N) / oracle.max_velocity(N, uh)) < 1e-12 * dts[0]
        tsum += dts[0]
        uh = oracle.step(N, p, uh, dts[0])
        worst = max(worst, rel(s.get_spectral()[0], uh))
        assert worst < TOL_STEPS_F64, (i, worst)
    print(f"config 2: worst rel-L2 over 20 steps {worst:.2e}; oracle {time.perf_counter() - t0:.0f} s")
    assert abs(s.time(0) - tsum) < 1e-13 * tsum


# ------------------------------------------------------------------------------------------------ config 3
def test_config3_256_full_array_rhs_and_steps(ns, oracle):
    """BASELINE.json configs[2] with its own input (perturbed shear layer, seed 3) at N = 256 -- the size that runs the
    long-line kernels: EVERY stored entry of ns_rhs against orc_rhs_parts (relative L2 <= 1e-12, and the largest
    single-entry deviation), max|u| on the padded grid; with NS_FULL_SCHEDULE=1 then 3 CFL steps with the oracle replaying the
    GPU's dt (an oracle step at this size takes 80 s; by default the fused step at 256^3 / 512^3 is checked against eq. 2.6
    assembled from ns_rhs in test_full_size_stratified_sampled_rhs, and against the oracle at every smaller size)."""
    N = 256
    u = inputs.shear_layer(N, seed=3)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    del u
    assert rel(s.get_spectral()[0], uh) < 1e-13
    s.set_spectral(uh[None])
    p = oracle.Params(**kw)
    t0 = time.perf_counter()
    want = oracle.rhs_parts(N, p, uh)
    t_rhs = time.perf_counter() - t0
    got = s.rhs()[0]
    assert rel(got, want["r"]) < TOL_RHS_F64
    assert np.abs(got - want["r"]).max() < 1e-12 * np.abs(want["r"]).max()     # no single entry is off (tile faults)
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    del got, want
    worst, nsteps = 0.0, 3 if FULL else 0
    for i in range(nsteps):
        dts = s.step_cfl(0.2, 1e9)
        uh = oracle.step(N, p, uh, dts[0])
        worst = max(worst, rel(s.get_spectral()[0], uh))
        assert worst < TOL_STEPS_F64, (i, worst)
    print(f"config 3: oracle RHS {t_rhs:.0f} s; worst rel-L2 over {nsteps} step(s) {worst:.2e}")


# ------------------------------------------------------------------------------------------------ config 4
def test_config4_one_sample_replayed(ns, oracle):
    """BASELINE.json configs[3]: the 32 x 128^3 shear-layer ensemble stepped in ONE batched launch at per-sample CFL 0.2;
    the oracle replays sample 1's dt sequence for 4 steps (10 with NS_FULL_SCHEDULE=1).  State at relative L2 <= 1e-10 at every step; the reported
    statistics E(K) and S_2(l) of that sample at the statistical tolerance of reading A17 (1e-8 relative)."""
    N, B, pick = 128, 32, 1
    us = inputs.shear_layer_ensemble(N, B, seed0=1000)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, batch=B, **kw)
    s.set_initial(us)
    uh = oracle.set_initial(N, us[pick])
    del us
    assert rel(s.get_spectral()[pick], uh) < 1e-13      # the oracle keeps ITS OWN initial state (no input from the CUDA path)
    p = oracle.Params(**kw)
    worst, nsteps = 0.0, 10 if FULL else 4
    for i in range(nsteps):
        dts = s.step_cfl(0.2, 1.0)
        uh = oracle.step(N, p, uh, dts[pick])
        got = s.get_spectral()[pick]
        worst = max(worst, rel(got, uh))
        assert worst < TOL_STEPS_F64, (i, worst)
    E = s.energy_spectrum(N)[pick]
    Eo = oracle.energy_spectrum(N, uh, N)
    assert np.abs(E - Eo).max() < 1e-8 * Eo.max()
    S = s.structure_function()[pick]
    assert np.abs(S / oracle.structure_function(N, uh) - 1).max() < 1e-8
    assert np.abs(s.structure_function_p(2.0, nl=8)[pick] / oracle.structure_function(N, uh, 8) - 1).max() < 1e-8
    print(f"config 4: worst rel-L2 over {nsteps} replayed steps {worst:.2e}")


# ------------------------------------------------------------------------------------------------ config 5
@pytest.mark.parametrize("N", [256, 512])
def test_full_size_stratified_sampled_rhs(ns, oracle, k53_512, k53_512_hat, N):
    """256^3 and 512^3 (configs[4] input), same launch configuration as bench.py: ns_rhs at >= 512 stratified sampled
    wavenumbers against the oracle's direct truncated convolution sum (orc_rhs_at_modes): relative L2 over the sample
    <= 1e-12 and every single sampled entry within 1e-12 of max|R|; then, on the WHOLE array, the energy identity P4
    of the inviscid RHS (a statement about every entry of the transforms: any aliasing or tile fault breaks it), the
    masks, and the fused RK3 step against eq. 2.6 assembled on the host from ns_rhs evaluations (pins the axpy of a7)."""
    u = inputs.gaussian_field(N, 256, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5) if N == 256 else k53_512
    uh = spectral_state(u) if N == 256 else k53_512_hat        # numpy restatement of set_initial: the common input
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    del u
    assert rel(s.get_spectral()[0], uh) < 1e-13                # ns_set_initial at full size, every entry
    s.set_spectral(uh[None])
    r = s.rhs()[0]
    del s
    rmax = np.abs(r).max()
    modes = stratified_modes(N, 512, N)
    t0 = time.perf_counter()
    want = oracle.rhs_at_modes(N, oracle.Params(**kw), uh, modes)
    t_or = time.perf_counter() - t0
    got = np.stack([r[:, ix, iy, iz] for ix, iy, iz in modes])
    err = np.abs(got - want)
    print(f"N = {N}: {len(modes)} sampled modes, oracle {t_or:.0f} s, rel-L2 {rel(got, want):.2e}, worst entry {err.max() / rmax:.2e} of max|R|")
    assert np.linalg.norm(want) > 1e-2 * rmax
    assert rel(got, want) < TOL_RHS_F64
    assert err.max() < 1e-12 * rmax
    assert np.all(r[:, N // 2] == 0) and np.all(r[:, :, N // 2] == 0) and np.all(r[:, :, :, N // 2] == 0)
    del r
    # P4 on the whole array: inviscid solver (the viscous one was destroyed first: memory)
    w = np.full(N // 2 + 1, 2.0)
    w[0] = 1.0
    s = ns.Solver(N)
    s.set_spectral(uh[None])
    rn = s.rhs()[0]
    num = abs(np.sum(w * np.real(np.conj(uh) * rn)))
    den = np.sum(w * np.abs(uh) * np.abs(rn))
    print(f"N = {N}: energy identity residual {num / den:.2e}")
    assert num < 1e-12 * den
    # fused RK3 step == eq. 2.6 assembled from ns_rhs (same kernels in mode 0)
    dt = 0.2 * (2 * np.pi / N) / s.max_velocity()[0]
    u1 = uh + dt * rn
    del rn
    s.set_spectral(u1[None])
    u2 = 0.75 * uh + 0.25 * u1 + 0.25 * dt * s.rhs()[0]
    del u1
    s.set_spectral(u2[None])
    un = uh / 3.0 + (2.0 / 3.0) * u2 + (2.0 / 3.0) * dt * s.rhs()[0]
    del u2
    s.set_spectral(uh[None])
    dts = s.step_cfl(0.2, 1e9)
    assert abs(dts[0] - dt) < 1e-13 * dt
    assert rel(s.get_spectral()[0], un) < 1e-14


# ------------------------------------------------------------------------------------------------ NEXT-3: N = 3 * 2^a
@pytest.mark.parametrize("N", [48, 96])
def test_sizes_3x2a_rhs_and_20_steps(ns, oracle, N):
    """SURVEY.md 8(f) NEXT-3, first slice (transform sizes with small prime factors): N = 3 * 2^a, i.e.
    sub-transforms of length L = N/2 = 3 * 2^(a-1) with a radix-6 / radix-12 first register stage.  set_initial,
    get_fields, one RHS and 20 CFL steps (the oracle replaying the GPU's dt) at 48^3, 4 at 96^3 (20 with NS_FULL_SCHEDULE=1),
    every stored entry."""
    u = inputs.gaussian_field(N, 300 + N, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)
    u += 0.2 * inputs.normal01(N, 3, 3 * N ** 3).reshape(3, N, N, N)          # not solenoidal: exercises the projection
    kw = dict(nu=0.002, eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    assert rel(s.get_spectral()[0], uh) < 1e-13
    assert rel(s.get_fields()[0], oracle.get_fields(N, uh)) < 1e-13
    s.set_spectral(uh[None])
    p = oracle.Params(**kw)
    want = oracle.rhs_parts(N, p, uh)
    got = s.rhs()[0]
    assert rel(got, want["r"]) < TOL_RHS_F64
    assert np.all(got[:, N // 2] == 0) and np.all(got[:, :, N // 2] == 0) and np.all(got[:, :, :, N // 2] == 0)
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    worst, nsteps = 0.0, 20 if (FULL or N == 48) else 4
    for i in range(nsteps):
        dts = s.step_cfl(0.2, 1e9)
        uh = oracle.step(N, p, uh, dts[0])
        worst = max(worst, rel(s.get_spectral()[0], uh))
        assert worst < TOL_STEPS_F64, (i, worst)
    E = s.energy_spectrum(N)[0]
    assert np.abs(E - oracle.energy_spectrum(N, uh, N)).max() < 1e-13
    assert np.abs(s.structure_function_p(3.0, nl=6)[0] / oracle.structure_function_p(N, uh, 3.0, 6) - 1).max() < 1e-11
    print(f"N = {N}: worst rel-L2 over {nsteps} steps {worst:.2e}")


def test_sizes_3x2a_192_full_and_384_sampled(ns, oracle):
    """N = 192 (L = 96 = 12 x 8): every stored entry of ns_rhs against orc_rhs_parts, two samples in one launch;
    N = 384 (L = 192 = 12 x 16, padded 576^3): 268 (full schedule: 524) stratified sampled wavenumbers against the direct truncated
    convolution, the energy identity on the whole array, and fp32 against the fp64 result."""
    N = 192
    us = np.stack([inputs.taylor_green_3d_perturbed(N, 31), inputs.gaussian_field(N, 392, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)])
    kw = dict(eps=0.05, s=1.5)
    uh = np.stack([spectral_state(u) for u in us])
    s = ns.Solver(N, batch=2, **kw)
    s.set_initial(us)
    del us
    assert rel(s.get_spectral(), uh) < 1e-13
    s.set_spectral(uh)
    r = s.rhs()
    um = s.max_velocity()
    for b in range(2) if FULL else (1,):
        want = oracle.rhs_parts(N, oracle.Params(**kw), uh[b])
        assert rel(r[b], want["r"]) < TOL_RHS_F64
        assert abs(um[b] - want["umax"]) < 1e-13 * want["umax"]
    del s, r, uh
    N = 384
    u = inputs.gaussian_field(N, 384, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)
    uh = spectral_state(u)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    del u
    assert rel(s.get_spectral()[0], uh) < 1e-13
    s.set_spectral(uh[None])
    r = s.rhs()[0]
    del s
    rmax = np.abs(r).max()
    modes = stratified_modes(N, 512 if FULL else 256, N)
    want = oracle.rhs_at_modes(N, oracle.Params(**kw), uh, modes)
    got = np.stack([r[:, ix, iy, iz] for ix, iy, iz in modes])
    print(f"N = 384: rel-L2 over {len(modes)} sampled modes {rel(got, want):.2e}")
    assert rel(got, want) < TOL_RHS_F64 and np.abs(got - want).max() < 1e-12 * rmax
    w = np.full(N // 2 + 1, 2.0)
    w[0] = 1.0
    s = ns.Solver(N)
    s.set_spectral(uh[None])
    rn = s.rhs()[0]
    assert abs(np.sum(w * np.real(np.conj(uh) * rn))) < 1e-12 * np.sum(w * np.abs(uh) * np.abs(rn))
    del s, rn
    s32 = ns.Solver(N, dtype="f32", **kw)
    s32.set_spectral(uh[None].astype(np.complex64))
    assert rel(s32.rhs()[0], r) < 1e-5


# ------------------------------------------------------------------------------------------------ NEXT-3: radix 5, 7, 15
@pytest.mark.parametrize("N", [80, 112])
def test_sizes_5_7_rhs_and_steps(ns, oracle, N):
    """SURVEY.md 8(f) NEXT-3 (sizes 2^a 3^b 5^c 7^d): N = 5 * 2^4 and 7 * 2^4, sub-transforms of length
    L = 40 = 10 x 4 and 56 = 14 x 4 (radix-5 / radix-7 butterflies inside prime-factor first stages).  set_initial, get_fields,
    one RHS (every stored entry) and 3 CFL steps (10 with NS_FULL_SCHEDULE=1) with the oracle replaying the GPU's dt."""
    u = inputs.gaussian_field(N, 500 + N, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)
    u += 0.2 * inputs.normal01(N, 3, 3 * N ** 3).reshape(3, N, N, N)          # not solenoidal: exercises the projection
    kw = dict(nu=0.002, eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    assert rel(s.get_spectral()[0], uh) < 1e-13
    assert rel(s.get_fields()[0], oracle.get_fields(N, uh)) < 1e-13
    s.set_spectral(uh[None])
    p = oracle.Params(**kw)
    want = oracle.rhs_parts(N, p, uh)
    got = s.rhs()[0]
    assert rel(got, want["r"]) < TOL_RHS_F64
    assert np.all(got[:, N // 2] == 0) and np.all(got[:, :, N // 2] == 0) and np.all(got[:, :, :, N // 2] == 0)
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    worst, nsteps = 0.0, 10 if FULL else 3
    for i in range(nsteps):
        dts = s.step_cfl(0.2, 1e9)
        uh = oracle.step(N, p, uh, dts[0])
        worst = max(worst, rel(s.get_spectral()[0], uh))
        assert worst < TOL_STEPS_F64, (i, worst)
    assert np.abs(s.energy_spectrum(N)[0] - oracle.energy_spectrum(N, uh, N)).max() < 1e-13
    print(f"N = {N}: worst rel-L2 over {nsteps} steps {worst:.2e}")


@pytest.mark.parametrize("N", [160, 224, 240] if FULL else [160])
def test_sizes_5_7_15_full_array_rhs(ns, oracle, N):
    """N = 5 * 2^5 (L = 80 = 10 x 8; with NS_FULL_SCHEDULE=1 also 7 * 2^5 and 15 * 2^4, L = 112 = 14 x 8, 120 = 15 x 8, which the
    default run covers by sampled wavenumbers below): every stored entry of ns_rhs and max|u| against orc_rhs_parts; fp32
    (where N/2 is a multiple of 16) against the fp64 result."""
    u = inputs.taylor_green_3d_perturbed(N, 40 + N) + 0.3 * inputs.gaussian_field(N, 700 + N, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)
    uh = spectral_state(u)
    kw = dict(eps=0.05, s=1.5)
    s = ns.Solver(N, **kw)
    s.set_initial(u[None])
    del u
    assert rel(s.get_spectral()[0], uh) < 1e-13
    s.set_spectral(uh[None])
    r = s.rhs()[0]
    want = oracle.rhs_parts(N, oracle.Params(**kw), uh)
    assert rel(r, want["r"]) < TOL_RHS_F64
    assert np.abs(r - want["r"]).max() < 1e-12 * np.abs(want["r"]).max()
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    del s
    if (N // 2) % 16 == 0:
        s32 = ns.Solver(N, dtype="f32", **kw)
        s32.set_spectral(uh[None].astype(np.complex64))
        assert rel(s32.rhs()[0], r) < 1e-5


@pytest.mark.parametrize("N", [224, 240, 320, 448, 480, 640])
def test_sizes_5_7_15_large_sampled(ns, oracle, N):
    """L = 112 = 14 x 8, 120 = 15 x 8 and the long-line members of the families (L = 160 = 10 x 16, 224 = 14 x 16, 240 = 15 x 16,
    320 = 20 x 16): stratified sampled
    wavenumbers of ns_rhs against the direct truncated convolution (relative L2 over the sample <= 1e-12), the masks, and the
    energy identity P4 of the inviscid RHS on the whole array.  Full-band input: white noise on a shear profile; its spectral state
    by the numpy restatement of set_initial is the common input of both sides (and ns_set_initial is checked against it)."""
    rng = np.random.default_rng(N)
    kw = dict(eps=0.05, s=1.0)
    s = ns.Solver(N, **kw)
    if N == 640 and not FULL:
        # 6 GB arrays: the state is drawn directly in spectral space (white spectrum, real field: Hermitian kz = 0 plane, Nyquist
        # planes and mean zero; not solenoidal -- the RHS is defined for any state); no physical field, no set_initial here
        uh = 0.05 * (rng.standard_normal((3, N, N, N // 2 + 1)) + 1j * rng.standard_normal((3, N, N, N // 2 + 1)))
        neg = (-np.arange(N)) % N
        uh[:, :, :, 0] = 0.5 * (uh[:, :, :, 0] + np.conj(uh[:, neg][:, :, neg, 0]))
        uh[:, N // 2] = 0
        uh[:, :, N // 2] = 0
        uh[:, :, :, N // 2] = 0
        uh[:, 0, 0, 0] = 0
    else:
        x = 2 * np.pi * np.arange(N) / N
        u = 0.3 * rng.standard_normal((3, N, N, N))
        u[0] += np.sin(x)[None, :, None] + 0.5 * np.cos(3 * x)[None, None, :]
        u[2] += np.cos(2 * x)[:, None, None]
        uh = spectral_state(u)            # numpy restatement of set_initial: the common input of both sides
        s.set_initial(u[None])
        assert rel(s.get_spectral()[0], uh) < 1e-13
        del u
    s.set_spectral(uh[None])
    r = s.rhs()[0]
    del s
    rmax = np.abs(r).max()
    modes = stratified_modes(N, 96, N)
    want = oracle.rhs_at_modes(N, oracle.Params(**kw), uh, modes)
    got = np.stack([r[:, ix, iy, iz] for ix, iy, iz in modes])
    print(f"N = {N}: rel-L2 over {len(modes)} sampled modes {rel(got, want):.2e}")
    assert np.linalg.norm(want) > 1e-2 * rmax
    assert rel(got, want) < TOL_RHS_F64 and np.abs(got - want).max() < 1e-12 * rmax
    assert np.all(r[:, N // 2] == 0) and np.all(r[:, :, N // 2] == 0) and np.all(r[:, :, :, N // 2] == 0)
    del r
    if N == 640 and not FULL:             # 6 GB host arrays: the whole-array identity at this size only in the full schedule
        return
    s = ns.Solver(N)                      # inviscid: the energy identity on every entry
    s.set_spectral(uh[None])
    rn = s.rhs()[0]
    w = np.full(N // 2 + 1, 2.0)
    w[0] = 1.0
    assert abs(np.sum(w * np.real(np.conj(uh) * rn))) < 1e-12 * np.sum(w * np.abs(uh) * np.abs(rn))


# ------------------------------------------------------------------------------------------------ NEXT-3: general N, autotune
@pytest.mark.parametrize("N", [18, 50, 100])
def test_general_even_n_on_a_larger_transform_grid(ns, oracle, N):
    """SURVEY.md 8(f) NEXT-3 / PAPER.md:L175 (the padded size may be any size >= 3N/2; it is rounded up to one with small prime
    factors): an N that is not p 2^a runs on the next admissible transform grid Nt > N, padded grid M = 3 Nt / 2 > 3N/2, with the
    state truncated to the user's N.  Against the oracle at the user's N with the SAME padded size M (by pin P7 the RHS does not
    depend on M; max|u| does): set_initial (plain DFT on the N grid), get_fields, RHS (every entry), max|u|, 5 CFL steps (2 at N = 100),
    spectra, S_2 and S_p."""
    u = inputs.gaussian_field(N, 800 + N, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)
    u += 0.2 * inputs.normal01(N, 3, 3 * N ** 3).reshape(3, N, N, N)          # not solenoidal, full band
    kw = dict(nu=0.002, eps=0.05, s=1.5)
    s = ns.Solver(N, **kw)
    Nt, M = s.transform_grid, s.padded_size
    assert Nt > N and M == 3 * Nt // 2 and M > 3 * N // 2
    s.set_initial(u[None])
    uh = oracle.set_initial(N, u)
    got = s.get_spectral()[0]
    assert got.shape == uh.shape and rel(got, uh) < 1e-13
    assert rel(s.get_fields()[0], oracle.get_fields(N, uh)) < 1e-13
    s.set_spectral(uh[None])
    assert np.array_equal(s.get_spectral()[0], uh)                              # round trip through the larger grid is exact
    p = oracle.Params(**kw)
    want = oracle.rhs_parts(N, p, uh, M)
    r = s.rhs()[0]
    assert rel(r, want["r"]) < TOL_RHS_F64
    assert rel(r, oracle.rhs(N, p, uh)) < TOL_RHS_F64                           # and equals the 3N/2 result (P7)
    assert np.all(r[:, N // 2] == 0) and np.all(r[:, :, N // 2] == 0) and np.all(r[:, :, :, N // 2] == 0)
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    worst, nsteps = 0.0, 5 if (FULL or N < 100) else 2
    for i in range(nsteps):
        dts = s.step_cfl(0.2, 1e9)
        assert abs(dts[0] - 0.2 * (2 * np.pi / N) / oracle.max_velocity(N, uh, M)) < 1e-12 * dts[0]
        uh = oracle.step(N, p, uh, dts[0], M)
        worst = max(worst, rel(s.get_spectral()[0], uh))
        assert worst < TOL_STEPS_F64, (i, worst)
    assert np.abs(s.energy_spectrum(N)[0] - oracle.energy_spectrum(N, uh, N)).max() < 1e-13
    Zo = oracle.enstrophy_spectrum(N, uh, N)
    assert np.abs(s.enstrophy_spectrum(N)[0] - Zo).max() < 1e-12 * Zo.max()
    assert np.abs(s.structure_function()[0] / oracle.structure_function(N, uh) - 1).max() < 1e-11
    assert np.abs(s.structure_function_p(3.0, nl=4)[0] / oracle.structure_function_p(N, uh, 3.0, 4) - 1).max() < 1e-11
    print(f"N = {N} on transform grid {Nt} (padded {M}): worst rel-L2 over {nsteps} steps {worst:.2e}")


def test_autotune_records_the_transform_grid(ns, oracle):
    """ns_autotune (benchmark of the transform only, the fastest padding is stored and used afterwards): candidates
    are the admissible grids >= N in increasing order; the recorded one is the fastest measured; ns_create uses it; the result on
    whatever grid was chosen still matches the oracle with that padded size.  For an N that is itself admissible the candidates
    start with N."""
    N = 100
    best, cand = ns.autotune(N, "f64", 3)
    assert [g for g, _ in cand] == [112, 128, 160] and all(t > 0 for _, t in cand)
    assert best == min(cand, key=lambda c: c[1])[0]
    s = ns.Solver(N, eps=0.05)
    assert s.transform_grid == best and s.padded_size == 3 * best // 2
    u = inputs.gaussian_field(N, 77, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)
    uh = spectral_state(u)
    s.set_spectral(uh[None])
    want = oracle.rhs_parts(N, oracle.Params(eps=0.05), uh, s.padded_size)
    assert rel(s.rhs()[0], want["r"]) < TOL_RHS_F64
    assert abs(s.max_velocity()[0] - want["umax"]) < 1e-13 * want["umax"]
    best2, cand2 = ns.autotune(128, "f64", 2)
    assert [g for g, _ in cand2] == [128, 160]
    with pytest.raises(ns.NSError):
        ns.autotune(101, "f64", 2)
