"""GPU tests of the multi-device solver (include/ns_mg.h): one sample decomposed into ky / px slabs over P
ranks driven by one process.  This machine has ONE GPU, so the device list names device 0 several times: the P ranks share the
GPU, every slab pass, both exchanges, the event ordering between the rank streams and the cross-rank max|u| reduction run
exactly as they would over NVLink peers -- only the copies stay on one device.  Checked against the CPU oracle and, bit for
bit, against the single-device path of ns.h (per line the arithmetic is identical)."""
import numpy as np
import pytest

from paper_2401_09843_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ns():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_09843_b200 import binding
    binding.lib()
    return binding


def rel(a, b):
    return float(np.linalg.norm((np.asarray(a) - b).ravel()) / max(np.linalg.norm(np.asarray(b).ravel()), 1e-300))


def field(N, seed):
    u = inputs.gaussian_field(N, seed, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5)
    return u + 0.1 * inputs.normal01(seed, 3, 3 * N ** 3).reshape(3, N, N, N)


@pytest.mark.parametrize("N,P", [(64, 1), (64, 4), (96, 3)])
def test_mg_rhs_and_steps_against_the_oracle(ns, oracle, N, P):
    """RHS (every stored entry), max|u| and 3 CFL steps of the slab-decomposed solver against the oracle (which replays dt)."""
    kw = dict(nu=0.002, eps=0.05, s=1.0)
    uh = oracle.set_initial(N, field(N, 40 + N + P))
    s = ns.SolverMG(N, [0] * P, **kw)
    s.set_spectral(uh)
    assert np.array_equal(s.get_spectral(), uh)
    p = oracle.Params(**kw)
    want = oracle.rhs_parts(N, p, uh)
    r = s.rhs()
    assert rel(r, want["r"]) < 1e-12
    assert np.all(r[:, N // 2] == 0) and np.all(r[:, :, N // 2] == 0) and np.all(r[:, :, :, N // 2] == 0)
    assert abs(s.max_velocity() - want["umax"]) < 1e-13 * want["umax"]
    worst, tsum = 0.0, 0.0
    for i in range(3):
        dt = s.step_cfl(0.2, 1e9)
        assert abs(dt - 0.2 * (2 * np.pi / N) / oracle.max_velocity(N, uh)) < 1e-12 * dt
        tsum += dt
        uh = oracle.step(N, p, uh, dt)
        worst = max(worst, rel(s.get_spectral(), uh))
        assert worst < 1e-10, (i, worst)
    assert abs(s.time() - tsum) < 1e-13 * tsum
    assert s.exchange_bytes() == 8 * (3 * N // 2) * N * (N // 2) * 16 // P * (P - 1)
    print(f"N = {N}, P = {P}: worst rel-L2 over 3 steps {worst:.2e}; exchange {s.exchange_bytes() / 1e6:.1f} MB per RHS")


@pytest.mark.parametrize("N,P,dtype", [(128, 4, "f64"), (256, 2, "f64"), (256, 4, "f32")])
def test_mg_is_bitwise_the_single_device_result(ns, N, P, dtype):
    """Sizes that run the line-pair z kernel and the tensor-memory column kernels on slabs: RHS, per-step dt and the state after 3
    CFL steps + 1 fixed step are BIT-IDENTICAL to the single-device solver of ns.h (same kernels per line; the slab exchange only
    moves data, the max reduction is exact)."""
    kw = dict(eps=0.05, s=1.5, dtype=dtype)
    one = ns.Solver(N, **kw)
    one.set_initial(field(N, 7 + N)[None])
    uh = one.get_spectral()[0]
    s = ns.SolverMG(N, [0] * P, **kw)
    s.set_spectral(uh)
    assert np.array_equal(s.get_spectral(), uh)
    assert np.array_equal(s.rhs(), one.rhs()[0])
    assert s.max_velocity() == one.max_velocity()[0]
    for _ in range(3):
        assert s.step_cfl(0.2, 1e9) == one.step_cfl(0.2, 1e9)[0]
    s.step(1e-3)
    one.step(1e-3)
    assert np.array_equal(s.get_spectral(), one.get_spectral()[0])
    assert s.time() == one.time(0)
    assert s.kernel_launches() > 0 and s.device_bytes() > 0


def test_mg_errors(ns):
    with pytest.raises(ns.NSError):
        ns.SolverMG(64, [0, 0, 0])            # 64 is not divisible by 3
    with pytest.raises(ns.NSError):
        ns.SolverMG(64, [0, 99])              # no such device
    with pytest.raises(ns.NSError):
        ns.SolverMG(50, [0, 0])               # not a transform grid
    s = ns.SolverMG(64, [0, 0])
    with pytest.raises(ns.NSError):
        s.rhs()                               # no state yet
