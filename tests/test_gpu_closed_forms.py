"""The CUDA path against closed forms the paper and the mathematics fix (no oracle involved): the same pins the
oracle is held to (P3, P4, P10, P11 of DESIGN.md), run through the C ABI on the GPU."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pss():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_02410_b200 as p
    p.binding.lib()
    return p


@pytest.mark.parametrize("n,dx", [((64,), (0.5,)), ((32, 64), (1.0, 0.7)), ((1024, 1024), (1.0, 1.0)), ((16, 8, 32), (1.0, 2.0, 0.5))])
def test_p4_linear_diffusion_mode_decay(pss, n, dx):
    """noiseless dt phi + D q^2 phi = 0: every mode equals phi_q(0) (1 + dt D q^2)^-steps (Eq. 18)"""
    D, dt, steps = 0.8, 0.05, 7
    s = pss.System(n, dx, dt, prec="f64", seed=1)
    f = s.add_field("phi", True)
    s.add_linear(f, {"coef": D, "q2_pow": 1})
    s.finalize()
    x0 = np.random.default_rng(2).standard_normal(n[::-1])
    s.set_field(f, x0)
    s.step(steps)
    spec0 = np.fft.rfftn(x0)
    qs = [2 * np.pi * np.fft.fftfreq(nj, dj) for nj, dj in zip(n, dx)]
    qs[0] = qs[0][: n[0] // 2 + 1].copy()
    qs[0][-1] = np.pi / dx[0]
    grids = np.meshgrid(*qs[::-1], indexing="ij")
    q2 = sum(g ** 2 for g in grids)
    want = spec0 / (1 + dt * D * q2) ** steps
    got = s.get_field_fourier(f)
    assert np.max(np.abs(got - want)) <= 1e-11 * np.max(np.abs(want))


@pytest.mark.parametrize("prec,tol", [("f32", 2e-6), ("f64", 1e-13)])
def test_p3_uniform_cubic_decay_recurrence(pss, prec, tol):
    """dt phi = -phi^3 on a uniform field (Eq. 4): exactly phi_{n+1} = phi_n - dt phi_n^3, and close to
    the closed form phi0 / sqrt(1 + 2 phi0^2 t)"""
    dt, steps, phi0 = 0.01, 200, 0.9
    s = pss.System((64, 32), (1.0, 1.0), dt, prec=prec, seed=1)
    f = s.add_field("phi", True)
    s.add_term(f, {"coef": -1.0}, [f, f, f])
    s.set_dealias(pss.DEALIAS_OFF)
    s.finalize()
    s.set_field(f, np.full((32, 64), phi0))
    s.step(steps)
    v = phi0
    for _ in range(steps):
        v = v - dt * v ** 3
    x = s.get_field(f).astype(np.float64)
    assert np.max(np.abs(x - v)) <= tol
    assert abs(v - phi0 / np.sqrt(1 + 2 * phi0 ** 2 * dt * steps)) < 5e-3


def test_p11_kpz_single_mode_one_step(pss):
    """h = A cos(q x), one noiseless KPZ step (Eq. 12; A15): mode 0 gains dt (lam/2) A^2 q^2 / 2 * N,
    mode 2q gets -dt (lam/2) A^2 q^2 / 4 * N / (1 + dt nu (2q)^2), mode q decays by 1 / (1 + dt nu q^2)"""
    nx, ny, A, nu, lam, dt, m = 64, 32, 0.3, 1.0, 2.0, 0.01, 3
    s = pss.System((nx, ny), (1.0, 1.0), dt, prec="f64", seed=1)
    h = s.add_field("h", True)
    gx = s.add_field("gx", False)
    gy = s.add_field("gy", False)
    s.add_aux_def(gx, {"coef": 1.0, "iq_pow": (1, 0, 0)}, h)
    s.add_aux_def(gy, {"coef": 1.0, "iq_pow": (0, 1, 0)}, h)
    s.add_linear(h, {"coef": nu, "q2_pow": 1})
    s.add_term(h, {"coef": 0.5 * lam}, [gx, gx])
    s.add_term(h, {"coef": 0.5 * lam}, [gy, gy])
    s.finalize()
    q = 2 * np.pi * m / nx
    x = np.arange(nx)
    s.set_field(h, np.tile(A * np.cos(q * x), (ny, 1)))
    s.step(1)
    spec = s.get_field_fourier(h)
    N = nx * ny
    assert abs(spec[0, 0] - dt * (lam / 2) * A ** 2 * q ** 2 / 2 * N) <= 1e-9 * N
    assert abs(spec[0, 2 * m] - (-dt * (lam / 2) * A ** 2 * q ** 2 / 4 * N / (1 + dt * nu * (2 * q) ** 2))) <= 1e-9 * N
    assert abs(spec[0, m] - (A / 2 * N) / (1 + dt * nu * q ** 2)) <= 1e-9 * N
    mask = np.ones_like(spec, dtype=bool)
    mask[0, [0, m, 2 * m]] = False
    assert np.max(np.abs(spec[mask])) <= 1e-9 * N


def test_p10_rotation_growth_factor(pss):
    """dt u = v, dt v = -u as explicit linear cross terms from time-t values (A11): u^2 + v^2 grows by exactly
    (1 + dt^2) per step"""
    dt, steps = 0.05, 10
    s = pss.System((32, 16), (1.0, 1.0), dt, prec="f64", seed=1)
    u = s.add_field("u", True)
    v = s.add_field("v", True)
    s.add_term(u, {"coef": 1.0}, [v])
    s.add_term(v, {"coef": -1.0}, [u])
    s.finalize()
    rng = np.random.default_rng(4)
    u0, v0 = rng.standard_normal((16, 32)), rng.standard_normal((16, 32))
    s.set_field(u, u0)
    s.set_field(v, v0)
    s.step(steps)
    e = s.get_field(u) ** 2 + s.get_field(v) ** 2
    assert np.max(np.abs(e / (u0 ** 2 + v0 ** 2) - (1 + dt ** 2) ** steps)) <= 1e-12
