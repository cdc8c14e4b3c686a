"""The state stays the spectrum of a REAL field over long runs (reading A25).

The state lives in Fourier space for the whole run.  On the planes kx = 0 and kx = nx/2 the half-spectrum holds both
members of every conjugate pair; rounding breaks phi(-k) = conj(phi(k)) there, the C2R transforms never see the
anti-Hermitian part, and Eq. 18 amplifies it by 1/(1 - dt L_q) per step wherever L_q > 0.  Before the projection of
pss.cu (k_hermitize, every pss_hermitian_period()-th step of the absolute step count) the headline workload was NaN after 2 10^4 steps."""
import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pss():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_02410_b200 as p
    p.binding.lib()
    return p


def anti_hermitian(spec):
    """max |phi(k) - conj(phi(-k))| over the planes kx = 0 and kx = nx/2 of a logical half-spectrum [kz][ky][kx]"""
    worst = 0.0
    for col in (0, spec.shape[-1] - 1):
        p = spec[..., col].astype(np.complex128)
        m = p
        for ax in range(p.ndim):
            m = np.roll(np.flip(m, axis=ax), 1, axis=ax)
        worst = max(worst, float(np.abs(p - np.conj(m)).max()))
    return worst


@pytest.mark.parametrize("name,n,steps,kernel", [("modelb_1024", (1024, 1024), 30000, "k_persist2d"),
                                                 ("sweep_256", (256, 256), 30000, None),
                                                 ("modelb_256c", (32, 32, 32), 12000, None),
                                                 ("modelb_128", (256,), 30000, None)])
def test_long_run_keeps_the_state_hermitian_and_finite(pss, name, n, steps, kernel):
    cfg = wl.make_config(name, n=n)
    g, ids = wl.build(pss, cfg, prec="f32")
    assert g.fused_kernel_name == kernel
    phi = ids["phi"]
    g.step(steps)
    spec = g.get_field_fourier(phi)
    assert np.isfinite(spec.view(np.float32)).all()
    big = float(np.abs(spec).max())
    assert anti_hermitian(spec) <= 1e-4 * big, (anti_hermitian(spec), big)      # a few steps of rounding, not e^(t/4)
    x = g.get_field(phi)
    assert np.isfinite(x).all() and float(np.abs(x).max()) < 2.0                   # inside the double well (|phi| ~ 1)
    period = g.hermitian_period
    assert period == (128 if name == "nematic_1024" else 1024)
    g.step(period - g.step_count % period)                                        # straight after a projection: exact
    spec = g.get_field_fourier(phi)
    assert anti_hermitian(spec) == 0.0


@pytest.mark.parametrize("name,n", [("modelb_1024", (1024, 1024)), ("modelb_128", (64, 64)), ("nematic_1024", (32, 32)),
                                    ("modelb_256c", (16, 16, 32)), ("modelb_128", (128,))])
def test_projection_keeps_step_splitting_and_checkpoints_bit_identical(pss, name, n):
    """the projection is tied to the absolute step number: pss_step(a); pss_step(b) == pss_step(a + b) across it, and a
    checkpoint taken exactly on a projection step (or anywhere else) resumes bit for bit"""
    cfg = wl.make_config(name, n=n)
    dyn_names = list(cfg["ic"].keys())
    whole, ids = wl.build(pss, cfg, prec="f32")
    PERIOD = whole.hermitian_period
    assert PERIOD == (128 if name == "nematic_1024" else 1024)
    whole.step(2 * PERIOD + 44)
    want = {nm: whole.get_field_fourier(ids[nm]).view(np.uint32) for nm in dyn_names}
    split, _ = wl.build(pss, cfg, prec="f32")
    for k in (PERIOD - 28, 28, 1, PERIOD - 1, 44):                                # calls end on both projection steps among others
        split.step(k)
    assert split.step_count == whole.step_count
    for nm in dyn_names:
        assert np.array_equal(split.get_field_fourier(ids[nm]).view(np.uint32), want[nm]), nm
    for at in (PERIOD, PERIOD + 7):
        a, _ = wl.build(pss, cfg, prec="f32")
        a.step(at)
        ckpt = {nm: a.get_field_fourier(ids[nm]) for nm in dyn_names}
        c, _ = wl.build(pss, cfg, prec="f32", set_ic=False)
        for nm in dyn_names:
            c.set_field_fourier(ids[nm], ckpt[nm])
        c.set_step_count(at)
        c.step(2 * PERIOD + 44 - at)
        for nm in dyn_names:
            assert np.array_equal(c.get_field_fourier(ids[nm]).view(np.uint32), want[nm]), (nm, at)
