"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (one pss_step(n)
call per run of n steps), against the CPU oracle on the same seeded inputs and the same noise stream.

Tolerances: north_star — relative L2 <= 1e-5 after 1 step, <= 1e-3 after 1000 steps (fp32);
<= 1e-12 / 1e-9 (fp64).  Config 4 (nematic): 250-step horizon, reading A20 of DESIGN.md.
Intermediate horizons (10-20 steps) use 10x the 1-step tolerance.
"""
import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as wl

pytestmark = pytest.mark.gpu

import os

import parity_util as pu
from parity_util import TOL1, TOLN, rel_l2


@pytest.fixture(scope="module")
def pss():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_02410_b200 as p
    p.binding.lib()
    return p


def both(pss, oracle, cfg, prec):
    return pu.both(wl, pss, oracle, cfg, prec)


def check(g, o, dyn, tol, what):
    return pu.compare_fields(g, o, dyn, tol, what)


def run_horizons(pss, oracle, cfg, prec, horizons, what):
    return pu.run_horizons(wl, pss, oracle, cfg, prec, horizons, what)


# Long horizon of the two configurations whose oracle takes minutes per 1000 steps (256^3: ~2.4 steps/s, KPZ 4096^2:
# ~1.3 steps/s on 16 cores).  Default: 200 / 100 steps at FULL size so that the whole `-m gpu` suite stays inside the
# driver's time limit; the 1000-step tolerance itself is tested on 64^3 / 512^2 in test_gpu_parity.py, and
# PSS_FULL_HORIZON=1000 runs the full-size comparison to 1000 steps (result recorded in DESIGN.md section 3).
FULL_HORIZON = int(os.environ.get("PSS_FULL_HORIZON", "0"))


# config 2: 2D Model B 1024^2, fp32 (the headline; persistent fused kernel) and fp64 (generic kernels)
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_config2_modelb_1024_1000_steps(pss, oracle, prec):
    cfg = wl.make_config("modelb_1024")
    g = run_horizons(pss, oracle, cfg, prec, [(1, TOL1[prec]), (1000, TOLN[prec])], "config 2 (1024^2)")
    assert bool(g.uses_fused_kernel) == (prec == "f32"), "the headline config must run the kernel bench.py times"


def test_config2_noise_bits_full_size(pss, oracle):
    cfg = wl.make_config("modelb_1024")
    g, o, dyn = both(pss, oracle, cfg, "f32")
    for step in (0, 999):
        bg, zg = g.debug_noise(dyn[0], step)
        bo, zo = o.debug_noise(dyn[0], step)
        assert np.array_equal(bg, bo)
        assert np.max(np.abs(zg - zo)) <= 3e-6


def test_config2_other_dealias_rules_full_size(pss, oracle):
    """forced 2/3 rule (literal BASELINE wording, A6) and no mask: the un-pruned fused instantiation"""
    for rule in (1, 2):
        cfg = wl.make_config("modelb_1024")
        g, ids = wl.build(pss, cfg, prec="f32", dealias=rule)
        o, _ = wl.build(oracle, cfg, prec="f32", dealias=rule)
        g.step(1)
        o.step(1)
        check(g, o, [ids["phi"]], TOL1["f32"], "config 2 dealias=%d, 1 step" % rule)
        g.step(19)
        o.step(19)
        check(g, o, [ids["phi"]], 10 * TOL1["f32"], "config 2 dealias=%d, 20 steps" % rule)


# config 3: 3D Model B 256^3 fp32
def test_config3_modelb_256_cubed(pss, oracle):
    cfg = wl.make_config("modelb_256c")
    n = FULL_HORIZON or 200
    run_horizons(pss, oracle, cfg, "f32", [(1, TOL1["f32"]), (10, 10 * TOL1["f32"]), (n, TOLN["f32"])], "config 3 (256^3)")


# config 4: nematic 1024^2 fp32, parity horizon 250 steps (A20)
def test_config4_nematic_1024(pss, oracle):
    cfg = wl.make_config("nematic_1024")
    run_horizons(pss, oracle, cfg, "f32", [(1, TOL1["f32"]), (250, 1e-3)], "config 4 (nematic 1024^2)")


# config 5: KPZ 4096^2 fp32
def test_config5_kpz_4096(pss, oracle):
    cfg = wl.make_config("kpz_4096")
    n = FULL_HORIZON or 100
    run_horizons(pss, oracle, cfg, "f32", [(1, TOL1["f32"]), (20, 10 * TOL1["f32"]), (n, TOLN["f32"])], "config 5 (KPZ 4096^2)")


# config 5b: the Model-B lattice sweep 256^2 .. 8192^2
@pytest.mark.parametrize("n", [256, 512, 2048, 4096, 8192])
def test_sweep_modelb(pss, oracle, n):
    cfg = wl.make_config("sweep_%d" % n)
    run_horizons(pss, oracle, cfg, "f32", [(1, TOL1["f32"]), (5, 10 * TOL1["f32"])], "sweep %d^2" % n)


def test_fullsize_step_splitting_is_bit_identical(pss):
    """pss_step(a); pss_step(b) == pss_step(a+b) bit for bit in the fused kernel (P14 at full size)"""
    cfg = wl.make_config("modelb_1024")
    a, ids = wl.build(pss, cfg, prec="f32")
    b, _ = wl.build(pss, cfg, prec="f32")
    a.step(3)
    a.step(4)
    b.step(7)
    f = ids["phi"]
    assert np.array_equal(a.get_field_fourier(f).view(np.uint32), b.get_field_fourier(f).view(np.uint32))
    m = a.get_field_fourier(f)[0, 0]
    assert m.imag == 0.0


# ---------------------------------------------------------------------------------------------
# properties that hold at any size, checked on the CUDA path alone at the headline size
# ---------------------------------------------------------------------------------------------
def test_config2_full_run_conserves_mass_and_phase_separates(pss):
    """config 2 in full: 10^4 steps of the headline workload in the launch configuration bench.py times.
    Conserved dynamics keep the q = 0 mode bit-identical (P5); the off-critical quench coarsens towards the
    phases +-sqrt(-a/b) = +-1 and stays finite."""
    cfg = wl.make_config("modelb_1024")
    g, ids = wl.build(pss, cfg, prec="f32")
    f = ids["phi"]
    m0 = g.get_field_fourier(f)[0, 0]
    v0 = float(np.var(g.get_field(f)))
    g.step(5000)
    g.step(5000)
    assert g.step_count == 10000 and g.uses_fused_kernel
    spec = g.get_field_fourier(f)
    assert spec[0, 0].real == m0.real and spec[0, 0].imag == 0.0
    x = g.get_field(f).astype(np.float64)
    assert np.all(np.isfinite(x))
    assert abs(x.mean() - 0.1) < 1e-5
    assert np.var(x) > 50 * v0 and np.abs(x).max() < 1.5      # domains have formed, amplitudes bounded by the phases
    assert np.mean(x > 0.5) > 0.3                             # majority phase near +1 (mean 0.1)


def test_fused_kernel_stationary_structure_factor(pss):
    """oracle-independent pin of the noise amplitude and Hermitian rule of the persistent kernel (A1, P6):
    linear conserved dynamics d phi = -(a q^2 + k q^4) phi + noise D q^2 at 1024^2; the stationary
    <|phi_q|^2> = (N/dV) 2 D q^2 / (lam (2 + dt lam)), lam = a q^2 + k q^4, averaged over many modes."""
    n, dt, a, k, D = 1024, 0.05, 1.0, 1.0, 0.02
    s = pss.System((n, n), (1.0, 1.0), dt, prec="f32", seed=31337)
    f = s.add_field("phi", True)
    s.add_linear(f, {"coef": a, "q2_pow": 1})
    s.add_linear(f, {"coef": k, "q2_pow": 2})
    s.add_term(f, {"coef": 0.0, "q2_pow": 1}, [f, f, f])      # a product group with zero weight: fused-kernel eligible
    s.set_noise(f, D, 2)
    s.finalize()
    assert s.uses_fused_kernel
    s.set_field(f, np.zeros((n, n), np.float32))
    ky = np.fft.fftfreq(n, 1.0 / n)[:, None]
    kx = np.arange(n // 2 + 1)[None, :]
    q2 = (2 * np.pi / n) ** 2 * (kx ** 2 + ky ** 2)
    lam = a * q2 + k * q2 ** 2
    with np.errstate(divide="ignore", invalid="ignore"):
        S_th = n * n * 2 * D * q2 / (lam * (2 + dt * lam))
    sel = (q2 > 0.5) & (kx > 0) & (kx < n // 2)               # relaxation time 1/lam < 2: decorrelated between samples
    s.step(400)
    acc, cnt = np.zeros_like(q2), 0
    for _ in range(12):
        s.step(100)
        spec = s.get_field_fourier(f)
        acc += np.abs(spec.astype(np.complex128)) ** 2
        cnt += 1
    ratio = (acc / cnt)[sel] / S_th[sel]
    assert abs(ratio.mean() - 1.0) < 0.01, ratio.mean()       # ~3e5 modes x 12 samples
    # boundary planes kx = 0 and kx = n/2 carry the same variance (Hermitian rule)
    for col in (0, n // 2):
        m = (q2[:, col] > 0.5)
        r = (acc / cnt)[m, col] / S_th[m, col]
        assert abs(r.mean() - 1.0) < 0.08, (col, r.mean())


def test_config3_full_length_conserves_mass(pss):
    """config 3 in full: 2000 steps of 3D Model B 256^3; the q = 0 mode stays bit-identical, the field finite"""
    cfg = wl.make_config("modelb_256c")
    g, ids = wl.build(pss, cfg, prec="f32")
    f = ids["phi"]
    m0 = g.get_field_fourier(f)[0, 0, 0]
    g.step(2000)
    spec = g.get_field_fourier(f)
    assert spec[0, 0, 0].real == m0.real and spec[0, 0, 0].imag == 0.0
    x = g.get_field(f)
    assert np.all(np.isfinite(x)) and np.abs(x).max() < 1.5 and float(np.var(x)) > 1e-3


def test_config5_full_length_kpz_growth(pss):
    """config 5 in full: 5000 steps of KPZ 4096^2 from h = 0.  The mean height obeys d<h>/dt = (lambda/2) <|grad h|^2>
    (the q = 0 mode of Eq. 18: L(0) = 0, noise adds a zero-mean term), so it grows monotonically and the interface
    roughens; everything stays finite."""
    cfg = wl.make_config("kpz_4096")
    g, ids = wl.build(pss, cfg, prec="f32")
    h = ids["h"]
    n = 4096 * 4096
    means, widths = [], []
    for _ in range(5):
        g.step(1000)
        spec = g.get_field_fourier(h)
        assert np.all(np.isfinite(spec.view(np.float32)))
        means.append(float(spec[0, 0].real) / n)
        widths.append(float(np.sqrt((np.sum(np.abs(spec[:, 1:-1].astype(np.complex128)) ** 2) * 2
                                     + np.sum(np.abs(spec[:, [0, -1]].astype(np.complex128)) ** 2)
                                     - abs(spec[0, 0]) ** 2) / n ** 2)))
    assert g.step_count == 5000
    assert all(b > a for a, b in zip(means, means[1:])), means      # lambda > 0: the surface moves up
    assert widths[-1] > widths[0] * 0.9 and widths[-1] < 10.0, widths


def test_persistent_kernel_scheduling_switches_do_not_change_the_result(pss):
    """PSS_NOISE_GATE (noise warps paused while their group computes) and PSS_P2D_PRIO (group 0 first in phase C) only
    move work in time: the fields are bit-identical with either switched off.  (That an ensemble replica, one k_persist2d
    launch per replica, is bit-identical to the single system with its seed is checked at 1024^2 in
    test_gpu_ensemble.py::test_replicas_equal_single_systems_and_oracle.)"""
    import os
    cfg = wl.make_config("modelb_1024")
    ref, ids = wl.build(pss, cfg, prec="f32")
    assert ref.fused_kernel_name == "k_persist2d"
    ref.step(6)
    want = ref.get_field_fourier(ids["phi"]).view(np.uint32)
    for var in ("PSS_NOISE_GATE", "PSS_P2D_PRIO"):
        os.environ[var] = "0"
        try:
            g, _ = wl.build(pss, cfg, prec="f32")
            g.step(2)
            g.step(4)
            got = g.get_field_fourier(ids["phi"]).view(np.uint32)
        finally:
            del os.environ[var]
        assert np.array_equal(got, want), var
