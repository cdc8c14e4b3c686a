"""GPU parity: the CUDA path (through the C ABI of include/pss.h) against the CPU oracle, element by
element on the same seeded inputs and the same noise stream.

Tolerances are BASELINE.json's north_star: relative L2 <= 1e-5 after 1 step and <= 1e-3 after 1000
steps in fp32; <= 1e-12 / 1e-9 in fp64.  Noise bits are compared bit-exactly.
"""
import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as wl

pytestmark = pytest.mark.gpu

import parity_util as pu
from parity_util import TOL1, TOLN, rel_l2, compare_fields


@pytest.fixture(scope="module")
def pss():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_02410_b200 as p
    p.binding.lib()
    return p


def both(pss, oracle, cfg, prec, dealias=None):
    return pu.both(wl, pss, oracle, cfg, prec, dealias)


# ---------------------------------------------------------------------------------------------
# transforms alone: set_field / get_field round trip and the half-spectrum against the oracle R2C
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [(64,), (8,), (4096,), (128, 128), (32, 8), (8, 64), (1024, 16), (16, 16, 16),
                               (32, 8, 16), (8, 32, 64)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_set_get_roundtrip_and_spectrum(pss, oracle, n, prec):
    cfg = wl.make_config("modelb_128", n=n)
    g, ids = wl.build(pss, cfg, prec=prec)
    rng = np.random.default_rng(7)
    x = rng.standard_normal(n[::-1]).astype(g.rdtype)
    g.set_field(ids["phi"], x)
    back = g.get_field(ids["phi"])
    tol = 2e-6 if prec == "f32" else 1e-14
    assert rel_l2(back, x) <= tol
    spec = g.get_field_fourier(ids["phi"])
    ref = oracle.r2c(x.astype(np.float64))
    assert rel_l2(np.stack([spec.real, spec.imag]), np.stack([ref.real, ref.imag])) <= tol


# ---------------------------------------------------------------------------------------------
# noise stream: Philox words bit-exact, z within libm-vs-CUDA ulps (SURVEY 8(c) "noise bits")
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [(64,), (32, 16), (16, 8, 8), (128, 128)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_noise_bits_bit_exact(pss, oracle, n, prec):
    cfg = wl.make_config("modelb_128", n=n)
    g, o, dyn = both(pss, oracle, cfg, prec)
    for step in (0, 1, 12345678901):
        bg, zg = g.debug_noise(dyn[0], step)
        bo, zo = o.debug_noise(dyn[0], step)
        assert np.array_equal(bg, bo)
        tol = 3e-6 if prec == "f32" else 1e-13
        assert np.max(np.abs(zg - zo)) <= tol


def test_philox_matches_curand_known_answer(pss, oracle):
    """P8: the counter layout (m, step, field) reaches Philox as the oracle states it."""
    cfg = wl.make_config("modelb_128", n=(16, 8))
    g, o, dyn = both(pss, oracle, cfg, "f32")
    bg, _ = g.debug_noise(dyn[0], 5)
    seed = cfg["seed"]
    for (ky, kx) in [(0, 0), (3, 7), (7, 8)]:
        m = ky * 9 + kx
        w = oracle.philox((m, 0, 5, dyn[0]), (seed & 0xffffffff, seed >> 32))
        assert tuple(int(v) for v in bg[ky, kx]) == w


# ---------------------------------------------------------------------------------------------
# one step and a short run, every model, small lattices spanning several tiles + ragged tails
# ---------------------------------------------------------------------------------------------
CASES = [
    ("modelb_128", (128, 128)), ("modelb_128", (64, 32)), ("modelb_128", (16, 256)), ("modelb_128", (256,)),
    ("modelb_128", (8,)), ("modelb_256c", (32, 16, 16)), ("modelb_256c", (16, 32, 64)),
    ("kpz_4096", (128, 64)), ("kpz_4096", (512,)), ("kpz_4096", (16, 16, 32)),
    ("nematic_1024", (64, 64)), ("nematic_1024", (32, 128)),
]


@pytest.mark.parametrize("name,n", CASES)
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_one_step_and_short_run(pss, oracle, name, n, prec):
    cfg = wl.make_config(name, n=n)
    g, o, dyn = both(pss, oracle, cfg, prec)
    g.step(1)
    o.step(1)
    compare_fields(g, o, dyn, TOL1[prec], "%s %s 1 step" % (name, n))
    g.step(49)
    o.step(49)
    assert g.step_count == 50
    compare_fields(g, o, dyn, 10 * TOL1[prec], "%s %s 50 steps" % (name, n))


@pytest.mark.parametrize("dealias", [1, 2])
@pytest.mark.parametrize("name,n", [("modelb_128", (64, 64)), ("kpz_4096", (32, 64)), ("modelb_256c", (16, 16, 16))])
def test_other_dealias_rules(pss, oracle, name, n, dealias):
    cfg = wl.make_config(name, n=n)
    g, o, dyn = both(pss, oracle, cfg, "f32", dealias=dealias)
    g.step(3)
    o.step(3)
    compare_fields(g, o, dyn, 3e-5, "%s dealias=%d" % (name, dealias))


def test_anisotropic_spacing(pss, oracle):
    cfg = wl.make_config("kpz_4096", n=(32, 64), dx=(0.5, 1.25))
    g, o, dyn = both(pss, oracle, cfg, "f64")
    g.step(5)
    o.step(5)
    compare_fields(g, o, dyn, 1e-11, "anisotropic dx")


# ---------------------------------------------------------------------------------------------
# config 1 in full: 128^2, 1000 steps, both precisions
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_config1_modelb_128_1000_steps(pss, oracle, prec):
    cfg = wl.make_config("modelb_128")
    g, o, dyn = both(pss, oracle, cfg, prec)
    g.step(1)
    o.step(1)
    compare_fields(g, o, dyn, TOL1[prec], "config 1, 1 step")
    g.step(999)
    o.step(999)
    e = compare_fields(g, o, dyn, TOLN[prec], "config 1, 1000 steps")
    print("config1 %s 1000 steps rel L2 %.3e" % (prec, e))


# ---------------------------------------------------------------------------------------------
# the 1000-step tolerance on the 3D path (k_mid) and the KPZ path (odd-derivative factors), reduced lattices:
# PAPER.md:128-135 iterated 1000 times, north_star's <= 1e-3 (fp32) / <= 1e-9 (fp64)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,n", [("modelb_256c", (64, 64, 64)), ("kpz_4096", (512, 512))])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_1000_steps_3d_and_kpz_reduced(pss, oracle, name, n, prec):
    cfg = wl.make_config(name, n=n)
    pu.run_horizons(wl, pss, oracle, cfg, prec, [(1, TOL1[prec]), (1000, TOLN[prec])], "%s %s" % (name, n))


def test_nematic_horizon_250_steps(pss, oracle):
    """A20: config 4 is chaotic; the parity horizon is 250 steps (here on 128^2)."""
    cfg = wl.make_config("nematic_1024", n=(128, 128))
    g, o, dyn = both(pss, oracle, cfg, "f32")
    g.step(250)
    o.step(250)
    compare_fields(g, o, dyn, 1e-3, "nematic 128^2 250 steps")


# ---------------------------------------------------------------------------------------------
# stepping semantics and conservation (properties that hold at any size)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,n", [("modelb_128", (64, 64)), ("kpz_4096", (32, 32)), ("modelb_256c", (16, 16, 16)),
                                    ("modelb_128", (128,))])
def test_step_splitting_is_bit_identical(pss, name, n):
    cfg = wl.make_config(name, n=n)
    a, ids = wl.build(pss, cfg, prec="f32")
    b, _ = wl.build(pss, cfg, prec="f32")
    a.step(3)
    a.step(4)
    b.step(7)
    f = ids[list(cfg["ic"].keys())[0]]
    assert np.array_equal(a.get_field_fourier(f).view(np.uint32), b.get_field_fourier(f).view(np.uint32))


def test_conserved_mean_is_bit_identical(pss):
    cfg = wl.make_config("modelb_1024", n=(128, 64))
    g, ids = wl.build(pss, cfg, prec="f32")
    m0 = g.get_field_fourier(ids["phi"])[0, 0]
    g.step(20)
    m1 = g.get_field_fourier(ids["phi"])[0, 0]
    assert m0.real == m1.real and m1.imag == 0.0


def test_error_codes_on_gpu(pss):
    b = pss.binding
    with pytest.raises(b.PssError) as e:
        pss.System((100, 64), (1.0, 1.0), 0.01)
    assert e.value.code == b.EUNSUPPORTED
    s = pss.System((64, 64), (1.0, 1.0), 0.01)
    f = s.add_field("phi", True)
    with pytest.raises(b.PssError) as e:
        s.add_linear(f, {"q2_pow": -1})
    assert e.value.code == b.EINVAL
    s.finalize(bind=False)
    with pytest.raises(b.PssError) as e:
        s.step(1)
    assert e.value.code == b.ESTATE


def test_p8_philox_matches_curand_device_api(pss, oracle):
    """P8: the oracle's Philox4x32-10 block and the words the CUDA path draws equal cuRAND's device
    generator (curand_init + curand4) for the same key and counter — an implementation neither side wrote."""
    import ctypes
    from compare import build as compare_build
    lib = ctypes.CDLL(compare_build.build())
    lib.cmp_curand_philox_block.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.POINTER(ctypes.c_uint32)]

    def curand_block(ctr, key):
        out = (ctypes.c_uint32 * 4)()
        rc = lib.cmp_curand_philox_block(key[0] | (key[1] << 32), ctr[2] | (ctr[3] << 32), 4 * (ctr[0] | (ctr[1] << 32)), out)
        assert rc == 0
        return tuple(int(v) for v in out)

    rng = np.random.default_rng(11)
    cases = [((0, 0, 0, 0), (0, 0)), ((1, 0, 0, 0), (0, 0)), ((0, 0, 1, 0), (0, 0))]
    for _ in range(12):   # offset = 4 * (c0 | c1 << 32) must fit 64 bits: c1 < 2^30
        cases.append(((int(rng.integers(0, 2 ** 32)), int(rng.integers(0, 2 ** 30)), int(rng.integers(0, 2 ** 32)),
                       int(rng.integers(0, 2 ** 32))), tuple(int(v) for v in rng.integers(0, 2 ** 32, 2))))
    for ctr, key in cases:
        assert oracle.philox(ctr, key) == curand_block(ctr, key), (ctr, key)
    # and the words the product draws for (seed, step, field, mode) are that block
    cfg = wl.make_config("modelb_128", n=(16, 8))
    g, ids = wl.build(pss, cfg, prec="f32")
    bits, _ = g.debug_noise(ids["phi"], 7)
    seed = cfg["seed"]
    for (ky, kx) in [(0, 0), (5, 3), (7, 8)]:
        m = ky * 9 + kx
        assert tuple(int(v) for v in bits[ky, kx]) == curand_block((m, 0, 7, ids["phi"]), (seed & 0xffffffff, seed >> 32))
