"""GPU parity for SURVEY.md 8(f) item 2: intermediate fields with their own lhs (a rational
multiplier num(q)/den(q)) and intermediate fields that are products (one extra round of the step kernels per dependency
level), built through the equation-string front end on both sides, CUDA path vs. oracle."""
import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as wl
from paper_2405_02410_b200.equations import Model
from parity_util import TOL1, compare_fields

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pss():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_02410_b200 as p
    p.binding.lib()
    return p


def build(api, n, prec, describe, dt=0.01, seed=2405024107, dx=None):
    dx = dx or (1.0,) * len(n)
    s = api.System(n, dx, dt, prec=prec, seed=seed)
    m = Model(s)
    describe(m)
    s.finalize()
    dtype = np.float32 if prec == "f32" else np.float64
    dyn = [(name, fid) for name, (fid, d) in m.fields.items() if d]
    for i, (name, fid) in enumerate(dyn):
        s.set_field(fid, wl.uniform_field(seed, i, tuple(n)[::-1], -0.1, 0.1, dtype))
    return s, [fid for _, fid in dyn]


def run(pss, oracle, n, prec, describe, steps=20, dt=0.01, what=""):
    g, dyn = build(pss, n, prec, describe, dt)
    o, dyn_o = build(oracle, n, prec, describe, dt)
    assert dyn == dyn_o
    g.step(1)
    o.step(1)
    compare_fields(g, o, dyn, TOL1[prec], "%s %s 1 step" % (what, n))
    g.step(steps - 1)
    o.step(steps - 1)
    compare_fields(g, o, dyn, 10 * TOL1[prec], "%s %s %d steps" % (what, n, steps))
    return g


def screened(m):
    """psi + psi*q^2 = -q^2*phi used both in a product and as an explicit linear term"""
    m.add_parameter("D", 0.01)
    m.create_field("phi", True)
    m.create_field("psi", False)
    m.add_equation("psi + psi*q^2 = -q^2*phi")
    m.add_equation("dt phi + q^4*phi = -q^2*psi*phi + 0.5*psi - q^2*phi^3")
    m.add_noise("phi", "D*q^2")


def model_b_through_mu(m):
    """Model B with the chemical potential as a product-defined intermediate field: mu = phi^3 - phi + q^2 phi,
    dt phi = -q^2 mu (fully explicit), conserved noise"""
    m.add_parameter("D", 0.01)
    m.create_field("phi", True)
    m.create_field("mu", False)
    m.add_equation("mu = phi^3 - phi + q^2*phi")
    m.add_equation("dt phi = -q^2*mu")
    m.add_noise("phi", "D*q^2")


def three_levels(m):
    """a = phi*phi, b = a*phi + a (level 2), dt phi + q^2 phi = -q^2*b*a (uses levels 1 and 2), two dynamic fields"""
    m.create_field("phi", True)
    m.create_field("u", True)
    m.create_field("a", False)
    m.create_field("b", False)
    m.add_equation("a = phi*u")
    m.add_equation("b = a*phi + 0.5*a")
    m.add_equation("dt phi + q^2*phi = -q^2*b*a + 0.1*b")
    m.add_equation("dt u + q^2*u = a - u^3")
    m.add_noise("u", "0.001")


def model_h_stream(m):
    """Binary fluid in stream-function form: mu = phi^3 - phi + k q^2 phi (level 1); Stokes flow driven by the
    capillary force, eta q^4 w = d_x mu d_y phi - d_y mu d_x phi (level 2, an intermediate field with an lhs);
    v = (d_y w, -d_x w); dt phi = -q^2 mu - v.grad phi"""
    m.add_parameter("k", 1.0)
    m.add_parameter("eta", 2.0)
    m.add_parameter("D", 0.005)
    m.create_field("phi", True)
    for name in ("mu", "dxphi", "dyphi", "dxmu", "dymu", "w", "vx", "vy"):
        m.create_field(name, False)
    m.add_equation("mu = phi^3 - phi + k*q^2*phi")
    m.add_equation("dxphi = iqx*phi")
    m.add_equation("dyphi = iqy*phi")
    m.add_equation("dxmu = iqx*mu")
    m.add_equation("dymu = iqy*mu")
    m.add_equation("eta*q^4*w = dxmu*dyphi - dymu*dxphi")
    m.add_equation("vx = iqy*w")
    m.add_equation("vy = -iqx*w")
    m.add_equation("dt phi + k*q^4*phi = -q^2*phi^3 + q^2*phi - vx*dxphi - vy*dyphi")
    m.add_noise("phi", "D*q^2")


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("n", [(64, 32), (16, 32, 16), (128,)])
def test_intermediate_field_with_lhs(pss, oracle, n, prec):
    run(pss, oracle, n, prec, screened, what="screened")


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("n", [(64, 64), (32, 128), (16, 16, 32)])
@pytest.mark.parametrize("describe", [model_b_through_mu, three_levels])
def test_product_defined_intermediate_fields(pss, oracle, n, prec, describe):
    g = run(pss, oracle, n, prec, describe, dt=0.002, what=describe.__name__)
    assert g.launch_count > 0


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_model_h_stream_function_form(pss, oracle, prec):
    run(pss, oracle, (64, 64), prec, model_h_stream, dt=0.005, what="model H")


def test_model_h_at_512_squared(pss, oracle):
    run(pss, oracle, (512, 512), "f32", model_h_stream, steps=10, dt=0.005, what="model H")


def test_unsupported_combinations(pss):
    b = pss.binding
    s = pss.System((64,), (1.0,), 0.01)
    m = Model(s)
    model_b_through_mu(m)
    with pytest.raises(b.PssError) as e:
        s.finalize(bind=False)
    assert e.value.code == b.EUNSUPPORTED          # 1D: no rounds
    s = pss.System((32, 32), (1.0, 1.0), 0.01)
    m = Model(s)
    m.create_field("phi", True)
    m.create_field("psi", False)
    m.add_equation("psi + iqx*psi = phi")           # complex denominator
    m.add_equation("dt phi = -psi*phi")
    with pytest.raises(b.PssError) as e:
        s.finalize(bind=False)
    assert e.value.code == b.EUNSUPPORTED


def test_model_h_workload_at_1024_squared(pss, oracle):
    """the `modelh_1024` workload bench.py can time (three rounds of the step kernels per time step), full size"""
    cfg = wl.make_config("modelh_1024")
    g, ids = wl.build(pss, cfg, prec="f32")
    o, _ = wl.build(oracle, cfg, prec="f32")
    g.step(1)
    o.step(1)
    compare_fields(g, o, [ids["phi"]], TOL1["f32"], "modelh_1024 1 step")
    g.step(9)
    o.step(9)
    compare_fields(g, o, [ids["phi"]], 10 * TOL1["f32"], "modelh_1024 10 steps")
    assert not g.uses_fused_kernel
