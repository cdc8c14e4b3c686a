"""GPU tests of the boundary's semantics beyond the BASELINE workloads: device-pointer set/get, a caller-supplied
stream, field systems without products, multi-field explicit linear terms, 1/|q| operators, the paper's own Model-B
listing parameters.  All through the C ABI, all against the CPU oracle."""
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


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.linalg.norm(b.ravel())
    return np.linalg.norm((a - b).ravel()) / (den if den > 0 else 1.0)


@pytest.mark.parametrize("n", [(256, 128), (1024, 1024), (32, 16, 64)])
def test_device_pointer_set_get_matches_host_path(pss, n):
    """pss_set_field / pss_get_field with on_device = 1 (torch CUDA tensors) equal the host-pointer path bit for bit"""
    import torch
    cfg = wl.make_config("modelb_1024" if len(n) == 2 else "modelb_256c", n=n)
    a, ids = wl.build(pss, cfg, prec="f32")
    b, _ = wl.build(pss, cfg, prec="f32", set_ic=False)
    ic = wl.initial_conditions(cfg, np.float32)["phi"]
    b.set_field(ids["phi"], torch.from_numpy(ic).cuda())
    a.step(5)
    b.step(5)
    out = torch.empty(ic.shape, dtype=torch.float32, device="cuda")
    b.get_field(ids["phi"], out=out)
    assert np.array_equal(a.get_field(ids["phi"]).view(np.uint32), out.cpu().numpy().view(np.uint32))


def test_caller_supplied_stream(pss, oracle):
    import torch
    st = torch.cuda.Stream()
    cfg = wl.make_config("modelb_1024")
    g, ids = wl.build(pss, cfg, prec="f32", stream=st)
    o, _ = wl.build(oracle, cfg, prec="f32")
    g.step(3)
    o.step(3)
    st.synchronize()
    assert rel_l2(g.get_field(ids["phi"]), o.get_field(ids["phi"])) <= 1e-5


def rotation(s):
    """du/dt = v, dv/dt = -u - 0.5 q^2 v: explicit linear cross terms (A8, A11), an implicit term, no products"""
    u = s.add_field("u", True)
    v = s.add_field("v", True)
    s.add_term(u, {"coef": 1.0}, [v])
    s.add_term(v, {"coef": -1.0}, [u])
    s.add_linear(v, {"coef": 0.5, "q2_pow": 1})
    s.set_noise(u, 0.01, 0)
    return u, v


@pytest.mark.parametrize("n", [(64,), (64, 32), (16, 16, 16)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_two_fields_linear_cross_terms(pss, oracle, n, prec):
    rng = np.random.default_rng(3)
    systems = []
    for api in (pss, oracle):
        s = api.System(n, (1.0,) * len(n), 0.02, prec=prec, seed=77)
        u, v = rotation(s)
        s.finalize()
        systems.append((s, u, v))
    dt = np.float32 if prec == "f32" else np.float64
    u0 = rng.standard_normal(n[::-1]).astype(dt)
    v0 = rng.standard_normal(n[::-1]).astype(dt)
    for s, u, v in systems:
        s.set_field(u, u0)
        s.set_field(v, v0)
        s.step(25)
    (g, u, v), (o, _, _) = systems
    tol = 1e-5 if prec == "f32" else 1e-12
    assert rel_l2(g.get_field(u), o.get_field(u)) <= tol
    assert rel_l2(g.get_field(v), o.get_field(v)) <= tol


def screened(s):
    """d phi/dt = -|q| phi - (psi)^2 with psi = (1/|q|) d_x phi: the 1/q keyword (A10) and an odd
    derivative (A9) inside a product"""
    f = s.add_field("phi", True)
    psi = s.add_field("psi", False)
    s.add_aux_def(psi, {"coef": 1.0, "invq_pow": 1, "iq_pow": (1, 0, 0)}, f)
    s.add_linear(f, {"coef": 1.0, "q2_pow": 1, "invq_pow": 1})
    s.add_term(f, {"coef": -1.0}, [psi, psi])
    s.set_noise(f, 0.02, -1)
    return f


@pytest.mark.parametrize("n", [(128,), (64, 64), (16, 32, 16)])
def test_inverse_q_operators_and_negative_noise_power(pss, oracle, n):
    rng = np.random.default_rng(5)
    x0 = 0.3 * rng.standard_normal(n[::-1])
    res = []
    for api in (pss, oracle):
        s = api.System(n, (0.7,) * len(n), 0.01, prec="f64", seed=9)
        f = screened(s)
        s.finalize()
        s.set_field(f, x0)
        s.step(10)
        res.append(s.get_field(f))
    assert rel_l2(res[0], res[1]) <= 1e-11


def test_paper_listing_parameters(pss, oracle):
    """the paper's own Model-B listing and Fig. 1 run: -a = b = 1, k = 4, dt = 0.1, 256^2, noiseless"""
    cfg = wl.make_config("modelb_1024", n=(256, 256), dt=0.1, k=4.0, D=0.0)
    g, ids = wl.build(pss, cfg, prec="f32")
    o, _ = wl.build(oracle, cfg, prec="f32")
    g.step(100)
    o.step(100)
    a, b = g.get_field(ids["phi"]), o.get_field(ids["phi"])
    assert rel_l2(a, b) <= 1e-4
    m0 = wl.initial_conditions(cfg, np.float64)["phi"].mean()
    assert abs(a.astype(np.float64).mean() - m0) <= 1e-6          # conserved dynamics keep the mean


def test_nematic_other_dealias_rules(pss, oracle):
    for rule in (1, 2):
        cfg = wl.make_config("nematic_1024", n=(64, 128))
        g, ids = wl.build(pss, cfg, prec="f64", dealias=rule)
        o, _ = wl.build(oracle, cfg, prec="f64", dealias=rule)
        g.step(5)
        o.step(5)
        for name in ("Qxx", "Qxy"):
            assert rel_l2(g.get_field(ids[name]), o.get_field(ids[name])) <= 1e-11


@pytest.mark.parametrize("name,n", [("modelb_1024", (1024, 1024)), ("kpz_4096", (64, 128)), ("modelb_256c", (16, 32, 16)),
                                    ("nematic_1024", (64, 64)), ("modelb_128", (256,))])
def test_checkpoint_resume_is_bit_identical(pss, name, n):
    """state = half-spectra + step counter (counter-based noise): a restored run continues bit for bit"""
    cfg = wl.make_config(name, n=n)
    a, ids = wl.build(pss, cfg, prec="f32")
    b, _ = wl.build(pss, cfg, prec="f32")
    dyn = [ids[nm] for nm in cfg["ic"].keys()]
    a.step(9)
    ckpt = {f: a.get_field_fourier(f) for f in dyn}
    step = a.step_count
    a.step(8)
    c, _ = wl.build(pss, cfg, prec="f32", set_ic=False)
    for f in dyn:
        c.set_field_fourier(f, ckpt[f])
    c.set_step_count(step)
    c.step(8)
    b.step(17)
    assert c.step_count == 17
    for f in dyn:
        ref = b.get_field_fourier(f).view(np.uint32)
        assert np.array_equal(a.get_field_fourier(f).view(np.uint32), ref)
        assert np.array_equal(c.get_field_fourier(f).view(np.uint32), ref)


def test_system_on_a_device_that_is_not_current(pss):
    """the library records the workspace's device in pss_bind and makes it current inside every entry
    point.  With two or more GPUs: build on cuda:1 while cuda:0 is current; with one GPU: the guard is a no-op and the
    call sequence is checked with an explicit (non-default) stream."""
    import torch
    from paper_2405_02410_b200 import workloads as wl
    cfg = wl.make_config("modelb_128", n=(64, 64))
    ref, ids = wl.build(pss, cfg, prec="f32")
    ref.step(5)
    want = ref.get_field_fourier(ids["phi"])
    if torch.cuda.device_count() >= 2:
        torch.cuda.set_device(0)
        g, _ = wl.build(pss, cfg, prec="f32", device="cuda:1")
        g.step(5)
        assert torch.cuda.current_device() == 0
    else:
        st = torch.cuda.Stream()
        g, _ = wl.build(pss, cfg, prec="f32", stream=st)
        g.step(5)
    got = g.get_field_fourier(ids["phi"])
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))


def test_set_step_count_needs_a_finalized_system(pss):
    b = pss.binding
    s = pss.System((64, 64), (1.0, 1.0), 0.01)
    s.add_field("phi", True)
    with pytest.raises(b.PssError) as e:
        s.set_step_count(3)
    assert e.value.code == b.ESTATE
