"""GPU parity for the Dirichlet frames of PAPER.md section V (callbacks): CUDA path vs. oracle."""
import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as wl
from parity_util import TOL1, compare_fields

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pss():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_02410_b200 as p
    p.binding.lib()
    return p


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_heat_baths_fig2(pss, oracle, prec):
    """the paper's Fig. 2 set-up: 256 sites, T(x,0) = 5, baths of width 10 at 10 and 0"""
    n = 256
    sysm = []
    for api in (pss, oracle):
        s = api.System((n,), (1.0,), 2.0, prec=prec, seed=1)
        f = s.add_field("T", True)
        s.add_linear(f, {"coef": 1.0, "q2_pow": 1})
        s.set_frame(f, 0, 10, 10.0, 10, 0.0)
        s.finalize()
        s.set_field(f, np.full(n, 5.0, dtype=s.rdtype))
        sysm.append((s, f))
    (g, f), (o, _) = sysm
    g.step(1)
    o.step(1)
    compare_fields(g, o, [f], TOL1[prec], "heat baths, 1 step")
    g.step(499)
    o.step(499)
    compare_fields(g, o, [f], 50 * TOL1[prec], "heat baths, 500 steps")
    T = g.get_field(f)
    assert np.allclose(T[:10], 10.0, atol=1e-4) and np.allclose(T[246:], 0.0, atol=1e-4)


@pytest.mark.parametrize("name,n,frames", [("modelb_128", (64, 32), [(0, 4, 1.0, 4, -1.0)]),
                                           ("modelb_128", (32, 64), [(1, 3, 0.5, 0, 0.0), (0, 2, -0.5, 2, -0.5)]),
                                           ("modelb_256c", (16, 16, 32), [(2, 4, 1.0, 4, -1.0)]),
                                           ("kpz_4096", (64, 64), [(0, 5, 0.0, 5, 0.0)])])
def test_frames_on_the_baseline_models(pss, oracle, name, n, frames):
    cfg = wl.make_config(name, n=n)
    both = []
    for api in (pss, oracle):
        dxs = (float(cfg["dx"]),) * len(n)
        s = api.System(n, dxs, cfg["dt"], prec="f32", seed=cfg["seed"])
        ids = wl.MODELS[cfg["model"]](s, **cfg["params"])
        f = ids[list(cfg["ic"].keys())[0]]
        for fr in frames:
            s.set_frame(f, *fr)
        s.finalize()
        for nm, arr in wl.initial_conditions(cfg, np.float32).items():
            s.set_field(ids[nm], arr)
        both.append((s, f))
    (g, f), (o, _) = both
    g.step(1)
    o.step(1)
    compare_fields(g, o, [f], TOL1["f32"], "%s %s frames, 1 step" % (name, n))
    g.step(19)
    o.step(19)
    compare_fields(g, o, [f], 10 * TOL1["f32"], "%s %s frames, 20 steps" % (name, n))


def test_frame_on_the_persistent_kernel(pss, oracle):
    """1024^2 Model B with a frame: every step is its own launch of the persistent kernel (prologue + one step)"""
    cfg = wl.make_config("modelb_1024")
    both = []
    for api in (pss, oracle):
        s = api.System(cfg["n"], (1.0, 1.0), cfg["dt"], prec="f32", seed=cfg["seed"])
        ids = wl.model_b(s, **cfg["params"])
        s.set_frame(ids["phi"], 0, 8, 1.0, 8, -1.0)
        s.finalize()
        s.set_field(ids["phi"], wl.initial_conditions(cfg, np.float32)["phi"])
        both.append((s, ids["phi"]))
    (g, f), (o, _) = both
    assert g.uses_fused_kernel
    g.step(3)
    o.step(3)
    compare_fields(g, o, [f], 3 * TOL1["f32"], "1024^2 frame, 3 steps")


def test_frames_in_an_ensemble_match_single_systems(pss):
    """every replica gets its frame; replica r stays bit-identical to the single system with seed + r"""
    cfg = wl.make_config("modelb_128", n=(64, 64))

    def make(seed, replicas):
        s = pss.System(cfg["n"], (1.0, 1.0), cfg["dt"], prec="f32", seed=seed, replicas=replicas)
        ids = wl.model_b(s, **cfg["params"])
        s.set_frame(ids["phi"], 1, 3, 0.5, 3, -0.5)
        s.finalize()
        return s, ids["phi"]

    ic = wl.initial_conditions(cfg, np.float32)["phi"]
    e, f = make(cfg["seed"], 3)
    for r in range(3):
        e.select_replica(r)
        e.set_field(f, ic + 0.01 * r)
    e.step(7)
    for r in range(3):
        s, _ = make(cfg["seed"] + r, 1)
        s.set_field(f, ic + 0.01 * r)
        s.step(7)
        e.select_replica(r)
        assert np.array_equal(e.get_field_fourier(f).view(np.uint32), s.get_field_fourier(f).view(np.uint32)), r
