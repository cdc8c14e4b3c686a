"""CPU-side tests of the C-ABI library (no GPU, no compute calls): it loads, exports every symbol include/pss.h
declares, validates the field system, and reports the algorithmic byte counts of SURVEY.md 8(d)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pss():
    import paper_2405_02410_b200 as p
    p.binding.lib()
    return p


def test_library_exports_every_declared_symbol(pss):
    hdr = open(os.path.join(ROOT, "include", "pss.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(pss_[a-z_0-9]+)\s*\(", hdr)))
    assert len(declared) >= 20
    lib = pss.binding.lib()
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(pss.binding.SYMBOLS) == declared


def test_product_does_not_reference_the_oracle():
    """the product path (package + C sources) never imports, links or loads anything under oracle/"""
    pkg = os.path.join(ROOT, "paper_2405_02410_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "libopss" not in src and "opss_" not in src, f


def test_comparison_build_exports_its_symbol(pss):
    from compare import build as compare_build
    lib = ctypes.CDLL(compare_build.build())
    assert hasattr(lib, "cmp_cufft_modelb")


def test_error_codes_without_a_device(pss):
    b = pss.binding
    with pytest.raises(b.PssError) as e:
        pss.System((100, 64), (1.0, 1.0), 0.01)          # not a power of two (A17)
    assert e.value.code == b.EUNSUPPORTED
    with pytest.raises(b.PssError) as e:
        pss.System((4, 64), (1.0, 1.0), 0.01)            # below the GPU minimum of 8
    assert e.value.code == b.EUNSUPPORTED
    with pytest.raises(b.PssError) as e:
        pss.System((64, 64), (1.0, -1.0), 0.01)
    assert e.value.code == b.EINVAL
    s = pss.System((64, 64), (1.0, 1.0), 0.01)
    f = s.add_field("phi", True)
    with pytest.raises(b.PssError) as e:
        s.add_field("phi", True)                         # duplicate name
    assert e.value.code == b.EINVAL
    with pytest.raises(b.PssError) as e:
        s.add_linear(f, {"q2_pow": -1})
    assert e.value.code == b.EINVAL
    with pytest.raises(b.PssError) as e:
        s.add_term(f, {"coef": 1.0}, [f] * 5)            # product of more than 4 factors
    assert e.value.code == b.EUNSUPPORTED
    aux = s.add_field("g", False)
    with pytest.raises(b.PssError) as e:
        s.add_linear(aux, {"coef": 1.0})                 # implicit term on an aux field
    assert e.value.code == b.EINVAL
    with pytest.raises(b.PssError) as e:
        s.finalize(bind=False)                           # aux field without a definition
    assert e.value.code == b.EINVAL
    s.add_aux_def(aux, {"coef": 1.0, "iq_pow": (1, 0, 0)}, f)
    assert s.finalize(bind=False) > 0
    with pytest.raises(b.PssError) as e:
        s.add_field("late", True)                        # add_* after finalize
    assert e.value.code == b.ESTATE
    with pytest.raises(b.PssError) as e:
        s.step(1)                                        # step before bind
    assert e.value.code == b.ESTATE
    assert s.step_count == 0 and s.launch_count == 0


@pytest.mark.parametrize("name,b_alg,b_model", [
    ("modelb_1024", 20.0, 24.0), ("kpz_4096", 80.0 / 3.0, 32.0), ("nematic_1024", 232.0 / 3.0, 104.0),
    ("modelb_256c", 30.0, 40.0)])
def test_algorithmic_bytes_per_site(pss, name, b_alg, b_model):
    """pss_model_bytes_per_step against the per-site figures of SURVEY.md 8(d) (fp32)"""
    from paper_2405_02410_b200 import workloads as wl
    cfg = wl.make_config(name)
    n = cfg["n"]
    dx = (float(cfg["dx"]),) * len(n)
    s = pss.System(n, dx, cfg["dt"], prec="f32", seed=1)
    wl.MODELS[cfg["model"]](s, **cfg["params"])
    s.finalize(bind=False)
    sites = 1
    for v in n:
        sites *= v
    assert s.model_bytes_per_step(True) / sites == pytest.approx(b_alg, rel=1e-12)
    assert s.model_bytes_per_step(False) / sites == pytest.approx(b_model, rel=1e-12)


def test_workspace_size_scales_with_the_field_system(pss):
    from paper_2405_02410_b200 import workloads as wl
    sizes = {}
    for name in ("modelb_1024", "nematic_1024"):
        cfg = wl.make_config(name)
        s = pss.System(cfg["n"], (1.0, 1.0), cfg["dt"])
        wl.MODELS[cfg["model"]](s, **cfg["params"])
        sizes[name] = s.finalize(bind=False)
    arr = 1024 * 513 * 8
    assert sizes["modelb_1024"] >= 4 * arr            # state + one factor + one group + scratch
    assert sizes["nematic_1024"] >= (2 + 9 + 2 + 1) * arr
