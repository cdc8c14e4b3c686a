"""Equation-string front end: the paper's listings, parsed, give the same
boundary calls as the hand-written sequences of workloads.py, and the same trajectories on the oracle.  CPU only."""
import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as wl
from paper_2405_02410_b200.equations import EquationError, Model


class Recorder:
    """stands in for a System: records the builder calls with field NAMES instead of ids"""

    def __init__(self, ndim=2):
        self.ndim = ndim
        self.names = []
        self.calls = []

    @staticmethod
    def _op(d):
        iq = tuple(d.get("iq_pow", (0, 0, 0))) + (0, 0, 0)
        return (round(float(d.get("coef", 1.0)), 12), int(d.get("q2_pow", 0)), int(d.get("invq_pow", 0)), iq[:3])

    def add_field(self, name, dynamic=True):
        self.names.append(name)
        self.calls.append(("field", name, bool(dynamic)))
        return len(self.names) - 1

    def add_linear(self, f, op):
        self.calls.append(("linear", self.names[f], self._op(op)))

    def add_aux_def(self, a, op, src):
        self.calls.append(("aux_def", self.names[a], self._op(op), self.names[src]))

    def add_aux_lhs(self, a, op):
        self.calls.append(("aux_lhs", self.names[a], self._op(op)))

    def add_aux_term(self, a, op, factors):
        self.calls.append(("aux_term", self.names[a], self._op(op), tuple(self.names[f] for f in factors)))

    def add_term(self, f, op, factors):
        self.calls.append(("term", self.names[f], self._op(op), tuple(self.names[g] for g in factors)))

    def set_noise(self, f, D, qpow):
        self.calls.append(("noise", self.names[f], float(D), int(qpow)))


def by_kind(calls):
    return sorted(calls, key=lambda c: (c[0], repr(c[1:])))


def test_paper_listing_diffusion():
    """createField / addParameter / addEquation / addNoise"""
    r = Recorder()
    m = Model(r)
    m.create_field("phi", True)
    m.add_parameter("D", 1.0)
    m.add_equation("dt phi + D*q^2*phi = 0")
    m.add_noise("phi", "D")
    h = Recorder()
    wl.diffusion(h, D=1.0, noise=1.0)
    assert r.calls == h.calls


def test_paper_listing_model_b():
    """PAPER.md:216-227 (Eq. 20) with the conserved noise of PAPER.md:196-199"""
    r = Recorder()
    m = Model(r)
    m.add_parameter("a", -1.0)
    m.add_parameter("b", 1.0)
    m.add_parameter("k", 4.0)
    m.create_field("phi", 1)
    m.add_equation("dt phi + (a*q^2 + k*q^4)*phi = -b*q^2*phi^3")
    m.add_parameter("D", 0.01)
    m.add_noise("phi", "D*q^2")
    h = Recorder()
    wl.model_b(h, a=-1.0, b=1.0, k=4.0, D=0.01)
    assert r.calls == h.calls


def test_paper_listing_intermediate_fields():
    """operators act on the whole product; an intermediate field carries the single-field operator;
    an intermediate field with its own lhs, psi + psi*q^2 = -q^2*phi"""
    r = Recorder()
    m = Model(r)
    m.create_field("phi", True)
    m.create_field("psi", True)
    m.create_field("lapphi", False)
    m.add_equation("dt phi = psi*lapphi")
    m.add_equation("lapphi = -q^2*phi")
    m.add_equation("dt psi = -q^2*phi*psi")
    assert r.calls[3:] == [("term", "phi", (1.0, 0, 0, (0, 0, 0)), ("psi", "lapphi")),
                           ("aux_def", "lapphi", (-1.0, 1, 0, (0, 0, 0)), "phi"),
                           ("term", "psi", (-1.0, 1, 0, (0, 0, 0)), ("phi", "psi"))]
    r = Recorder()
    m = Model(r)
    m.create_field("phi", True)
    m.create_field("psi", False)
    m.add_equation("psi + psi * q^2 = -q^2*phi")
    assert r.calls[2:] == [("aux_lhs", "psi", (1.0, 0, 0, (0, 0, 0))), ("aux_lhs", "psi", (1.0, 1, 0, (0, 0, 0))),
                           ("aux_def", "psi", (-1.0, 1, 0, (0, 0, 0)), "phi")]
    r = Recorder()
    m = Model(r)
    m.create_field("phi", True)
    m.create_field("mu", False)
    m.add_equation("mu = phi^3 - phi + q^2*phi")          # a product-defined intermediate field
    assert ("aux_term", "mu", (1.0, 0, 0, (0, 0, 0)), ("phi", "phi", "phi")) in r.calls
    assert ("aux_def", "mu", (-1.0, 0, 0, (0, 0, 0)), "phi") in r.calls and ("aux_def", "mu", (1.0, 1, 0, (0, 0, 0)), "phi") in r.calls


def test_keywords_and_kpz_against_the_hand_written_sequence():
    """iqx / iqy, parameter arithmetic, division by a constant (reading A15 of DESIGN.md for the KPZ coefficients)"""
    r = Recorder()
    m = Model(r)
    m.add_parameter("nu", 1.0)
    m.add_parameter("lam", 2.0)
    m.create_field("h", True)
    m.create_field("gx", False)
    m.create_field("gy", False)
    m.add_equation("gx = iqx*h")
    m.add_equation("gy = iqy*h")
    m.add_equation("dt h + nu*q^2*h = lam/2*gx^2 + lam*gy*gy/2")
    m.add_noise("h", "1.0")
    h = Recorder()
    wl.kpz(h, nu=1.0, lam=2.0, D=1.0)
    assert by_kind(r.calls) == by_kind(h.calls)
    # 1/q, iqz^2, powers of parentheses, unary minus
    r = Recorder(ndim=3)
    m = Model(r)
    m.create_field("u", True)
    m.add_parameter("c", 0.5)
    m.add_equation("dt u + (c*q^2)^2*u - iqz^2*u = -(1/q)*u*u + 1/q^3*iqx*iqy*u")
    assert r.calls[1:] == [("linear", "u", (0.25, 2, 0, (0, 0, 0))), ("linear", "u", (-1.0, 0, 0, (0, 0, 2))),
                           ("term", "u", (-1.0, 0, 1, (0, 0, 0)), ("u", "u")),
                           ("term", "u", (1.0, 0, 3, (1, 1, 0)), ("u",))]
    r = Recorder()
    m = Model(r)
    m.create_field("phi", True)
    m.add_noise("phi", "0.3*q^2*1/q")
    assert r.calls[-1] == ("noise", "phi", 0.3, 1)


@pytest.mark.parametrize("bad", ["dt phi + q^3*phi = 0", "dt phi + phi*phi = 0", "dt phi = 1.0", "dt phi = q*phi",
                                 "dt phi = phi/phi", "dt phi = nope*phi", "dt phi = 2 phi", "phi = phi"])
def test_rejected_input(bad):
    r = Recorder()
    m = Model(r)
    m.create_field("phi", True)
    with pytest.raises(EquationError):
        m.add_equation(bad)
    with pytest.raises(EquationError):
        m.create_field("dt", True)
    with pytest.raises(EquationError):
        m.add_noise("phi", "iqx")


def test_parsed_and_hand_written_systems_give_the_same_trajectory(oracle):
    """the parsed Model-B listing and workloads.model_b drive the oracle to bit-identical fields"""
    cfg = wl.make_config("modelb_128", n=(16, 16))
    a, ids = wl.build(oracle, cfg, prec="f64")
    s = oracle.System(cfg["n"], (1.0, 1.0), cfg["dt"], prec="f64", seed=cfg["seed"])
    m = Model(s)
    for k, v in cfg["params"].items():
        m.add_parameter(k, v)
    m.create_field("phi", True)
    m.add_equation("dt phi + (a*q^2 + k*q^4)*phi = -b*q^2*phi^3")
    m.add_noise("phi", "D*q^2")
    s.finalize()
    s.set_field(m.ids()["phi"], wl.initial_conditions(cfg)["phi"])
    a.step(20)
    s.step(20)
    assert np.array_equal(a.get_field(ids["phi"]), s.get_field(m.ids()["phi"]))


def _readme_python_blocks():
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    return re.findall(r"```python\n(.*?)```", open(os.path.join(root, "README.md")).read(), flags=re.S)


def test_readme_equation_example_is_stable(oracle):
    """The front-page equation-string example, run as printed (the oracle's System standing in for the GPU one): the
    stiff k*q^4 term must sit on the implicit side (reading A8 makes anything on the rhs explicit; with k = 4, dt = 0.01,
    dx = 1 an explicit k*q^4 has an Euler factor of about -14 at the top mode), so 100 steps from a noisy start stay
    finite and bounded."""
    blocks = [b for b in _readme_python_blocks() if "add_equation" in b]
    assert len(blocks) == 1
    src = blocks[0]
    assert "pss.System(" in src and "dt phi + k*q^4*phi" in src

    class _Shim:                                   # `pss.System` of the snippet -> the CPU oracle, smaller lattice
        @staticmethod
        def System(n, dx, dt, **kw):
            return oracle.System((64, 64), dx, dt, **kw)

    env = {"pss": _Shim}
    exec(compile(src, "README.md", "exec"), env)
    s, phi = env["s"], env["phi"]
    rng = np.random.default_rng(7)
    s.set_field(phi, (0.1 * rng.standard_normal((64, 64))).astype(np.float32))
    s.step(100)
    x = np.asarray(s.get_field(phi), dtype=np.float64)
    assert np.isfinite(x).all()
    assert np.max(np.abs(x)) < 2.0                 # frames are +-1, the bulk stays inside the double well
