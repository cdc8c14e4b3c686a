"""Seeded synthetic workloads shared by the CUDA path and the oracle (inputs only).

This module holds NONE of the method's arithmetic: it only
  * generates initial conditions from a seed (reading A16 of DESIGN.md), and
  * states each workload's field system as the sequence of boundary calls (pss.h section
    "Worked mapping"), through whichever binding object it is handed (``api.System``).

The paper's benchmark workload is Model B on N x N power-of-two lattices started from "a small
random perturbation over a uniform state"; there is no dataset.  The
configs below are BASELINE.json's five configurations with the seeds of DESIGN.md.
"""
import numpy as np

# --------------------------------------------------------------------------------------------
# initial conditions: u24 = (w0 >> 8) * 2^-24 with w = Philox4x32-10(counter=(site_lo, site_hi,
# 0, 0x49430000 | field), key=seed); phi0 = lo + (hi - lo) * u24 in double, cast by the caller.
# --------------------------------------------------------------------------------------------
_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def _ic_words(seed, field, nsites):
    site = np.arange(nsites, dtype=np.uint64)
    c0 = site & _MASK
    c1 = site >> _S32
    c2 = np.zeros(nsites, dtype=np.uint64)
    c3 = np.full(nsites, (0x49430000 | (int(field) & 0xFFFF)), dtype=np.uint64)
    k0 = int(seed) & 0xFFFFFFFF
    k1 = (int(seed) >> 32) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        n0 = (p1 >> _S32) ^ c1 ^ np.uint64(k0)
        n1 = p1 & _MASK
        n2 = (p0 >> _S32) ^ c3 ^ np.uint64(k1)
        n3 = p0 & _MASK
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0 = (k0 + _W0) & 0xFFFFFFFF
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return c0


def uniform_field(seed, field, shape, lo, hi, dtype=np.float64):
    """phi0 over a lattice of ``shape`` (slowest axis first, x last): lo + (hi-lo)*u24."""
    n = int(np.prod(shape))
    w0 = _ic_words(seed, field, n)
    u24 = (w0 >> np.uint64(8)).astype(np.float64) * (1.0 / 16777216.0)
    return (lo + (hi - lo) * u24).reshape(shape).astype(dtype)


# --------------------------------------------------------------------------------------------
# field systems, stated through the boundary calls
# --------------------------------------------------------------------------------------------
def model_b(s, a=-1.0, b=1.0, k=1.0, D=0.0):
    """dt phi + (a q^2 + k q^4) phi = -b q^2 phi^3, conserved noise D q^2."""
    f = s.add_field("phi", True)
    s.add_linear(f, {"coef": a, "q2_pow": 1})
    s.add_linear(f, {"coef": k, "q2_pow": 2})
    s.add_term(f, {"coef": -b, "q2_pow": 1}, [f, f, f])
    if D > 0:
        s.set_noise(f, D, 2)
    return {"phi": f}


def diffusion(s, D=1.0, noise=0.0):
    """dt phi + D q^2 phi = 0 with non-conserved noise."""
    f = s.add_field("phi", True)
    s.add_linear(f, {"coef": D, "q2_pow": 1})
    if noise > 0:
        s.set_noise(f, noise, 0)
    return {"phi": f}


def kpz(s, nu=1.0, lam=2.0, D=1.0):
    """dt h = nu lap h + (lam/2)|grad h|^2 + noise (Eq. 12; reading A15)."""
    ndim = s.ndim
    h = s.add_field("h", True)
    s.add_linear(h, {"coef": nu, "q2_pow": 1})
    ids = {"h": h}
    for j in range(ndim):
        g = s.add_field("g" + "xyz"[j], False)
        iq = [0, 0, 0]
        iq[j] = 1
        s.add_aux_def(g, {"coef": 1.0, "iq_pow": tuple(iq)}, h)
        s.add_term(h, {"coef": 0.5 * lam}, [g, g])
        ids["g" + "xyz"[j]] = g
    if D > 0:
        s.set_noise(h, D, 0)
    return ids


def nematic(s, A=-1.0, C=1.0, K=1.0, lam=1.0, alpha=-2.0, eta=1.0, D=1e-3):
    """2D wet active nematic, reading A14 of DESIGN.md (equations are BASELINE.json's, not the paper's)."""
    qxx = s.add_field("Qxx", True)
    qxy = s.add_field("Qxy", True)
    for q in (qxx, qxy):
        s.add_linear(q, {"coef": A})
        s.add_linear(q, {"coef": K, "q2_pow": 1})
    r = alpha / eta
    psi = s.add_field("psi_s", False)          # stream function
    s.add_aux_def(psi, {"coef": -2.0 * r, "invq_pow": 4, "iq_pow": (1, 1, 0)}, qxx)
    s.add_aux_def(psi, {"coef": r, "invq_pow": 4, "iq_pow": (2, 0, 0)}, qxy)
    s.add_aux_def(psi, {"coef": -r, "invq_pow": 4, "iq_pow": (0, 2, 0)}, qxy)
    vx = s.add_field("vx", False)
    s.add_aux_def(vx, {"coef": 1.0, "iq_pow": (0, 1, 0)}, psi)
    vy = s.add_field("vy", False)
    s.add_aux_def(vy, {"coef": -1.0, "iq_pow": (1, 0, 0)}, psi)
    om = s.add_field("omega", False)
    s.add_aux_def(om, {"coef": 1.0, "q2_pow": 1}, psi)
    exx = s.add_field("Exx", False)
    s.add_aux_def(exx, {"coef": 1.0, "iq_pow": (1, 0, 0)}, vx)
    exy = s.add_field("Exy", False)
    s.add_aux_def(exy, {"coef": 0.5, "iq_pow": (1, 0, 0)}, vy)
    s.add_aux_def(exy, {"coef": 0.5, "iq_pow": (0, 1, 0)}, vx)
    grads = {}
    for name, q in (("Qxx", qxx), ("Qxy", qxy)):
        for j, ax in enumerate("xy"):
            g = s.add_field("d%s%s" % (ax, name), False)
            iq = [0, 0, 0]
            iq[j] = 1
            s.add_aux_def(g, {"coef": 1.0, "iq_pow": tuple(iq)}, q)
            grads[(name, ax)] = g
    one = {"coef": 1.0}
    # Qxx
    s.add_term(qxx, {"coef": -1.0}, [vx, grads[("Qxx", "x")]])
    s.add_term(qxx, {"coef": -1.0}, [vy, grads[("Qxx", "y")]])
    s.add_term(qxx, {"coef": lam}, [exx])
    s.add_term(qxx, {"coef": -1.0}, [om, qxy])
    s.add_term(qxx, {"coef": -C}, [qxx, qxx, qxx])
    s.add_term(qxx, {"coef": -C}, [qxy, qxy, qxx])
    # Qxy
    s.add_term(qxy, {"coef": -1.0}, [vx, grads[("Qxy", "x")]])
    s.add_term(qxy, {"coef": -1.0}, [vy, grads[("Qxy", "y")]])
    s.add_term(qxy, {"coef": lam}, [exy])
    s.add_term(qxy, dict(one), [om, qxx])
    s.add_term(qxy, {"coef": -C}, [qxx, qxx, qxy])
    s.add_term(qxy, {"coef": -C}, [qxy, qxy, qxy])
    if D > 0:
        s.set_noise(qxx, D, 0)
        s.set_noise(qxy, D, 0)
    return {"Qxx": qxx, "Qxy": qxy, "psi_s": psi, "vx": vx, "vy": vy, "omega": om,
            "Exx": exx, "Exy": exy}


def model_h(s, k=1.0, eta=2.0, D=0.005):
    """Binary fluid ("model H" class) in stream-function form, stated through the equation-string
    front end: chemical potential mu = phi^3 - phi + k q^2 phi (a product-defined intermediate field), Stokes flow driven
    by the capillary force, eta q^4 w = d_x mu d_y phi - d_y mu d_x phi (an intermediate field with its own lhs),
    v = (d_y w, -d_x w), dt phi = -q^2 mu - v.grad phi with the stiff part implicit.  The paper's own Model H listing is
    not in the paper; this is a model of the same structure (several intermediate fields, two dependency levels)."""
    from .equations import Model
    m = Model(s)
    m.add_parameter("k", k)
    m.add_parameter("eta", eta)
    m.add_parameter("D", D)
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
    if D > 0:
        m.add_noise("phi", "D*q^2")
    return m.ids()


# --------------------------------------------------------------------------------------------
# BASELINE.json configs (seeds: DESIGN.md "Input recipe")
# --------------------------------------------------------------------------------------------
CONFIGS = {
    "modelb_128": dict(model="model_b", n=(128, 128), dx=1.0, dt=0.01, steps=1000, seed=2405024101,
                       params=dict(a=-1.0, b=1.0, k=1.0, D=0.01), ic={"phi": (-0.1, 0.1)}),
    "modelb_1024": dict(model="model_b", n=(1024, 1024), dx=1.0, dt=0.01, steps=10000, seed=2405024102,
                        params=dict(a=-1.0, b=1.0, k=1.0, D=0.05), ic={"phi": (0.05, 0.15)}),
    "modelb_256c": dict(model="model_b", n=(256, 256, 256), dx=1.0, dt=0.005, steps=2000, seed=2405024103,
                        params=dict(a=-1.0, b=1.0, k=1.0, D=0.01), ic={"phi": (-0.1, 0.1)}),
    "nematic_1024": dict(model="nematic", n=(1024, 1024), dx=1.0, dt=0.01, steps=250, seed=2405024104,
                         params=dict(A=-1.0, C=1.0, K=1.0, lam=1.0, alpha=-2.0, eta=1.0, D=1e-3),
                         ic={"Qxx": (-0.01, 0.01), "Qxy": (-0.01, 0.01)}),
    "kpz_4096": dict(model="kpz", n=(4096, 4096), dx=1.0, dt=0.01, steps=5000, seed=2405024105,
                     params=dict(nu=1.0, lam=2.0, D=1.0), ic={"h": None}),
}
for _e in range(8, 14):  # Model-B lattice sweep 256^2 .. 8192^2 (config-2 equation)
    _n = 1 << _e
    CONFIGS["sweep_%d" % _n] = dict(model="model_b", n=(_n, _n), dx=1.0, dt=0.01, steps=1000, seed=2405024106,
                                    params=dict(a=-1.0, b=1.0, k=1.0, D=0.05), ic={"phi": (0.05, 0.15)})

# not a BASELINE config: the multi-round path on the lattice of the headline
CONFIGS["modelh_1024"] = dict(model="model_h", n=(1024, 1024), dx=1.0, dt=0.005, steps=1000, seed=2405024108,
                              params=dict(k=1.0, eta=2.0, D=0.005), ic={"phi": (-0.1, 0.1)})

MODELS = {"model_b": model_b, "kpz": kpz, "nematic": nematic, "diffusion": diffusion, "model_h": model_h}


def make_config(name, n=None, **over):
    """copy of a config, optionally on a smaller lattice ``n`` (same equation, same seed)."""
    cfg = dict(CONFIGS[name])
    cfg["params"] = dict(cfg["params"])
    if n is not None:
        cfg["n"] = tuple(int(v) for v in n)
    for k, v in over.items():
        if k in cfg["params"]:
            cfg["params"][k] = v
        else:
            cfg[k] = v
    return cfg


def initial_conditions(cfg, dtype=np.float64, ids=None):
    """{field name: array shaped n[::-1]} from the config's seed (A16).  The Philox counter carries the field id:
    ``ids[name]`` when the caller has them (``build``), else the position in ``cfg["ic"]`` (the same number for every
    workload here, whose dynamic fields are created first)."""
    shape = tuple(cfg["n"])[::-1]
    out = {}
    for pos, (name, rng) in enumerate(cfg["ic"].items()):
        fid = pos if ids is None else ids[name]
        if rng is None:
            out[name] = np.zeros(shape, dtype=dtype)
        else:
            out[name] = uniform_field(cfg["seed"], fid, shape, rng[0], rng[1], dtype)
    return out


def build(api, cfg, prec="f32", dealias=None, set_ic=True, **sys_kwargs):
    """Create, describe, finalize (and bind, on the product side) one system through ``api.System``.

    ``api`` is either ``paper_2405_02410_b200`` (CUDA product) or the oracle binding; both expose
    the same method names.  Returns (system, ids).
    """
    n = tuple(cfg["n"])
    dx = cfg["dx"]
    dxs = tuple(dx) if isinstance(dx, (tuple, list)) else (float(dx),) * len(n)
    s = api.System(n, dxs, cfg["dt"], prec=prec, seed=cfg["seed"], **sys_kwargs)
    ids = MODELS[cfg["model"]](s, **cfg["params"])
    if dealias is not None:
        s.set_dealias(dealias)
    s.finalize()
    if set_ic:
        dtype = np.float32 if prec == "f32" else np.float64
        for name, arr in initial_conditions(cfg, dtype, ids).items():
            s.set_field(ids[name], arr)
    return s, ids
