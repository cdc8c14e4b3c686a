"""Shared comparison helpers of the `-m gpu` parity tests (numpy only; no method arithmetic).

Two metrics per dynamic field, both CUDA path vs. oracle on the same seeded inputs:
  * relative L2 over the real-space field (north_star's tolerance, PAPER.md:125 iterated), and
  * a per-mode check on the half-spectrum: max_q |phi_q(gpu) - phi_q(oracle)| / (rms + |phi_q(oracle)|), rms = the rms
    magnitude of the q != 0 modes (a mode much larger than the rest, e.g. the mean, is measured against itself).  An
    L2 over 10^6..10^8 sites can dilute one wrong boundary-plane or Nyquist mode at the long horizons (one mode of
    typical size that is entirely wrong has ratio ~0.5); rounding errors are spread over all modes, so their maximum
    over M modes stays within a few sigma of the L2 figure.  The bound is MODE_FACTOR x the L2 tolerance.
"""
import numpy as np

TOL1 = {"f32": 1e-5, "f64": 1e-12}
TOLN = {"f32": 1e-3, "f64": 1e-9}
MODE_FACTOR = 30.0


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.linalg.norm(b.ravel())
    return np.linalg.norm((a - b).ravel()) / (den if den > 0 else 1.0)


def mode_err(spec_g, spec_o):
    """max_q |d phi_q| / (rms_{q != 0} |phi_q(oracle)| + |phi_q(oracle)|), on the logical half-spectrum"""
    g = np.asarray(spec_g).astype(np.complex128).ravel()
    o = np.asarray(spec_o).astype(np.complex128).ravel()
    d = np.abs(g - o)
    mag2 = np.abs(o) ** 2
    if mag2.size > 1:
        rms = np.sqrt((mag2.sum() - mag2[0]) / (mag2.size - 1))
    else:
        rms = 0.0
    if rms == 0.0:
        rms = max(np.sqrt(mag2.max()), 1.0)
    rel = d / (rms + np.sqrt(mag2))
    j = int(np.argmax(rel))
    return float(rel[j]), j


def compare_fields(g, o, dyn, tol, what, modes=True, quiet=False):
    """assert both metrics for every field id in ``dyn``; returns the worst relative L2"""
    worst, worst_m = 0.0, 0.0
    for f in dyn:
        a, b = g.get_field(f), o.get_field(f)
        assert np.all(np.isfinite(a)), what
        e = rel_l2(a, b)
        worst = max(worst, e)
        assert e <= tol, "%s: field %d rel L2 %.3e > %.1e" % (what, f, e, tol)
        if modes:
            sg = g.get_field_fourier(f)
            so = o.get_field_fourier_f64(f) if hasattr(o, "get_field_fourier_f64") else o.get_field_fourier(f)
            assert sg.shape == so.shape
            em, j = mode_err(sg, so)
            worst_m = max(worst_m, em)
            assert em <= MODE_FACTOR * tol, "%s: field %d mode %s: |d phi_q| / rms|phi_q| = %.3e > %.1e" % (
                what, f, np.unravel_index(j, sg.shape), em, MODE_FACTOR * tol)
    if not quiet:
        print("%s: rel L2 %.3e (tol %.1e), worst mode %.3e" % (what, worst, tol, worst_m))
    return worst


def both(wl, pss, oracle, cfg, prec, dealias=None):
    g, ids = wl.build(pss, cfg, prec=prec, dealias=dealias)
    o, ids_o = wl.build(oracle, cfg, prec=prec, dealias=dealias)
    assert ids == ids_o
    return g, o, [ids[name] for name in cfg["ic"].keys()]


def run_horizons(wl, pss, oracle, cfg, prec, horizons, what, dealias=None):
    """horizons: [(total steps, tolerance), ...] increasing; each increment is ONE pss_step(n) call."""
    g, o, dyn = both(wl, pss, oracle, cfg, prec, dealias)
    done = 0
    for total, tol in horizons:
        g.step(total - done)
        o.step(total - done)
        done = total
        assert g.step_count == total
        compare_fields(g, o, dyn, tol, "%s %s, %d steps" % (what, prec, total))
    return g
