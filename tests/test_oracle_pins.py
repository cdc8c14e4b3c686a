"""Pins of the CPU oracle against what the paper and the mathematics fix (P1..P14).

None of these compares the oracle with itself: each expected value is a closed form, a brute-force
O(N^2)/O(N^3) sum written out with numpy, a library routine (numpy.fft, ATen's Philox), a value the
paper prints, or an exact invariant.  All run on CPU ("-m 'not gpu'").
"""
import itertools
import math

import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as W


# ------------------------------------------------------------------------------------------ P1
def _dft_matrix(n, sign):
    j = np.arange(n)
    return np.exp(sign * 2j * np.pi * np.outer(j, j) / n)


@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64])
def test_p1_fft_equals_dft_definition(oracle, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal((5, n)) + 1j * rng.standard_normal((5, n))
    for sign in (-1, +1):
        want = x @ _dft_matrix(n, sign).T        # X[k] = sum_n x[n] exp(sign 2 pi i n k / N)
        got = oracle.fft_lines(x, sign)
        assert np.abs(got - want).max() < 1e-12 * n


@pytest.mark.parametrize("shape", [(16,), (8, 16), (4, 8, 16), (2, 2, 4), (32, 8)])
def test_p1_r2c_c2r_multidim(oracle, shape):
    rng = np.random.default_rng(sum(shape))
    r = rng.standard_normal(shape)
    # brute-force multi-dimensional DFT from the definition, one axis at a time with explicit matrices
    full = r.astype(np.complex128)
    for ax, n in enumerate(shape):
        full = np.moveaxis(np.tensordot(_dft_matrix(n, -1), np.moveaxis(full, ax, 0), axes=1), 0, ax)
    want = full[..., : shape[-1] // 2 + 1]
    got = oracle.r2c(r)
    assert np.abs(got - want).max() < 1e-11
    assert np.abs(got - np.fft.rfftn(r)).max() < 1e-11          # library special case
    back = oracle.c2r(got, shape[-1])
    assert np.abs(back - r).max() < 1e-13                        # C2R(R2C(x)) = x, carries 1/N
    # Parseval on the full spectrum
    assert abs((np.abs(full) ** 2).sum() / r.size - (r ** 2).sum()) < 1e-10


# ------------------------------------------------------------------------------------------ P8
def test_p8_philox_known_answers(oracle):
    # tests/golden/philox4x32_10_kat.txt: Random123 known-answer vectors (Salmon et al., SC'11)
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    n = 0
    for line in open(path):
        line = line.split("#")[0].split()
        if not line:
            continue
        v = [int(t, 16) for t in line]
        assert oracle.philox(v[0:4], v[4:6]) == tuple(v[6:10])
        n += 1
    assert n >= 2


def test_p8_philox_matches_aten_engine(oracle, tmp_path):
    """Library pin: ATen's at::philox_engine (torch/include/ATen/core/PhiloxRNGEngine.h) run on the host."""
    import ctypes
    import os
    import subprocess
    torch = pytest.importorskip("torch")
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    if not os.path.exists(os.path.join(inc, "ATen", "core", "PhiloxRNGEngine.h")):
        pytest.skip("ATen Philox header not present")
    src = tmp_path / "aten_philox.cpp"
    src.write_text(
        '#include <ATen/core/PhiloxRNGEngine.h>\n'
        'extern "C" void aten_block(unsigned long long seed, unsigned long long sub,\n'
        '                           unsigned long long off, unsigned int* out) {\n'
        '  at::philox_engine e(seed, sub, off);\n'
        '  for (int i = 0; i < 4; ++i) out[i] = e();\n'
        '}\n')
    so = tmp_path / "aten_philox.so"
    r = subprocess.run(["g++", "-std=c++17", "-O1", "-shared", "-fPIC", "-I", inc, "-o", str(so), str(src)],
                       capture_output=True, text=True)
    if r.returncode != 0:
        pytest.skip("cannot compile ATen Philox shim: " + r.stderr[-300:])
    lib = ctypes.CDLL(str(so))
    lib.aten_block.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.POINTER(ctypes.c_uint32)]
    rng = np.random.default_rng(8)
    cases = [((0, 0, 0, 0), (0, 0)), ((0xFFFFFFFF,) * 4, (0xFFFFFFFF,) * 2)]
    for _ in range(64):
        cases.append((tuple(int(v) for v in rng.integers(0, 2 ** 32, 4)), tuple(int(v) for v in rng.integers(0, 2 ** 32, 2))))
    for ctr, key in cases:
        out = (ctypes.c_uint32 * 4)()
        # engine: key = seed, counter = (offset_lo, offset_hi, subsequence_lo, subsequence_hi)
        lib.aten_block(key[0] | (key[1] << 32), ctr[2] | (ctr[3] << 32), ctr[0] | (ctr[1] << 32), out)
        assert oracle.philox(ctr, key) == tuple(int(v) for v in out)


def test_p8_noise_counter_layout(oracle):
    """bits of mode m at (seed, step, field) are Philox(ctr=(m_lo,m_hi,step_lo,(step_hi&0xffff)<<16|field), key=seed)."""
    seed = 0x1234567890ABCDEF
    s = oracle.System((8, 4), (1.0, 1.0), 0.1, prec="f32", seed=seed)
    f0 = s.add_field("a", True)
    f1 = s.add_field("b", True)
    s.finalize()
    step = (5 << 32) | 77
    bits, _ = s.debug_noise(f1, step)
    nxh = 5
    for ky, kx in [(0, 0), (3, 4), (2, 1)]:
        m = ky * nxh + kx
        want = oracle.philox((m, 0, 77, (5 << 16) | f1), (seed & 0xFFFFFFFF, seed >> 32))
        assert tuple(int(v) for v in bits[ky, kx]) == want
    assert f0 == 0


# ------------------------------------------------------------------------------------------ P2
def _signed(k, n):
    return k if k <= n // 2 else k - n


def _step_product_hat(oracle, phi0, dealias, order=3):
    """P_hat of phi^order via one explicit step of dt phi = -phi^order (Eq. 4/6/8)."""
    n = phi0.shape[-1]
    dt = 0.125
    s = oracle.System(phi0.shape[::-1], (1.0,) * phi0.ndim, dt, prec="f64", seed=1)
    f = s.add_field("phi", True)
    s.add_term(f, {"coef": -1.0}, [f] * order)
    s.set_dealias(dealias)
    s.finalize()
    s.set_field(f, phi0)
    h0 = s.get_field_fourier_f64(f)
    s.step(1)
    h1 = s.get_field_fourier_f64(f)
    return h0, (h0 - h1) / dt, s


@pytest.mark.parametrize("n", [8, 16])
def test_p2_cubic_product_is_direct_convolution(oracle, n):
    """Eq. 5 discretised: (phi^3)^_q = N^-2 sum_{k,l} phi_k phi_l phi_{q-k-l}; O(N^3) brute force."""
    rng = np.random.default_rng(n)
    phi0 = rng.standard_normal(n)
    full = np.fft.fft(phi0)
    # unmasked: circular convolution
    _, P, _ = _step_product_hat(oracle, phi0, oracle.DEALIAS_OFF)
    for q in range(n // 2 + 1):
        acc = 0j
        for k in range(n):
            for l in range(n):
                acc += full[k] * full[l] * full[(q - k - l) % n]
        assert abs(P[q] - acc / n ** 2) < 1e-12 * max(1.0, abs(acc))
    # masked (paper rule, cubic => keep |s(k)| < N/4 strictly): NON-wrapping convolution on the kept band
    _, Pm, s = _step_product_hat(oracle, phi0, oracle.DEALIAS_PAPER)
    keep = [k for k in range(n) if 4 * abs(_signed(k, n)) < n]
    for q in range(n // 2 + 1):
        if 4 * abs(_signed(q, n)) >= n:
            continue
        acc = 0j
        for k in keep:
            for l in keep:
                for m in keep:
                    if _signed(k, n) + _signed(l, n) + _signed(m, n) == _signed(q, n):   # no wrap
                        acc += full[k] * full[l] * full[m]
        assert abs(Pm[q] - acc / n ** 2) < 1e-12 * max(1.0, abs(acc)), q
    mask = s.debug_mask(0)
    assert [int(v) for v in mask] == [1 if 4 * k < n else 0 for k in range(n // 2 + 1)]


def test_p2_quadratic_two_thirds_rule_2d(oracle):
    """n = 2 gives the two-thirds rule; product equals the non-wrapping 2-D convolution."""
    ny, nx = 8, 16
    rng = np.random.default_rng(3)
    phi0 = rng.standard_normal((ny, nx))
    full = np.fft.fft2(phi0)
    _, P, s = _step_product_hat(oracle, phi0, oracle.DEALIAS_PAPER, order=2)
    mask = s.debug_mask(0)
    keepx = [k for k in range(nx) if 3 * abs(_signed(k, nx)) < nx]
    keepy = [k for k in range(ny) if 3 * abs(_signed(k, ny)) < ny]
    for ky in range(ny):
        for kx in range(nx // 2 + 1):
            assert mask[ky, kx] == (1 if (ky in keepy and kx in keepx) else 0)
    for qy in keepy:
        for qx in [k for k in keepx if k <= nx // 2]:
            acc = 0j
            for ky, kx in itertools.product(keepy, keepx):
                ly, lx = _signed(qy, ny) - _signed(ky, ny), _signed(qx, nx) - _signed(kx, nx)
                if 3 * abs(ly) < ny and 3 * abs(lx) < nx:
                    acc += full[ky, kx] * full[ly % ny, lx % nx]
            assert abs(P[qy, qx] - acc / (nx * ny)) < 1e-11 * max(1.0, abs(acc))


# ------------------------------------------------------------------------------------------ P3
def test_p3_uniform_cubic_decay(oracle):
    """dt phi = -phi^3 (Eq. 4) on a uniform field: exact Euler recurrence; closed form as dt -> 0."""
    phi0, T = 0.8, 1.0
    errs = []
    for nsteps in (50, 100, 200):
        dt = T / nsteps
        s = oracle.System((8, 8), (1.0, 1.0), dt, prec="f64", seed=1)
        f = s.add_field("phi", True)
        s.add_term(f, {"coef": -1.0}, [f, f, f])
        s.finalize()
        s.set_field(f, np.full((8, 8), phi0))
        s.step(nsteps)
        got = s.get_field(f)
        p = phi0
        for _ in range(nsteps):
            p = p - dt * p ** 3
        assert np.abs(got - p).max() < 1e-13
        errs.append(abs(got[0, 0] - phi0 / math.sqrt(1 + 2 * phi0 ** 2 * T)))
    assert errs[0] / errs[1] == pytest.approx(2.0, rel=0.05)     # first order in dt
    assert errs[1] / errs[2] == pytest.approx(2.0, rel=0.05)
    assert errs[2] < 2e-3


# ------------------------------------------------------------------------------------------ P4
@pytest.mark.parametrize("n,dx", [((16,), (0.5,)), ((8, 16), (1.0, 0.7)), ((4, 8, 8), (1.0, 2.0, 0.5))])
def test_p4_linear_diffusion_mode_decay(oracle, n, dx):
    """noiseless dt phi + D q^2 phi = 0: every mode is phi_q(0) (1 + dt D q^2)^-n exactly (Eq. 18)."""
    D, dt, nsteps = 0.7, 0.05, 7
    s = oracle.System(n, dx, dt, prec="f64", seed=1)
    ids = W.diffusion(s, D=D)
    s.finalize()
    rng = np.random.default_rng(4)
    phi0 = rng.standard_normal(n[::-1])
    s.set_field(ids["phi"], phi0)
    h0 = np.fft.rfftn(phi0)
    s.step(nsteps)
    h = s.get_field_fourier_f64(ids["phi"])
    q2 = np.zeros(h.shape)
    for ax, (nj, dxj) in enumerate(zip(n, dx)):          # n is x-first; array axes are reversed
        k = np.fft.fftfreq(nj, d=dxj) * 2 * np.pi
        if ax == 0:
            k = np.abs(k[: nj // 2 + 1]); k[-1] = np.pi / dxj
        shp = [1] * len(n); shp[len(n) - 1 - ax] = k.size
        q2 = q2 + (k.reshape(shp)) ** 2
    want = h0 / (1 + dt * D * q2) ** nsteps
    assert np.abs(h - want).max() < 1e-12 * np.abs(h0).max()


# ------------------------------------------------------------------------------------------ P5
def test_p5_conserved_mean_is_bit_identical(oracle):
    cfg = W.make_config("modelb_128", n=(16, 16))
    s, ids = W.build(oracle, cfg, prec="f64")
    m0 = s.get_field_fourier_f64(ids["phi"])[0, 0]
    for _ in range(5):
        s.step(3)
        m = s.get_field_fourier_f64(ids["phi"])[0, 0]
        assert m.real == m0.real and m.imag == m0.imag


# ------------------------------------------------------------------------------------------ P6
def test_p6_stationary_structure_factor(oracle):
    """linear noisy equation dt phi + (a + k q^2) phi = noise: <|phi_q|^2> = (N/dV) 2D~/(lam (2 + dt lam))."""
    nx = ny = 8
    dx, dt, a, k, D = 0.8, 0.05, 1.0, 0.5, 0.3
    s = oracle.System((nx, ny), (dx, dx), dt, prec="f64", seed=99)
    s.set_threads(1)
    f = s.add_field("phi", True)
    s.add_linear(f, {"coef": a})
    s.add_linear(f, {"coef": k, "q2_pow": 1})
    s.set_noise(f, D, 2)                      # conserved: D~ = D q^2
    s.finalize()
    s.set_field(f, np.zeros((ny, nx)))
    s.step(400)                               # relax (slowest rate a = 1 -> 20 time units)
    acc = np.zeros((ny, nx // 2 + 1))
    nsamp = 6000
    for _ in range(nsamp):
        s.step(2)
        acc += np.abs(s.get_field_fourier_f64(f)) ** 2
    acc /= nsamp
    qx = 2 * np.pi * np.arange(nx // 2 + 1) / (nx * dx)
    qy = 2 * np.pi * np.fft.fftfreq(ny, d=1.0) * ny / (ny * dx)
    q2 = qy[:, None] ** 2 + qx[None, :] ** 2
    lam = a + k * q2
    want = (nx * ny / dx ** 2) * 2 * D * q2 / (lam * (2 + dt * lam))
    assert acc[0, 0] == 0.0                   # conserved noise never touches the mean
    sel = q2 > 0
    ratio = acc[sel] / want[sel]
    assert abs(ratio.mean() - 1.0) < 0.02     # ~ 1/sqrt(nsamp * modes)
    assert np.abs(ratio - 1.0).max() < 0.12   # per mode, ~ 4.5 sigma of sqrt(2/nsamp_eff)


# ------------------------------------------------------------------------------------------ P7
@pytest.mark.parametrize("n", [(16,), (16, 8), (8, 4, 4)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_p7_noise_is_hermitian_unit_variance(oracle, n, prec):
    s = oracle.System(n, (1.0,) * len(n), 0.1, prec=prec, seed=7)
    f = s.add_field("phi", True)
    s.finalize()
    nx = n[0]
    zs = []
    for step in range(300):
        _, z = s.debug_noise(f, step)
        zs.append(z)
        if step < 3:
            re = oracle.c2r(z, nx)
            back = oracle.r2c(re)
            assert np.abs(back - z).max() < 1e-12        # no implicit projection: z is a real field's spectrum
            # same statement with the library transform
            assert np.abs(np.fft.rfftn(np.fft.irfftn(z, s=n[::-1], axes=tuple(range(len(n))))) - z).max() < 1e-12
    zs = np.array(zs)
    # self-conjugate modes are exactly real
    idx = np.indices(zs.shape[1:])
    kx = idx[-1]
    selfc = (kx == 0) | (kx == nx // 2)
    for ax, nj in enumerate(n[::-1][:-1]):
        selfc &= (idx[ax] == 0) | (idx[ax] == nj // 2)
    assert np.all(zs[:, selfc].imag == 0.0)
    var = (np.abs(zs) ** 2).mean(axis=0)
    assert abs(var.mean() - 1.0) < 5.0 / math.sqrt(zs.size)
    assert np.abs(var - 1.0).max() < 0.45               # 300 samples per mode
    assert abs(zs.mean()) < 4.0 / math.sqrt(zs.size)
    # real-space variance per site of the white field c2r(amp z), amp^2 = N: exactly 1 per site in expectation
    re = np.array([oracle.c2r(zs[i] * math.sqrt(np.prod(n)), nx) for i in range(100)])
    assert abs((re ** 2).mean() - 1.0) < 5.0 * math.sqrt(2.0 / re.size)


def test_p7_noise_amplitude_real_space_variance(oracle):
    """non-conserved noise, L = 0: after one step from 0, phi(x) has variance 2 D dt / dV per site (reading A1)."""
    n, dx, dt, D = (32, 32), (0.5, 0.25), 0.02, 0.7
    s = oracle.System(n, dx, dt, prec="f64", seed=11)
    f = s.add_field("phi", True)
    s.set_noise(f, D, 0)
    s.finalize()
    s.set_field(f, np.zeros(n[::-1]))
    s.step(1)
    v = s.get_field(f).var()
    assert v == pytest.approx(2 * D * dt / (dx[0] * dx[1]), rel=0.12)


@pytest.mark.parametrize("a", [-2, -1, 1, 2, 3])
@pytest.mark.parametrize("n,dx", [((16, 8), (0.5, 1.25)), ((8, 4, 4), (1.0, 0.7, 2.0)), ((32,), (0.3,))])
def test_p7_noise_amplitude_odd_and_negative_q_powers(oracle, a, n, dx):
    """noise prefactor "a power of q^2 and 1/q" (reading A13: D~ = D |q|^a, any integer a), with
    L = 0 and no rhs: one step from 0 gives phi_q = nu_q (Eq. 18), so
      (i)  mode by mode  phi_q / z_q = sqrt(2 D |q|^a dt N / dV)  (z_q: the unit Hermitian Gaussian pinned by P7;
           PAPER.md:113 Eq. 16 with reading A1), 0 at q = 0 for a < 0 (A10), and
      (ii) averaged over seeds  <|phi_q|^2> = 2 D |q|^a dt N / dV.
    |q| is written out here from the integer mode numbers (q_j = 2 pi s(k_j) / (N_j dx_j), Nyquist index -> pi/dx_j)."""
    dt, D = 0.02, 0.7
    ndim = len(n)
    N, dV = float(np.prod(n)), float(np.prod(dx))
    qs = []
    for j in range(ndim):
        k = np.arange(n[j] // 2 + 1) if j == 0 else np.fft.fftfreq(n[j], 1.0 / n[j])
        qs.append(2 * np.pi * np.abs(k) / (n[j] * dx[j]))
    grids = np.meshgrid(*qs[::-1], indexing="ij")            # slowest axis first, x last (the half-spectrum layout)
    qabs = np.sqrt(sum(g * g for g in grids))
    with np.errstate(divide="ignore"):
        qa = np.where(qabs > 0, qabs ** float(a), 0.0 if a < 0 else (1.0 if a == 0 else 0.0))
    amp2 = 2 * D * qa * dt * N / dV
    acc = np.zeros_like(amp2)
    nseed = 160
    for seed in range(nseed):
        s = oracle.System(n, dx, dt, prec="f64", seed=1000 + seed)
        f = s.add_field("phi", True)
        s.set_noise(f, D, a)
        s.finalize()
        s.set_field(f, np.zeros(n[::-1]))
        s.step(1)
        spec = s.get_field_fourier_f64(f)
        if seed < 3:
            _, z = s.debug_noise(f, 0)
            assert np.abs(spec - np.sqrt(amp2) * z).max() <= 1e-12 * max(1.0, np.sqrt(amp2).max())
            if a < 0:
                assert spec.flat[0] == 0.0
        acc += np.abs(spec) ** 2
    sel = amp2 > 0
    ratio = (acc / nseed)[sel] / amp2[sel]
    assert abs(ratio.mean() - 1.0) < 5.0 / math.sqrt(nseed * sel.sum())
    assert np.abs(ratio - 1.0).max() < 0.6                  # 160 samples per mode (chi^2 with 1-2 dof)


# ------------------------------------------------------------------------------------------ P9
def test_p9_odd_derivative_nyquist_and_inverse_q(oracle):
    nx, ny, dx = 16, 8, 0.5
    s = oracle.System((nx, ny), (dx, dx), 0.1, prec="f64", seed=1)
    f = s.add_field("phi", True)
    g = s.add_field("g", False)
    s.add_aux_def(g, {"coef": 1.0, "iq_pow": (1, 0, 0)}, f)
    u = s.add_field("u", True)
    s.add_term(u, {"coef": 1.0}, [g])          # dt u = d phi/dx, explicit linear
    w = s.add_field("w", True)
    s.add_term(w, {"coef": 1.0, "invq_pow": 1}, [f])   # dt w = |q|^-1 phi
    s.finalize()
    # operator values
    assert s.debug_op({"iq_pow": (1, 0, 0)}, (nx // 2, 3)) == 0
    assert s.debug_op({"iq_pow": (2, 0, 0)}, (nx // 2, 0)) == pytest.approx(-(np.pi / dx) ** 2)
    assert s.debug_op({"iq_pow": (1, 0, 0)}, (3, 0)) == pytest.approx(1j * 2 * np.pi * 3 / (nx * dx))
    assert s.debug_op({"iq_pow": (0, 1, 0)}, (0, ny - 1)) == pytest.approx(-1j * 2 * np.pi / (ny * dx))
    assert s.debug_op({"invq_pow": 1}, (0, 0)) == 0
    assert s.debug_op({"invq_pow": 2, "q2_pow": 1}, (0, 0)) == 0
    assert s.debug_op({"invq_pow": 2, "q2_pow": 1}, (2, 1)) == pytest.approx(1.0)
    assert s.debug_op({"q2_pow": 2, "coef": 3.0}, (1, 2)) == pytest.approx(
        3.0 * ((2 * np.pi / (nx * dx)) ** 2 + (2 * np.pi * 2 / (ny * dx)) ** 2) ** 2)
    x = np.arange(nx) * dx
    y = np.arange(ny) * dx
    L = nx * dx
    phi = np.cos(2 * np.pi * 3 * x / L)[None, :] * np.ones(ny)[:, None] + np.cos(np.pi * x / dx)[None, :] \
        + 0.3 * np.sin(2 * np.pi * y / (ny * dx))[:, None] + 2.0
    s.set_field(f, phi)
    s.set_field(u, np.zeros_like(phi))
    s.set_field(w, np.zeros_like(phi))
    s.step(1)
    du = s.get_field(u) / 0.1
    want = -(2 * np.pi * 3 / L) * np.sin(2 * np.pi * 3 * x / L)[None, :] * np.ones(ny)[:, None]
    assert np.abs(du - want).max() < 1e-12     # d/dx of the Nyquist cosine is 0; result is real
    what = s.get_field_fourier_f64(w)
    assert what[0, 0] == 0                     # 1/|q| := 0 at q = 0


# ------------------------------------------------------------------------------------------ P10
def test_p10_explicit_cross_terms_use_time_t_values(oracle):
    dt = 0.1
    s = oracle.System((8,), (1.0,), dt, prec="f64", seed=1)
    u = s.add_field("u", True)
    v = s.add_field("v", True)
    s.add_term(u, {"coef": 1.0}, [v])
    s.add_term(v, {"coef": -1.0}, [u])
    s.finalize()
    rng = np.random.default_rng(10)
    u0, v0 = rng.standard_normal(8), rng.standard_normal(8)
    s.set_field(u, u0)
    s.set_field(v, v0)
    e0 = u0 ** 2 + v0 ** 2
    for n in range(1, 6):
        s.step(1)
        e = s.get_field(u) ** 2 + s.get_field(v) ** 2
        assert np.abs(e / e0 - (1 + dt * dt) ** n).max() < 1e-13


# ------------------------------------------------------------------------------------------ P11
def test_p11_kpz_single_mode_one_step(oracle):
    nx, ny, dx, dt, nu, lam, A, m = 32, 8, 0.5, 0.01, 1.0, 2.0, 0.3, 3
    s = oracle.System((nx, ny), (dx, dx), dt, prec="f64", seed=1)
    ids = W.kpz(s, nu=nu, lam=lam, D=0.0)
    s.finalize()
    q = 2 * np.pi * m / (nx * dx)
    x = np.arange(nx) * dx
    s.set_field(ids["h"], (A * np.cos(q * x))[None, :] * np.ones((ny, 1)))
    s.step(1)
    h = s.get_field_fourier_f64(ids["h"])
    N = nx * ny
    # (lam/2) (dh/dx)^2 = (lam/2) A^2 q^2 sin^2 = (lam/2) A^2 q^2 (1 - cos 2qx)/2
    assert h[0, 0].real == pytest.approx(dt * (lam / 2) * A * A * q * q / 2 * N, rel=1e-12)
    assert h[0, 2 * m].real == pytest.approx(-dt * (lam / 2) * A * A * q * q / 4 * N / (1 + dt * nu * (2 * q) ** 2), rel=1e-12)
    assert h[0, m].real == pytest.approx(A * N / 2 / (1 + dt * nu * q * q), rel=1e-12)
    rest = h.copy()
    rest[0, 0] = rest[0, m] = rest[0, 2 * m] = 0
    assert np.abs(rest).max() < 1e-10


def test_p11_kpz_cole_hopf_convergence(oracle):
    """noiseless KPZ: W = exp(lam h / 2 nu) obeys the heat equation; error -> 0 linearly in dt."""
    nx, dx, nu, lam, T = 64, 1.0, 1.0, 2.0, 2.0
    x = np.arange(nx) * dx
    h0 = 0.5 * np.cos(2 * np.pi * x / (nx * dx)) + 0.2 * np.sin(4 * np.pi * x / (nx * dx))
    W0 = np.exp(lam * h0 / (2 * nu))
    q = 2 * np.pi * np.fft.rfftfreq(nx, d=dx)
    WT = np.fft.irfft(np.fft.rfft(W0) * np.exp(-nu * q * q * T), n=nx)
    hT = 2 * nu / lam * np.log(WT)
    errs = []
    for nsteps in (200, 400):
        s = oracle.System((nx,), (dx,), T / nsteps, prec="f64", seed=1)
        ids = W.kpz(s, nu=nu, lam=lam, D=0.0)
        s.finalize()
        s.set_field(ids["h"], h0)
        s.step(nsteps)
        errs.append(np.abs(s.get_field(ids["h"]) - hT).max())
    assert errs[1] < 2e-3
    assert errs[0] / errs[1] == pytest.approx(2.0, rel=0.1)


# ------------------------------------------------------------------------------------------ P12
def test_p12_nematic_invariants(oracle):
    nx = ny = 16
    dt = 0.01
    s = oracle.System((nx, ny), (1.0, 1.0), dt, prec="f64", seed=5)
    ids = W.nematic(s, D=0.0)
    # probes: dt p = aux (explicit linear) so that p_hat = dt * aux_hat after one step from 0
    probes = {}
    for name in ("vx", "vy", "omega", "psi_s"):
        p = s.add_field("probe_" + name, True)
        s.add_term(p, {"coef": 1.0}, [ids[name]])
        probes[name] = p
    s.finalize()
    rng = np.random.default_rng(12)
    s.set_field(ids["Qxx"], rng.standard_normal((ny, nx)))
    s.set_field(ids["Qxy"], rng.standard_normal((ny, nx)))
    for p in probes.values():
        s.set_field(p, np.zeros((ny, nx)))
    s.step(1)
    vx = s.get_field_fourier_f64(probes["vx"]) / dt
    vy = s.get_field_fourier_f64(probes["vy"]) / dt
    om = s.get_field_fourier_f64(probes["omega"]) / dt
    ps = s.get_field_fourier_f64(probes["psi_s"]) / dt
    qx = 2 * np.pi * np.arange(nx // 2 + 1) / nx
    qy = 2 * np.pi * np.fft.fftfreq(ny)
    qy_even = qy.copy(); qy_even[ny // 2] = np.pi
    QX, QY = np.meshgrid(qx, qy, indexing="xy")
    scale = np.abs(vx).max()
    assert scale > 0.1
    # incompressible everywhere, also on the Nyquist lines where odd derivatives vanish (A9)
    QXo = QX.copy(); QXo[:, nx // 2] = 0
    QYo = QY.copy(); QYo[ny // 2, :] = 0
    assert np.abs(QXo * vx + QYo * vy).max() < 1e-12 * scale
    assert vx[0, 0] == 0 and vy[0, 0] == 0                     # no mean flow (A10)
    q2 = QX ** 2 + np.meshgrid(qx, qy_even, indexing="xy")[1] ** 2
    assert np.abs(om - q2 * ps).max() < 1e-12 * np.abs(om).max()
    # away from Nyquist lines the stream-function form equals P_T . (i q . alpha Q)/(eta q^2)
    Qxx = np.fft.rfft2(s_get_initial(rng_seed=12, which=0, shape=(ny, nx)))
    Qxy = np.fft.rfft2(s_get_initial(rng_seed=12, which=1, shape=(ny, nx)))
    alpha, eta = -2.0, 1.0
    fx = 1j * (QX * Qxx + QY * Qxy) * alpha
    fy = 1j * (QX * Qxy - QY * Qxx) * alpha
    with np.errstate(divide="ignore", invalid="ignore"):
        qf = QX * fx + QY * fy
        vx_p = (fx - QX * qf / (QX ** 2 + QY ** 2)) / (eta * (QX ** 2 + QY ** 2))
    inner = np.ones_like(QX, dtype=bool)
    inner[ny // 2, :] = False; inner[:, nx // 2] = False; inner[0, 0] = False
    assert np.abs(vx[inner] - vx_p[inner]).max() < 1e-11 * scale


def s_get_initial(rng_seed, which, shape):
    rng = np.random.default_rng(rng_seed)
    a = rng.standard_normal(shape)
    b = rng.standard_normal(shape)
    return a if which == 0 else b


def test_p12_nematic_uniform_state_recurrence(oracle):
    nx = ny = 8
    dt, A, C = 0.01, -1.0, 1.0
    s = oracle.System((nx, ny), (1.0, 1.0), dt, prec="f64", seed=5)
    ids = W.nematic(s, A=A, C=C, D=0.0)
    s.finalize()
    a, b = 0.3, -0.2
    s.set_field(ids["Qxx"], np.full((ny, nx), a))
    s.set_field(ids["Qxy"], np.full((ny, nx), b))
    for _ in range(50):
        s.step(1)
        m2 = a * a + b * b
        a, b = (a - dt * C * m2 * a) / (1 + dt * A), (b - dt * C * m2 * b) / (1 + dt * A)
        assert np.abs(s.get_field(ids["Qxx"]) - a).max() < 1e-13
        assert np.abs(s.get_field(ids["Qxy"]) - b).max() < 1e-13
    s.step(3000)
    assert np.abs(np.hypot(s.get_field(ids["Qxx"]), s.get_field(ids["Qxy"])) - 1.0).max() < 1e-6  # |Q| -> sqrt(-A/C)


# ------------------------------------------------------------------------------------------ P13
def test_p13_model_b_free_energy_and_phases(oracle):
    """noiseless Model B: Eq. 19 free energy never increases; late time: phases near +-1."""
    n, dx, dt = 32, 1.0, 0.05
    s = oracle.System((n, n), (dx, dx), dt, prec="f64", seed=1)
    ids = W.model_b(s, a=-1.0, b=1.0, k=1.0, D=0.0)
    s.finalize()
    phi = W.uniform_field(13, 0, (n, n), -0.1, 0.1)
    s.set_field(ids["phi"], phi)
    qx = 2 * np.pi * np.fft.rfftfreq(n, d=dx)
    qy = 2 * np.pi * np.fft.fftfreq(n, d=dx)
    q2 = qy[:, None] ** 2 + qx[None, :] ** 2

    def free_energy(p):
        ph = np.fft.rfft2(p)
        wgt = np.full(ph.shape, 2.0); wgt[:, 0] = 1.0; wgt[:, -1] = 1.0
        grad2 = (wgt * q2 * np.abs(ph) ** 2).sum() / p.size       # sum_x |grad phi|^2 (Parseval)
        return (-0.5 * p ** 2 + 0.25 * p ** 4).sum() + 0.5 * grad2

    mean0 = phi.mean()
    F = [free_energy(phi)]
    for _ in range(40):
        s.step(50)
        F.append(free_energy(s.get_field(ids["phi"])))
    assert all(F[i + 1] <= F[i] + 1e-9 * abs(F[i]) for i in range(len(F) - 1))
    p = s.get_field(ids["phi"])
    assert abs(p.mean() - mean0) < 1e-13
    assert 0.9 < np.percentile(p, 97) < 1.1 and -1.1 < np.percentile(p, 3) < -0.9


# ------------------------------------------------------------------------------------------ P14
@pytest.mark.parametrize("name,n", [("modelb_128", (16, 16)), ("kpz_4096", (16, 8)), ("nematic_1024", (8, 8))])
def test_p14_step_splitting_is_bit_identical(oracle, name, n):
    cfg = W.make_config(name, n=n)
    s1, ids = W.build(oracle, cfg, prec="f32")
    s2, _ = W.build(oracle, cfg, prec="f32")
    s1.step(5)
    s2.step(2); s2.step(3)
    assert s1.step_count == s2.step_count == 5
    for f in cfg["ic"]:
        a, b = s1.get_field_fourier_f64(ids[f]), s2.get_field_fourier_f64(ids[f])
        assert np.array_equal(a, b)
        assert np.all(np.isfinite(a))


# ------------------------------------------------------------------------------------------ error behaviour
def test_oracle_error_codes(oracle):
    with pytest.raises(oracle.OracleError) as e:
        oracle.System((12, 8), (1.0, 1.0), 0.1)
    assert e.value.code == oracle.EUNSUPPORTED
    s = oracle.System((8, 8), (1.0, 1.0), 0.1)
    f = s.add_field("phi", True)
    g = s.add_field("g", False)
    g2 = s.add_field("g2", False)
    with pytest.raises(oracle.OracleError) as e:
        s.add_linear(g, {"coef": 1.0})                 # implicit term on an aux field
    assert e.value.code == oracle.EINVAL
    with pytest.raises(oracle.OracleError):
        s.add_aux_def(g, {"coef": 1.0}, g2)            # aux used before defined
    with pytest.raises(oracle.OracleError):
        s.add_linear(f, {"coef": 1.0, "q2_pow": -1})   # negative power
    with pytest.raises(oracle.OracleError):
        s.add_linear(f, {"coef": 1.0, "iq_pow": (0, 0, 1)})   # z derivative in 2-D
    with pytest.raises(oracle.OracleError) as e:
        s.add_term(f, {"coef": 1.0}, [f] * 5)
    assert e.value.code == oracle.EUNSUPPORTED
    with pytest.raises(oracle.OracleError) as e:
        s.step(1)
    assert e.value.code == oracle.ESTATE
    s.add_aux_def(g, {"coef": 1.0}, f)
    s.add_aux_def(g2, {"coef": 1.0}, g)
    s.finalize()
    with pytest.raises(oracle.OracleError) as e:
        s.add_field("late", True)
    assert e.value.code == oracle.ESTATE


# ------------------------------------------------------------------------------------------ P15, P16
@pytest.mark.parametrize("n,dx", [((16,), (0.7,)), ((8, 16), (1.0, 0.5)), ((4, 8, 8), (1.0, 2.0, 0.5))])
def test_p15_intermediate_field_with_its_own_lhs(oracle, n, dx):
    """"psi + psi*q^2 = -q^2 phi"  <=>  psi_q = -q^2 (1 + q^2)^-1 phi_q, mode by mode.  The
    intermediate field is observed through an explicit linear term dt u = psi: u_q(1) - u_q(0) = dt psi_q.  Also an
    lhs that vanishes at q = 0 ("q^2 psi = phi", a Poisson solve): psi_0 = 0 (reading A10)."""
    dt = 0.25
    rng = np.random.default_rng(15)
    phi0 = rng.standard_normal(n[::-1])
    qs = []
    for j in range(len(n)):
        k = np.arange(n[j] // 2 + 1) if j == 0 else np.fft.fftfreq(n[j], 1.0 / n[j])
        qs.append(2 * np.pi * np.abs(k) / (n[j] * dx[j]))
    q2 = sum(g * g for g in np.meshgrid(*qs[::-1], indexing="ij"))
    for lhs, num, expect in (
            ([{"coef": 1.0}, {"coef": 1.0, "q2_pow": 1}], {"coef": -1.0, "q2_pow": 1}, lambda: -q2 / (1.0 + q2)),
            ([{"coef": 1.0, "q2_pow": 1}], {"coef": 1.0}, lambda: np.where(q2 > 0, 1.0 / np.where(q2 > 0, q2, 1.0), 0.0)),
            ([{"coef": 2.0}], {"coef": 3.0, "q2_pow": 2}, lambda: 1.5 * q2 * q2)):
        s = oracle.System(n, dx, dt, prec="f64", seed=3)
        phi = s.add_field("phi", True)
        u = s.add_field("u", True)
        psi = s.add_field("psi", False)
        for o in lhs:
            s.add_aux_lhs(psi, o)
        s.add_aux_def(psi, num, phi)
        s.add_term(u, {"coef": 1.0}, [psi])
        s.finalize()
        s.set_field(phi, phi0)
        s.set_field(u, np.zeros(n[::-1]))
        ph = s.get_field_fourier_f64(phi)
        s.step(1)
        got = s.get_field_fourier_f64(u) / dt
        want = expect() * ph
        assert np.abs(got - want).max() <= 1e-12 * max(1.0, np.abs(want).max())
        assert np.array_equal(s.get_field_fourier_f64(phi), ph)          # a field without an equation does not move


@pytest.mark.parametrize("n", [8, 16])
def test_p16_two_level_product_is_the_nested_direct_convolution(oracle, n):
    """an intermediate field that is itself a product, mu = phi*phi, used in dt u = -q^2 (mu*phi).
    Both products are quadratic, so every factor copy is truncated at |s(k)| < N/3; expected value:
    the two nested O(N^2) NON-wrapping convolutions of Eq. 5 written out with the masks, and with no mask the circular ones."""
    rng = np.random.default_rng(100 + n)
    phi0 = rng.standard_normal(n)
    full = np.fft.fft(phi0)
    dt = 0.5
    for dealias in (oracle.DEALIAS_OFF, oracle.DEALIAS_PAPER):
        s = oracle.System((n,), (1.0,), dt, prec="f64", seed=1)
        phi = s.add_field("phi", True)
        u = s.add_field("u", True)
        mu = s.add_field("mu", False)
        s.add_aux_term(mu, {"coef": 1.0}, [phi, phi])
        s.add_term(u, {"coef": -1.0, "q2_pow": 1}, [mu, phi])
        s.set_dealias(dealias)
        s.finalize()
        s.set_field(phi, phi0)
        s.set_field(u, np.zeros(n))
        s.step(1)
        got = s.get_field_fourier_f64(u) / dt
        keep = [k for k in range(n) if dealias == oracle.DEALIAS_OFF or 3 * abs(_signed(k, n)) < n]
        wrap = dealias == oracle.DEALIAS_OFF
        muh = np.zeros(n, dtype=complex)
        for q in range(n):
            for k in keep:
                for l in keep:
                    if (wrap and (k + l - q) % n == 0) or (not wrap and _signed(k, n) + _signed(l, n) == _signed(q, n)):
                        muh[q] += full[k] * full[l] / n
        if not wrap:   # sums outside (-N/2, N/2] do not exist without wrapping: |k + l| < 2N/3 can exceed N/2 -> they alias
            muh = np.zeros(n, dtype=complex)
            for k in keep:
                for l in keep:
                    muh[(k + l) % n] += full[k] * full[l] / n   # what the lattice really holds (aliased outside the kept band)
        for q in range(n // 2 + 1):
            if not wrap and 3 * abs(_signed(q, n)) >= n:
                continue
            acc = 0j
            for k in keep:      # mu is a factor of a quadratic product: its copy is truncated too
                for l in keep:
                    if (wrap and (k + l - q) % n == 0) or (not wrap and _signed(k, n) + _signed(l, n) == _signed(q, n)):
                        acc += muh[k] * full[l] / n
            q2 = (2 * np.pi * q / n) ** 2
            assert abs(got[q] - (-q2) * acc) <= 1e-11 * max(1.0, abs(acc)), (dealias, q)


# ------------------------------------------------------------------------------------------ P17
def test_p17_dirichlet_frame_reaches_the_linear_steady_state(oracle):
    """PAPER.md:233-255 and Fig. 2: heat diffusion dT/dt = d2T/dx2 between two baths on 256 sites, T(x,0) = 5.  With the
    baths applied in a frame of width 10 (T(x < 10) = 10, T(x >= 246) = 0, set at the end of every step) the numerical
    steady state is the analytical straight line between the baths; with the baths on single sites the periodic
    representation leaves the artifact the paper shows (the profile stays far from the line)."""
    n, dt, steps = 256, 2.0, 20000
    x = np.arange(n)
    err = {}
    for w in (1, 10):
        s = oracle.System((n,), (1.0,), dt, prec="f64", seed=1)
        s.set_threads(1)
        f = s.add_field("T", True)
        s.add_linear(f, {"coef": 1.0, "q2_pow": 1})
        s.set_frame(f, 0, w, 10.0, w, 0.0)
        s.finalize()
        s.set_field(f, np.full(n, 5.0))
        s.step(steps)
        T = s.get_field(f)
        assert np.all(np.abs(T[:w] - 10.0) < 1e-12) and np.all(np.abs(T[n - w:]) < 1e-12)
        lo, hi = w - 1, n - w
        line = 10.0 * (hi - x) / (hi - lo)                    # T1 + (T2 - T1) x / L between the baths
        sel = (x >= lo) & (x <= hi)
        err[w] = np.abs(T - line)[sel].max()
    assert err[10] < 0.01 * 10.0
    assert err[1] > 0.2 * 10.0


def test_p17_frame_semantics_2d(oracle):
    """the frame is applied after Eq. 18, per axis, in the order given; elsewhere the field is what the step made it"""
    n, dt = (16, 8), 0.1
    rng = np.random.default_rng(17)
    phi0 = rng.standard_normal(n[::-1])
    a = oracle.System(n, (1.0, 1.0), dt, prec="f64", seed=5)
    fa = a.add_field("phi", True)
    a.add_linear(fa, {"coef": 1.0, "q2_pow": 1})
    a.finalize()
    b = oracle.System(n, (1.0, 1.0), dt, prec="f64", seed=5)
    fb = b.add_field("phi", True)
    b.add_linear(fb, {"coef": 1.0, "q2_pow": 1})
    b.set_frame(fb, 0, 2, 1.5, 3, -2.0)
    b.set_frame(fb, 1, 1, 7.0, 0, 0.0)
    b.finalize()
    a.set_field(fa, phi0)
    b.set_field(fb, phi0)
    a.step(1)
    b.step(1)
    want = a.get_field(fa).copy()
    want[:, :2] = 1.5
    want[:, 13:] = -2.0
    want[:1, :] = 7.0
    assert np.abs(b.get_field(fb) - want).max() < 1e-13
