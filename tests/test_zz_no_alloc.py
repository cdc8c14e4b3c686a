"""pss_debug_noise_noalloc: the entry point for callers that cannot allocate device memory.

Who they are: this library normally lives inside a PyTorch process.  There the caching allocator may already own almost
all of the GPU, so the cudaMalloc that pss_debug_noise issues can fail although memory "is free"; its cudaFree waits for
the whole device, which a monitoring thread of a running simulation must not cause; and while some other thread records
a CUDA graph in the global capture mode, cudaMalloc is forbidden outright.  pss_debug_noise_noalloc runs the same kernel
but parks its results in a fixed 16 MiB device array that belongs to libpss.so (capacity STATIC_NOISE_MAX_MODES modes,
one array per GPU, shared by all calls).

What is checked: on two calls in a row (different steps, so the second call finds the first call's values in the
array) the words and the Gaussian z equal those of pss_debug_noise.  Both paths run the same kernel, so the tolerance
the other noise tests use for z is met with zero difference and the words are compared bit for bit.  A lattice beyond the
capacity is refused with ETOOBIG before anything is launched.

The file sorts last on purpose (pytest -x stops at the first failure; one here must not hide the rest), needs nothing from
the tests before it and leaves nothing behind for a later run."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _model_b(pss, n, prec):
    s = pss.System(n, (1.0,) * len(n), dt=0.01, prec=prec, seed=20240502)
    phi = s.add_field("phi", True)
    s.add_linear(phi, {"coef": -1.0, "q2_pow": 1})
    s.add_linear(phi, {"coef": 1.0, "q2_pow": 2})
    s.add_term(phi, {"coef": -1.0, "q2_pow": 1}, [phi, phi, phi])
    s.set_noise(phi, 0.05, 2)
    s.finalize()
    return s, phi


@pytest.mark.parametrize("n,prec", [((128, 128), "f32"), ((64, 32, 16), "f64"), ((1024, 1024), "f32")])
def test_noalloc_noise_equals_the_allocating_path_on_two_calls_in_a_row(n, prec):
    import paper_2405_02410_b200 as pss
    s, phi = _model_b(pss, n, prec)
    assert int(np.prod(s.hshape)) <= pss.binding.STATIC_NOISE_MAX_MODES
    for step in (3, 4):                                   # two calls in a row through the shared array
        bits_s, z_s = s.debug_noise_noalloc(phi, step)
        bits_a, z_a = s.debug_noise(phi, step)
        assert np.array_equal(bits_s, bits_a), "Philox words differ at step %d" % step
        assert np.isfinite(z_s.view(s.rdtype)).all()
        assert np.max(np.abs(z_s - z_a)) == 0.0, "z differs at step %d" % step
    first, _ = s.debug_noise_noalloc(phi, 3)              # the array was overwritten in between: step 3 again
    again, _ = s.debug_noise(phi, 3)
    assert np.array_equal(first, again)
    assert not np.array_equal(first, bits_s)              # and steps 3 and 4 really are different draws


def test_noalloc_noise_refuses_a_lattice_beyond_the_fixed_array():
    import paper_2405_02410_b200 as pss
    s, phi = _model_b(pss, (2048, 1024), "f32")           # 1025 x 1024 modes > 1024 x 513
    before = s.launch_count
    with pytest.raises(pss.binding.PssError) as e:
        s.debug_noise_noalloc(phi, 0)
    assert e.value.code == pss.binding.ETOOBIG
    assert "PSS_STATIC_NOISE_MAX_MODES" in str(e.value)
    assert s.launch_count == before                       # nothing was launched
    s.debug_noise(phi, 0)                                 # the handle is still usable
