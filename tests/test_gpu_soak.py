"""Soak test of the persistent 1024^2 kernel's relaxed barrier arrivals (pss_persist2d.cuh, grid_arrive_relaxed).

A group that only READ its exchange block reports that with a relaxed reduction; the producers overwrite the block
after they have seen the count.  The PTX memory model does not order that write after the read; the hardware argument
(cp.async.wait_all has retired the reads) is in the kernel's source.  A violation would be a torn exchange block, i.e.
wrong field values: 10^6 consecutive time steps (2 10^6 exchanges on every one of 129 CTAs) are compared bit for bit,
at four points, with the first-generation kernel f2d::k_fused2d (PSS_PERSIST=0), which computes the same arithmetic
behind release/acquire barriers only."""
import os

import numpy as np
import pytest

from paper_2405_02410_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def test_a_million_steps_bit_identical_to_the_release_acquire_kernel():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2405_02410_b200 as pss
    cfg = wl.make_config("modelb_1024")
    fast, ids = wl.build(pss, cfg, prec="f32")
    os.environ["PSS_PERSIST"] = "0"
    try:
        safe, _ = wl.build(pss, cfg, prec="f32")
    finally:
        del os.environ["PSS_PERSIST"]
    assert fast.fused_kernel_name == "k_persist2d" and safe.fused_kernel_name == "k_fused2d"
    phi = ids["phi"]
    for _ in range(4):
        fast.step(250000)
        safe.step(250000)
        a = fast.get_field_fourier(phi)
        b = safe.get_field_fourier(phi)
        assert np.isfinite(a.view(np.float32)).all()
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32)), fast.step_count
    assert fast.step_count == 10 ** 6
    x = fast.get_field(phi)
    assert float(np.abs(x).max()) < 2.0 and abs(float(x.mean()) - 0.1) < 1e-3     # coarsened, mass conserved
