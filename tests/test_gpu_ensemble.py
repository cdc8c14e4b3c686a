"""Ensembles: R independent realisations of one field system stepped in the same launches.
Replica r must equal, bit for bit, the single system created with seed + r, and match the oracle run with that seed."""
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
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


CASES = [("modelb_128", (64, 64)), ("modelb_128", (128,)), ("kpz_4096", (32, 64)), ("modelb_256c", (16, 16, 32)),
         ("nematic_1024", (32, 32)), ("modelb_1024", (1024, 1024))]


@pytest.mark.parametrize("name,n", CASES)
def test_replicas_equal_single_systems_and_oracle(pss, oracle, name, n):
    R, steps = 3, 6
    cfg = wl.make_config(name, n=n)
    dyn_names = list(cfg["ic"].keys())
    ens, ids = wl.build(pss, cfg, prec="f32", set_ic=False, replicas=R)
    assert ens.replicas == R
    if n == (1024, 1024):   # the one-launch-per-replica path of the persistent kernel (seed + r, counters cleared per launch)
        assert ens.fused_kernel_name == "k_persist2d"
    for r in range(R):
        cr = dict(cfg, seed=cfg["seed"] + r)
        ens.select_replica(r)
        for nm, arr in wl.initial_conditions(cr, np.float32).items():
            ens.set_field(ids[nm], arr)
    ens.step(2)
    ens.step(steps - 2)
    assert ens.step_count == steps
    for r in range(R):
        cr = dict(cfg, seed=cfg["seed"] + r)
        one, _ = wl.build(pss, cr, prec="f32")
        assert one.fused_kernel_name == ens.fused_kernel_name
        one.step(steps)
        o, _ = wl.build(oracle, cr, prec="f32")
        o.step(steps)
        ens.select_replica(r)
        bg, _ = ens.debug_noise(ids[dyn_names[0]], 4)
        bo, _ = o.debug_noise(ids[dyn_names[0]], 4)
        assert np.array_equal(bg, bo)
        for nm in dyn_names:
            a = ens.get_field(ids[nm])
            if True:
                assert np.array_equal(a.view(np.uint32), one.get_field(ids[nm]).view(np.uint32)), (name, r, nm)
            assert rel_l2(a, o.get_field(ids[nm])) <= 1e-5, (name, r, nm)
    # replicas are different realisations
    ens.select_replica(0)
    a0 = ens.get_field(ids[dyn_names[0]])
    ens.select_replica(1)
    assert not np.array_equal(a0, ens.get_field(ids[dyn_names[0]]))


def test_replica_api_errors(pss):
    b = pss.binding
    s = pss.System((64, 64), (1.0, 1.0), 0.01)
    with pytest.raises(b.PssError) as e:
        s.set_replicas(0)
    assert e.value.code == b.EINVAL
    s.set_replicas(4)
    with pytest.raises(b.PssError) as e:
        s.select_replica(4)
    assert e.value.code == b.EINVAL
    f = s.add_field("phi", True)
    s.add_linear(f, {"coef": 1.0, "q2_pow": 1})
    s.finalize()
    with pytest.raises(b.PssError) as e:
        s.set_replicas(2)
    assert e.value.code == b.ESTATE
    s.select_replica(3)
