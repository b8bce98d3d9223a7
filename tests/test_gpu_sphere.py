"""K1 parity: the G-sphere index maps must be BIT-EXACT against the oracle (BASELINE.json north_star;
DESIGN.md readings 1-3): npw, kg, igfft equal as integers, kin equal bit for bit."""
import numpy as np
import pytest

import oracle
import synth
from util import config
from gpu_util import make_plan, lib_spheres, oracle_spheres, assert_spheres_equal

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["c0", "c1", "c2", "c3", "c4", "c1m", "c2m", "c4m", "aniso", "c3k2"])
def test_sphere_bitexact(name):
    cfg = synth.make_config(name, with_vloc=False)
    cfg = dict(cfg, natom=0, typat=np.zeros(0, np.int32), xred=np.zeros((0, 3)), types=[], dij=None)  # sphere only
    plan = make_plan(cfg)
    assert_spheres_equal(lib_spheres(plan), oracle_spheres(cfg))
    plan.destroy()


def test_sphere_random_triclinic():
    r = np.random.default_rng(7)
    for trial in range(6):
        A = np.diag(r.uniform(6, 12, 3)) + r.uniform(-1.5, 1.5, (3, 3))
        k = r.uniform(-0.5, 0.5, 3)
        ecut = float(r.uniform(1.0, 4.0))
        n = (30, 36, 40)
        fits, _, _ = oracle.sphere_extent(A, k, ecut, n)
        if not fits:
            continue
        cfg = dict(rprimd=A, kpt=k.reshape(1, 3), nkpt=1, ecut=ecut, ngfft=n, typat=np.zeros(0, np.int32),
                   xred=np.zeros((0, 3)), types=[], dij=None)
        plan = make_plan(cfg)
        assert_spheres_equal(lib_spheres(plan), oracle_spheres(cfg))
        plan.destroy()


def test_inclusive_boundary():
    """ecut := kin(m*) as computed by the rule: m* and -m* must be inside (<=, not <)."""
    cfg = synth.make_config("c0", with_vloc=False)
    e = oracle.kin_of(cfg["rprimd"], cfg["kpt"][0], (2, -1, 1))
    cfg2 = dict(cfg, ecut=e, natom=0, typat=np.zeros(0, np.int32), xred=np.zeros((0, 3)), types=[], dij=None)
    plan = make_plan(cfg2)
    kg, ig, kin = plan.get_kg(0)
    rows = {tuple(v) for v in kg}
    assert (2, -1, 1) in rows and (-2, 1, -1) in rows
    assert kin.max() == e
    assert_spheres_equal(lib_spheres(plan), oracle_spheres(cfg2))
    plan.destroy()


def test_grid_too_small_and_errors():
    import paper_2507_08578_b200 as dft
    cfg = synth.make_config("c0", with_vloc=False)
    with pytest.raises(dft.DftError) as ei:
        dft.Plan(dict(cfg, ngfft=(8, 8, 8)))
    assert ei.value.code == dft.DFT_ERR_GRID_TOO_SMALL
    with pytest.raises(dft.DftError) as ei:
        dft.Plan(dict(cfg, ngfft=(22, 20, 20)))           # 22 = 2*11
    assert ei.value.code == dft.DFT_ERR_UNSUPPORTED
    with pytest.raises(dft.DftError) as ei:
        dft.Plan(dict(cfg, ecut=60.0, ngfft=(60, 60, 60)))   # radial tables were made for ecut 8
    assert ei.value.code == dft.DFT_ERR_TABLE_RANGE
    plan = dft.Plan(cfg)
    import torch
    psi = torch.zeros((1, 2, plan.mpw), dtype=torch.complex128, device="cuda")
    with pytest.raises(dft.DftError) as ei:
        plan.apply_h(psi)
    assert ei.value.code == dft.DFT_ERR_NOT_READY
    with pytest.raises(dft.DftError) as ei:
        plan.set_option("no_such_option", 1)
    assert ei.value.code == dft.DFT_ERR_INVALID_ARG
    plan.destroy()
