"""dft_apply_vloc_noalloc (include/dft.h): the local term with its pass-to-pass scratch in a static device array inside the
library, for callers that cannot call cudaMalloc.  Checked against the existing path (dft_apply_h with terms = 2) on two calls
in a row.  This file is named to be collected last: the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

import paper_2507_08578_b200 as dft
import synth
from gpu_util import make_plan, lib_spheres

pytestmark = pytest.mark.gpu
TOL = 1e-10     # the per-band relative tolerance of every other parity test (north_star)


def _band_rel_err(got, ref):
    num = torch.linalg.vector_norm(got - ref, dim=-1)
    den = torch.linalg.vector_norm(ref, dim=-1)
    return float((num / den).max())


@pytest.mark.parametrize("name,nband", [("c1", 40), ("c3k2", 7), ("c1m", 6)])
def test_no_alloc_local_term_matches_existing_path_twice(name, nband):
    """c1 (72^3, 4.15 MB of scratch per band): 40 bands need three chunks of the 64 MiB array; c3k2: two k-points; c1m: a
    box where dft_apply_h itself takes the fused small-box kernel (a different kernel family: agreement to rounding)."""
    cfg = synth.make_config(name)
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    kins = [s[2] for s in sph]
    if name == "c1":
        assert plan.workspace_bytes_per_band * nband > 2 * dft.DFT_NOALLOC_SCRATCH_BYTES      # really more than one chunk
    psi1 = synth.gen_psi_torch(cfg, kins, "cuda", nband=nband)
    psi2 = synth.gen_psi_torch(dict(cfg, seed=cfg["seed"] + 77), kins, "cuda", nband=nband)
    plan.set_option("terms", 2)
    ref1 = plan.apply_h(psi1).clone()
    ref2 = plan.apply_h(psi2).clone()
    plan.set_option("terms", 15)
    out = torch.full_like(psi1, float("nan"))
    plan.apply_vloc_noalloc(psi1, out)            # first call: sets up the array's address for this device
    torch.cuda.synchronize()
    err1 = _band_rel_err(out, ref1)
    free_before = torch.cuda.mem_get_info()[0]
    plan.apply_vloc_noalloc(psi2, out)            # second call: same array, still holding the first call's data
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    err2 = _band_rel_err(out, ref2)
    assert err1 <= TOL and err2 <= TOL, "%s: %.3e / %.3e" % (name, err1, err2)
    for ik in range(plan.nkpt):                   # pad entries are written as 0, as by dft_apply_h
        assert bool((out[ik][:, int(plan.npw[ik]):] == 0).all())
    assert free_after >= free_before, "device memory in use grew across a call: free %d -> %d" % (free_before, free_after)
    plan.destroy()


def test_no_alloc_refuses_what_does_not_fit_and_unset_potential():
    """One band of a 256 x 256 x 80 box with 73 occupied planes needs more than the 64 MiB array: DFT_ERR_ALLOC with the
    sizes in the message; before dft_set_vloc: DFT_ERR_NOT_READY."""
    cfg = synth.make_config("c0", with_vloc=False, ecut=500.0, ngfft=(256, 256, 80), nband=1)
    plan = make_plan(cfg)
    assert plan.workspace_bytes_per_band > dft.DFT_NOALLOC_SCRATCH_BYTES
    psi = torch.zeros((1, 1, plan.mpw), dtype=torch.complex128, device="cuda")
    out = torch.empty_like(psi)
    with pytest.raises(dft.DftError) as e:
        plan.apply_vloc_noalloc(psi, out)
    assert e.value.code == dft.DFT_ERR_NOT_READY
    plan.set_vloc(torch.zeros((80, 256, 256), dtype=torch.float64, device="cuda"))
    with pytest.raises(dft.DftError) as e:
        plan.apply_vloc_noalloc(psi, out)
    assert e.value.code == dft.DFT_ERR_ALLOC and "static array" in str(e.value)
    plan.destroy()
