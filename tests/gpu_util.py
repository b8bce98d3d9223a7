"""Helpers of the GPU parity tests: build a plan from a synth config, run both sides."""
import numpy as np
import torch

import oracle
import synth
import paper_2507_08578_b200 as dft


def make_plan(cfg, options=None):
    plan = dft.Plan(cfg, options)
    if "vloc" in cfg:
        v = torch.as_tensor(cfg["vloc"], device="cuda")
        plan.set_vloc(v)
        torch.cuda.synchronize()
    return plan


def lib_spheres(plan):
    return [plan.get_kg(ik) for ik in range(plan.nkpt)]


def oracle_spheres(cfg):
    return [oracle.sphere(cfg["rprimd"], cfg["kpt"][ik], cfg["ecut"], cfg["ngfft"]) for ik in range(cfg["nkpt"])]


def assert_spheres_equal(lib_s, orc_s):
    for ik, ((kg, ig, kin), (okg, oig, okin)) in enumerate(zip(lib_s, orc_s)):
        assert len(ig) == len(oig), "k-point %d: npw %d != oracle %d" % (ik, len(ig), len(oig))
        assert np.array_equal(kg, okg), "kg differs at k-point %d" % ik
        assert np.array_equal(ig, oig), "igfft differs at k-point %d" % ik
        assert np.array_equal(kin.view(np.int64), okin.view(np.int64)), "kin not bit-equal at k-point %d" % ik


def gpu_apply(plan, psi_np):
    """psi_np [nkpt][nband][mpw] complex128 -> H psi as numpy, through dft_apply_h."""
    psi = torch.as_tensor(psi_np, device="cuda").contiguous()
    out = plan.apply_h(psi)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def oracle_apply(cfg, spheres, psi_np, terms=oracle.ALL, method=2, dij=None):
    out = np.zeros_like(psi_np)
    for ik, (kg, ig, kin) in enumerate(spheres):
        out[ik] = oracle.apply_h(cfg, ik, kg, ig, kin, psi_np[ik], method=method, terms=terms, dij=dij)
    return out


def band_rel_err(a, b):
    """max over k and bands of ||a-b||_2/||b||_2 (reading 17)."""
    a = a.reshape(-1, a.shape[-1]); b = b.reshape(-1, b.shape[-1])
    num = np.linalg.norm(a - b, axis=-1); den = np.linalg.norm(b, axis=-1)
    den = np.where(den == 0, 1.0, den)
    return float(np.max(num / den))


def nl_launches(plan, nband):
    """Launches of the non-local + kinetic part of one dft_apply_h: 1 where the one-launch kernel for tiny cells serves
    the call (csrc/nonlocal.cu: nproj <= 64 and nproj npw nband nkpt <= 1e6), else GEMM-1, D_ij, GEMM-2."""
    tiny = 0 < plan.nproj <= 64 and float(plan.nproj) * plan.mpw * nband * plan.nkpt <= 1e6
    return 1 if tiny else 3


def small_box_ok(plan):
    """True when the fused small-box kernel (fft_path = 3) can serve this plan; the plan's fft_path is left at 0."""
    try:
        plan.set_option("fft_path", 3)
    except dft.DftError as e:
        assert e.code == dft.DFT_ERR_UNSUPPORTED
        return False
    plan.set_option("fft_path", 0)
    return True
