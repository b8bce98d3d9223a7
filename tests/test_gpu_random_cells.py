"""Seeded random cells: triclinic lattices, random k-points (Gamma for the even seeds), cut-offs, atom positions, band
counts and FFT boxes between the tightest that holds the sphere and about three times that (box lengths with and without a two-radix
factorisation mixed).  Index maps bit-exact, H psi <= 1e-10 per band against the oracle on every code path that can
serve the cell (PAPER.md :456, Eq. 26 :470)."""
import numpy as np
import pytest
import torch

import oracle
import synth
from gpu_util import (make_plan, lib_spheres, oracle_spheres, assert_spheres_equal, gpu_apply, oracle_apply,
                      band_rel_err, small_box_ok)

pytestmark = pytest.mark.gpu
TOL = 1e-10
SMOOTH = [8, 9, 10, 12, 15, 16, 18, 20, 24, 25, 27, 30, 32, 36, 40, 45, 48, 50, 54, 60, 64]


def _random_cfg(seed):
    rng = np.random.default_rng(1000 + seed)
    rprimd = np.diag(rng.uniform(8.0, 13.0, 3)) + rng.uniform(-1.0, 1.0, (3, 3))
    nk = 2 if seed % 5 == 3 else 1
    kpt = np.zeros((nk, 3)) if seed % 2 == 0 else rng.uniform(-0.5, 0.5, (nk, 3))
    ecut = float(rng.uniform(1.5, 4.0) if seed < 10 else rng.uniform(4.0, 8.0))      # 50 .. 1200 plane waves
    xred = rng.uniform(0.0, 1.0, (7, 3))
    nband = int(rng.integers(1, 10))
    # extent of the sphere along each axis from the oracle's own enumeration in a box that surely holds it
    ext = np.zeros(3, int)
    for k in kpt:
        kg = oracle.sphere(rprimd, k, ecut, (64, 64, 64))[0]
        lo, hi = kg.min(axis=0), kg.max(axis=0)
        ext = np.maximum(ext, np.maximum(2 * hi + 1, -2 * lo))      # n must satisfy -(n/2) <= m <= (n-1)/2
    ngfft = []
    for c in range(3):
        fits = [n for n in SMOOTH if n >= ext[c]]
        ngfft.append(fits[int(rng.integers(0, 9))])                  # the tightest box or one of the next eight sizes
    cfg = synth.make_config("aniso5t", with_vloc=False, ecut=ecut, ngfft=tuple(ngfft), kpt=kpt, xred=xred, nband=nband)
    cfg["rprimd"] = np.ascontiguousarray(rprimd)
    cfg["vloc"] = synth.gen_vloc(cfg)
    return cfg


@pytest.mark.parametrize("seed", range(24))
def test_random_cell(seed):
    cfg = _random_cfg(seed)
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    assert_spheres_equal(sph, oracle_spheres(cfg))
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    ref = oracle_apply(cfg, sph, psi, method=1)
    gamma = plan.nkpt == 1 and not np.any(cfg["kpt"])
    paths = [0, 4, 1] + ([3] if small_box_ok(plan) else [])
    for path in paths:
        plan.set_option("fft_path", path)
        err = band_rel_err(gpu_apply(plan, psi), ref)
        assert err <= TOL, "seed %d box %s fft_path %d: %.3e" % (seed, cfg["ngfft"], path, err)
    plan.set_option("fft_path", 0)
    for key, val, back in (("gemm_3m", 0, 1), ("proj_mode", 1, 0)) + ((("gemm_sym", 1, 2),) if gamma else ()):
        plan.set_option(key, val)
        got = gpu_apply(plan, psi)
        err = band_rel_err(got, ref)
        assert err <= TOL, "seed %d %s = %d: %.3e" % (seed, key, val, err)
        for ik in range(plan.nkpt):
            assert np.all(got[ik][:, plan.npw[ik]:] == 0)
        plan.set_option(key, back)
    plan.destroy()


@pytest.mark.parametrize("seed", range(0, 12, 2))
def test_random_cell_gamma_storage(seed):
    """The even seeds are Gamma-point cells: the same random cell in real-symmetry storage (DESIGN.md
    reading 26) with the odd-parity couplings of D_ij removed, on the fused / five-pass / generic local paths, with and
    without the Strassen level (refused silently where nproj is not a multiple of 16)."""
    cfg = _random_cfg(seed)
    cfg["kpt"] = cfg["kpt"][:1]; cfg["nkpt"] = 1
    cfg["dij"] = synth.gamma_dij(cfg)
    plan = make_plan(cfg)
    kg, ig, kin = lib_spheres(plan)[0]
    plan.set_option("gamma_real", 1)
    hkin = plan.get_kg_gamma()[2]
    nb = cfg["nband"] + (cfg["nband"] & 1) + 2                    # even band counts >= 4, and one odd count below
    for nband in (nb, nb - 1):
        psi = synth.gen_psi(cfg, [hkin], nband=nband)[0]
        ref = oracle.apply_h_gamma(cfg, kg, ig, kin, psi, method=1)
        for path in (0, 4, 1):
            plan.set_option("fft_path", path)
            for strassen in (2, 1):
                plan.set_option("gemm_strassen", strassen)
                out = plan.apply_h_gamma(torch.as_tensor(psi, device="cuda").contiguous())
                torch.cuda.synchronize()
                got = out.cpu().numpy()
                err = band_rel_err(got, ref)
                assert err <= TOL, "seed %d nband %d fft_path %d strassen %d: %.3e" % (seed, nband, path, strassen, err)
                assert np.all(got[:, 0].imag == 0)
    plan.destroy()


@pytest.mark.parametrize("seed", range(1, 12, 2))
def test_random_cell_spinors(seed):
    """The odd seeds (general k-points): two-component spinors with a Hermitian 2 x 2 potential and a spin-dependent D
    (reading 27), fused 2 x 2 pass C where the box allows it, the Pauli form elsewhere (also on the generic kernels: box
    lengths without a two-radix factorisation)."""
    cfg = _random_cfg(seed)
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    v4, dspin = synth.spinor_inputs(cfg)
    plan.set_vloc_spinor(torch.as_tensor(v4, device="cuda"))
    plan.set_dij_spinor(dspin)
    nb = cfg["nband"]
    psi = synth.gen_psi(cfg, [s[2] for s in sph], nband=2 * nb).reshape(plan.nkpt, nb, 2, plan.mpw)
    ref = np.stack([oracle.apply_h_spinor(cfg, ik, *sph[ik], psi[ik], v4, dspin, method=1) for ik in range(plan.nkpt)])
    for path in (0, 4, 1):
        plan.set_option("fft_path", path)
        for fused in (1, 0):
            plan.set_option("spinor_fused", fused)
            out = plan.apply_h_spinor(torch.as_tensor(psi, device="cuda").contiguous())
            torch.cuda.synchronize()
            err = band_rel_err(out.cpu().numpy(), ref)
            assert err <= TOL, "seed %d fft_path %d spinor_fused %d: %.3e" % (seed, path, fused, err)
    plan.destroy()
