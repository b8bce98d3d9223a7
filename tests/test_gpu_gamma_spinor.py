"""Parity of the NEXT-row-4 CUDA paths with their oracle restatements: Gamma-point real-symmetry
storage (dft_apply_h_gamma: band pairs packed into one complex FFT, real projector GEMMs on the half sphere) and
two-component spinors (dft_apply_h_spinor).  Same bar as the scalar path: <= 1e-10 relative per band."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2507_08578_b200 as dft
from gpu_util import make_plan, lib_spheres, oracle_spheres, assert_spheres_equal, band_rel_err

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _gamma_setup(name, **over):
    cfg = synth.make_config(name, **over)
    cfg["dij"] = synth.gamma_dij(cfg)             # time-reversal-compatible D (reading 26)
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    assert_spheres_equal(sph, oracle_spheres(cfg))
    plan.set_option("gamma_real", 1)
    kg, ig, kin = sph[0]
    ih, ineg = oracle.gamma_half(kg)
    hkg, hig, hkin = plan.get_kg_gamma()
    assert len(hig) == (len(ig) + 1) // 2 == len(ih)
    assert np.array_equal(hkg, kg[ih]) and np.array_equal(hig, ig[ih])
    assert np.array_equal(hkin.view(np.int64), kin[ih].view(np.int64))
    return cfg, plan, (kg, ig, kin), hkin


def _gamma_gpu(plan, psi_np):
    out = plan.apply_h_gamma(torch.as_tensor(psi_np, device="cuda").contiguous())
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("name", ["c0", "c2m", "c4m"])
def test_gamma_small_cells_all_terms_and_paths(name):
    cfg, plan, (kg, ig, kin), hkin = _gamma_setup(name)
    psi = synth.gen_psi(cfg, [hkin])[0]                     # [nband][nhalf]; Im psi(0) != 0 on purpose: it must be ignored
    assert np.all(psi[:, 0].imag != 0)
    m = 1 if name == "c0" else 2
    for terms in (7, 1, 2, 4, 3, 6):
        plan.set_option("terms", terms)
        ref = oracle.apply_h_gamma(cfg, kg, ig, kin, psi, method=m, terms=terms)
        for path in (0, 4, 1):                              # fused small-box kernel, five-pass register path, generic path
            plan.set_option("fft_path", path)
            got = _gamma_gpu(plan, psi)
            err = band_rel_err(got, ref)
            assert err <= TOL, "%s terms=%d fft_path=%d: rel err %.3e" % (name, terms, path, err)
            assert np.all(got[:, 0].imag == 0)
    plan.destroy()


def test_gamma_and_symmetric_table_on_a_triclinic_cell_with_two_types():
    """aniso at k = 0: triclinic lattice, anisotropic box, an l = 2 type with 9 projectors next to the 8-projector type.
    Both k = 0 formulations (Gamma storage; real symmetric-table GEMMs for general complex bands) against the oracle."""
    cfg, plan, (kg, ig, kin), hkin = _gamma_setup("aniso", kpt=[[0.0, 0.0, 0.0]])
    psi = synth.gen_psi(cfg, [hkin])[0]
    ref = oracle.apply_h_gamma(cfg, kg, ig, kin, psi, method=1)
    assert band_rel_err(_gamma_gpu(plan, psi), ref) <= TOL
    plan.destroy()
    cfg = synth.make_config("aniso", kpt=[[0.0, 0.0, 0.0]])      # the recipe's dense D (couples l = 0, 1, 2): fine for complex bands
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    full = synth.gen_psi(cfg, [sph[0][2]])
    fref = oracle.apply_h(cfg, 0, *sph[0], full[0], method=1)
    for sym in (1, 0):
        plan.set_option("gemm_sym", sym)
        got = plan.apply_h(torch.as_tensor(full, device="cuda")).cpu().numpy()
        assert band_rel_err(got, fref[None]) <= TOL, sym
    plan.destroy()


@pytest.mark.parametrize("nband", [1, 3, 64, 65])
def test_gamma_band_counts(nband):
    """Odd band counts leave the last pair half empty; 65 bands = two GEMM band tiles."""
    cfg, plan, (kg, ig, kin), hkin = _gamma_setup("c2m")
    psi = synth.gen_psi(cfg, [hkin], nband=nband)[0]
    ref = oracle.apply_h_gamma(cfg, kg, ig, kin, psi)
    for path in (0, 4):
        plan.set_option("fft_path", path)
        err = band_rel_err(_gamma_gpu(plan, psi), ref)
        assert err <= TOL, "nband=%d path=%d: %.3e" % (nband, path, err)
    plan.destroy()


def test_gamma_matches_the_full_sphere_path_on_symmetric_input():
    """Same operator, two storages: dft_apply_h on the expanded symmetric vectors, restricted, equals dft_apply_h_gamma."""
    cfg, plan, (kg, ig, kin), hkin = _gamma_setup("c4m")
    ih, _ = oracle.gamma_half(kg)
    psi = synth.gen_psi(cfg, [hkin])[0]
    full = oracle.gamma_expand(kg, psi)
    out_full = plan.apply_h(torch.as_tensor(full[None], device="cuda")).cpu().numpy()[0]
    got = _gamma_gpu(plan, psi)
    assert band_rel_err(got[:, 1:], out_full[:, ih][:, 1:]) <= 1e-12
    plan.destroy()


@pytest.mark.parametrize("name", ["c0", "c2m"])
def test_gamma_chebyshev_filter(name):
    """dft_chebyshev_filter_gamma against the oracle's recurrence in Gamma storage (degrees 0, 1, 4, 7)."""
    cfg, plan, (kg, ig, kin), hkin = _gamma_setup(name)
    psi = synth.gen_psi(cfg, [hkin])[0]
    cen, e = 0.5 * float(kin.max()) + 1.0, 0.5 * float(kin.max()) + 0.5
    for deg in (0, 1, 4, 7):
        t = torch.as_tensor(psi, device="cuda").clone()
        got = plan.chebyshev_filter_gamma(t, deg, cen, e).cpu().numpy()
        ref = oracle.chebyshev_filter_gamma(cfg, kg, ig, kin, psi, deg, cen, e, method=1 if name == "c0" else 2)
        err = band_rel_err(got, ref)
        assert err <= TOL, "%s deg=%d: %.3e" % (name, deg, err)
    plan.destroy()


@pytest.mark.parametrize("name,nband", [("c4m", 8), ("c2m", 6), ("c4m", 66)])
def test_gamma_storage_with_the_strassen_level(name, nband):
    """gemm_strassen = 1 in Gamma storage (even band counts; odd ones keep the plain real GEMMs): H psi with term
    isolations and the Chebyshev recurrence against the oracle."""
    cfg, plan, (kg, ig, kin), hkin = _gamma_setup(name, nband=nband)
    plan.set_option("gemm_strassen", 1)
    psi = synth.gen_psi(cfg, [hkin], nband=nband)[0]
    for terms in (7, 4, 5):
        plan.set_option("terms", terms)
        ref = oracle.apply_h_gamma(cfg, kg, ig, kin, psi, terms=terms)
        got = _gamma_gpu(plan, psi)
        assert band_rel_err(got, ref) <= TOL, "%s terms=%d" % (name, terms)
        assert np.all(got[:, 0].imag == 0)
    plan.set_option("terms", 7)
    assert plan.last_launches() > 20                          # fourteen products + combinations: the Strassen path ran
    cen, e = 0.5 * float(kin.max()) + 1.0, 0.5 * float(kin.max()) + 0.5
    t = torch.as_tensor(psi, device="cuda").clone()
    got = plan.chebyshev_filter_gamma(t, 3, cen, e).cpu().numpy()
    assert band_rel_err(got, oracle.chebyshev_filter_gamma(cfg, kg, ig, kin, psi, 3, cen, e)) <= TOL
    odd = synth.gen_psi(cfg, [hkin], nband=nband - 1)[0]       # odd count: falls back to the plain real GEMMs
    assert band_rel_err(_gamma_gpu(plan, odd), oracle.apply_h_gamma(cfg, kg, ig, kin, odd)) <= TOL
    plan.destroy()


def test_gamma_refusals():
    cfg = synth.make_config("c0")                            # the recipe's dense D couples s and p projectors
    plan = make_plan(cfg)
    with pytest.raises(dft.DftError) as e:
        plan.set_option("gamma_real", 1)
    assert e.value.code == dft.DFT_ERR_INVALID_ARG
    with pytest.raises(dft.DftError) as e:                   # not enabled
        plan.apply_h_gamma(torch.zeros((1, 142), dtype=torch.complex128, device="cuda"))
    assert e.value.code == dft.DFT_ERR_NOT_READY
    dft.dft_set_dij(plan.h, synth.gamma_dij(cfg))
    plan.set_option("gamma_real", 1)
    with pytest.raises(dft.DftError) as e:                   # a later D_ij that breaks time reversal
        dft.dft_set_dij(plan.h, cfg["dij"])
    assert e.value.code == dft.DFT_ERR_INVALID_ARG
    plan.set_vector_potential([0.1, 0.0, -0.2])               # A != 0 breaks time reversal: refused, not ignored
    with pytest.raises(dft.DftError) as e:
        plan.apply_h_gamma(torch.zeros((1, 142), dtype=torch.complex128, device="cuda"))
    assert e.value.code == dft.DFT_ERR_UNSUPPORTED
    plan.set_vector_potential(None)
    plan.apply_h_gamma(torch.zeros((1, 142), dtype=torch.complex128, device="cuda"))
    plan.set_option("gamma_real", 0)
    plan.destroy()
    cfg = synth.make_config("c1m")                           # k = (1/4, 1/4, 1/4)
    cfg["dij"] = synth.gamma_dij(cfg)
    plan = make_plan(cfg)
    with pytest.raises(dft.DftError) as e:
        plan.set_option("gamma_real", 1)
    assert e.value.code == dft.DFT_ERR_UNSUPPORTED
    plan.destroy()


def _gamma_full_size(name, per_tile):
    """Full-size Gamma-storage run (all bands on the GPU); the oracle checks a seeded sample that hits every 64-band
    GEMM tile (first, last and seeded interior bands), both members of packed pairs included."""
    cfg, plan, (kg, ig, kin), hkin = _gamma_setup(name)
    nband = cfg["nband"]
    rng = np.random.default_rng(11)
    sample = set()
    for t0 in range(0, nband, 64):
        t1 = min(nband, t0 + 64)
        sample.update((t0, t1 - 1))
        sample.update(int(v) for v in rng.choice(np.arange(t0 + 1, t1 - 1), size=min(per_tile - 2, t1 - t0 - 2), replace=False))
    sample = sorted(sample)
    psi = synth.gen_psi_torch(cfg, [hkin], "cuda")[0]
    out = plan.apply_h_gamma(psi)
    torch.cuda.synchronize()
    ref = oracle.apply_h_gamma(cfg, kg, ig, kin, psi[sample].cpu().numpy())
    err = band_rel_err(out[sample].cpu().numpy(), ref)
    print("%s Gamma storage: nhalf %d, %d of %d bands oracle-checked (all %d GEMM band tiles): rel err %.2e"
          % (name, len(hkin), len(sample), nband, (nband + 63) // 64, err))
    assert err <= TOL, err
    plan.destroy()
    del psi, out
    torch.cuda.empty_cache()


def test_gamma_c2_full_size_sample():
    _gamma_full_size("c2", 10)       # 7 tiles x up to 10 = 66 of 432 bands, nhalf 62 145


def test_gamma_c4_full_size_sample():
    _gamma_full_size("c4", 4)        # 16 tiles x 4 = 64 of 1024 bands, nhalf 147 834


# ------------------------------------------------------------------------------------------------ spinors
def _spinor_gpu(plan, psi_np):
    out = plan.apply_h_spinor(torch.as_tensor(psi_np, device="cuda").contiguous())
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("name", ["c0", "c1m", "aniso", "c3k2"])
def test_spinor_all_terms_and_paths(name):
    cfg = synth.make_config(name)
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    assert_spheres_equal(sph, oracle_spheres(cfg))
    v4, dspin = synth.spinor_inputs(cfg)
    plan.set_vloc_spinor(torch.as_tensor(v4, device="cuda"))
    plan.set_dij_spinor(dspin)
    nb, mpw = cfg["nband"], plan.mpw
    base = synth.gen_psi(cfg, [s[2] for s in sph], nband=2 * nb)           # [nkpt][2 nb][mpw]: rows 2b + s
    psi = base.reshape(plan.nkpt, nb, 2, mpw)
    m = 1 if name in ("c0", "aniso") else 2
    for terms in (7, 1, 2, 4):
        plan.set_option("terms", terms)
        ref = np.stack([oracle.apply_h_spinor(cfg, ik, *sph[ik], psi[ik], v4, dspin, method=m, terms=terms)
                        for ik in range(plan.nkpt)])
        for path in (0, 4) if terms in (7, 2) else (0,):
            plan.set_option("fft_path", path)
            got = _spinor_gpu(plan, psi)
            err = band_rel_err(got, ref)
            assert err <= TOL, "%s terms=%d path=%d: rel err %.3e" % (name, terms, path, err)
            for ik in range(plan.nkpt):
                assert np.all(got[ik][:, :, plan.npw[ik]:] == 0)
    # back to the scalar D_ij on both components (dspin = NULL), spin-diagonal potential: two scalar applications
    plan.set_option("terms", 7); plan.set_option("fft_path", 0)
    plan.set_dij_spinor(None)
    vd = np.stack([cfg["vloc"], cfg["vloc"], np.zeros_like(cfg["vloc"]), np.zeros_like(cfg["vloc"])])
    plan.set_vloc_spinor(torch.as_tensor(vd, device="cuda"))
    got = _spinor_gpu(plan, psi)
    ref = plan.apply_h(torch.as_tensor(base, device="cuda")).cpu().numpy().reshape(got.shape)
    assert band_rel_err(got, ref) <= 1e-12
    plan.destroy()


@pytest.mark.parametrize("name,over", [("c1m", {}), ("aniso", {}), ("c3k2", {}), ("c0", {"ngfft": (20, 20, 180)}), ("c0", {"ngfft": (16, 20, 24)})],
                         ids=lambda v: v if isinstance(v, str) else "x".join(map(str, v.get("ngfft", ()))))
def test_spinor_local_term_fused_in_pass_c(name, over):
    """Five-pass register path: ONE local application with the 2 x 2 potential multiplied in pass C (the two components of a
    point in partner lanes of a warp; option spinor_fused = 1, default) against the four scalar applications of the Pauli
    decomposition (spinor_fused = 0) and the oracle; band chunks are rounded to whole spinor bands; a quarter of the
    launches."""
    cfg = synth.make_config(name, **over)
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    v4, dspin = synth.spinor_inputs(cfg)
    plan.set_vloc_spinor(torch.as_tensor(v4, device="cuda"))
    plan.set_dij_spinor(dspin)
    nb, mpw = 5, plan.mpw
    psi = synth.gen_psi(cfg, [s[2] for s in sph], nband=2 * nb).reshape(plan.nkpt, nb, 2, mpw)
    m = 1 if name in ("c0", "aniso") else 2
    plan.set_option("fft_path", 4)
    for terms in (2, 7):
        plan.set_option("terms", terms)
        ref = np.stack([oracle.apply_h_spinor(cfg, ik, *sph[ik], psi[ik], v4, dspin, method=m, terms=terms)
                        for ik in range(plan.nkpt)])
        for fused in (1, 0):
            plan.set_option("spinor_fused", fused)
            for chunk in (0, 2, 3, 7):
                plan.set_option("band_chunk", chunk)
                got = _spinor_gpu(plan, psi)
                err = band_rel_err(got, ref)
                assert err <= TOL, "%s terms=%d fused=%d chunk=%d: rel err %.3e" % (name, terms, fused, chunk, err)
                for ik in range(plan.nkpt):
                    assert np.all(got[ik][:, :, plan.npw[ik]:] == 0)
                if terms == 2 and chunk == 0:
                    assert plan.last_launches() == (5 * plan.nkpt if fused else 20 * plan.nkpt + 3)
    plan.destroy()


def test_spinor_c4_full_size_local_term_sample():
    """Full-size c4 box (180^3, radix pair 12 x 15, 295 667 plane waves): 160 spinor bands = 320 rows through the fused
    2 x 2 pass C in band chunks of whole spinor bands; the oracle checks the local term of a sample that sits on both sides
    of every chunk boundary (the non-local part of this cell is covered row by row by the scalar full-size test: the GEMMs
    see the same rows)."""
    cfg = synth.make_config("c4")
    plan = make_plan(cfg)
    (kg, ig, kin), = lib_spheres(plan)
    v4, dspin = synth.spinor_inputs(cfg)
    plan.set_vloc_spinor(torch.as_tensor(v4, device="cuda"))
    nsb = 160
    psi = synth.gen_psi_torch(cfg, [kin], "cuda", nband=2 * nsb)[0].reshape(1, nsb, 2, plan.mpw)
    plan.set_option("terms", 2)
    out = plan.apply_h_spinor(psi)
    torch.cuda.synchronize()
    assert plan.last_launches() % 5 == 0 and plan.last_launches() >= 10        # five passes per chunk, several chunks
    chunk = 2 * nsb // (plan.last_launches() // 5)                              # rows per chunk, roughly
    sample = sorted({0, nsb - 1, chunk // 2 - 1, chunk // 2, chunk // 2 + 1, nsb // 2})
    ref = oracle.apply_h_spinor(cfg, 0, kg, ig, kin, psi[0, sample].cpu().numpy(), v4, dspin, method=2, terms=2)
    err = band_rel_err(out[:, sample].cpu().numpy(), ref[None])
    print("c4 spinors, local term: %d of %d spinor bands oracle-checked: rel err %.2e" % (len(sample), nsb, err))
    assert err <= TOL, err
    plan.destroy()
    del psi, out
    torch.cuda.empty_cache()


def test_spinor_c2_full_size_sample():
    """Full-size c2 (128^3, radix pair 8 x 16, 1728 projectors): all 216 spinor bands on the GPU, every term with the spin-
    dependent D; the oracle checks first, last and two seeded interior spinor bands."""
    cfg = synth.make_config("c2")
    plan = make_plan(cfg)
    (kg, ig, kin), = lib_spheres(plan)
    v4, dspin = synth.spinor_inputs(cfg)
    plan.set_vloc_spinor(torch.as_tensor(v4, device="cuda"))
    plan.set_dij_spinor(dspin)
    nsb = cfg["nband"] // 2
    psi = synth.gen_psi_torch(cfg, [kin], "cuda")[0][:2 * nsb].reshape(1, nsb, 2, plan.mpw)
    out = plan.apply_h_spinor(psi)
    torch.cuda.synchronize()
    rng = np.random.default_rng(5)
    sample = sorted({0, nsb - 1} | {int(v) for v in rng.choice(np.arange(1, nsb - 1), size=2, replace=False)})
    ref = oracle.apply_h_spinor(cfg, 0, kg, ig, kin, psi[0, sample].cpu().numpy(), v4, dspin, method=2)
    err = band_rel_err(out[:, sample].cpu().numpy(), ref[None])
    print("c2 spinors, all terms: %d of %d spinor bands oracle-checked: rel err %.2e" % (len(sample), nsb, err))
    assert err <= TOL, err
    plan.destroy()
    del psi, out
    torch.cuda.empty_cache()


def test_spinor_with_vector_potential():
    """Velocity gauge (PAPER.md :340): the kinetic diagonal 1/2 |k+G+A|^2 acts on both components."""
    cfg = synth.make_config("c0")
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    v4, dspin = synth.spinor_inputs(cfg)
    plan.set_vloc_spinor(torch.as_tensor(v4, device="cuda"))
    plan.set_dij_spinor(dspin)
    a = [0.3, -0.1, 0.2]
    plan.set_vector_potential(a)
    kg, ig, kin = sph[0]
    psi = synth.gen_psi(cfg, [kin], nband=8).reshape(1, 4, 2, plan.mpw)
    ref = oracle.apply_h_spinor(cfg, 0, kg, ig, oracle.kin_vecpot(cfg["rprimd"], cfg["kpt"][0], kg, a), psi[0], v4, dspin, method=1)
    assert band_rel_err(_spinor_gpu(plan, psi), ref[None]) <= TOL
    plan.destroy()


def test_spinor_not_ready_without_potential():
    cfg = synth.make_config("c0")
    plan = make_plan(cfg)
    with pytest.raises(dft.DftError) as e:
        plan.apply_h_spinor(torch.zeros((1, 2, plan.mpw), dtype=torch.complex128, device="cuda"))
    assert e.value.code == dft.DFT_ERR_NOT_READY
    plan.destroy()
