"""Parity of the CUDA path (through the C ABI) with the oracle: H psi to <= 1e-10 relative per band
(BASELINE.json north_star), on the five configs and the extra cases of SURVEY.md 8(c)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2507_08578_b200 as dft
import synth
from gpu_util import (make_plan, lib_spheres, oracle_spheres, assert_spheres_equal, gpu_apply, oracle_apply,
                      band_rel_err, small_box_ok, nl_launches)

pytestmark = pytest.mark.gpu
TOL = 1e-10     # north_star: "relative error <= 1e-10 per band in FP64"


def _setup(name, **over):
    cfg = synth.make_config(name, **over)
    plan = make_plan(cfg)
    sph = lib_spheres(plan)
    assert_spheres_equal(sph, oracle_spheres(cfg))
    return cfg, plan, sph


@pytest.mark.parametrize("name", ["c0", "c1m", "c2m", "c4m", "aniso", "aniso8", "c3k2", "aniso5t"])
def test_small_cells_all_terms_and_isolations(name):
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    for terms in (7, 1, 2, 4, 3, 6):
        plan.set_option("terms", terms)
        got = gpu_apply(plan, psi)
        ref = oracle_apply(cfg, sph, psi, terms=terms, method=1 if name in ("c0", "aniso", "aniso8", "aniso5t") else 2)
        err = band_rel_err(got, ref)
        assert err <= TOL, "%s terms=%d: rel err %.3e" % (name, terms, err)
        for ik in range(plan.nkpt):                      # pad entries are written as 0
            assert np.all(got[ik][:, plan.npw[ik]:] == 0)
        if terms in (7, 4) and plan.nkpt == 1 and not np.any(cfg["kpt"][0]):
            plan.set_option("gemm_sym", 1)               # k = 0: real GEMMs on the half sphere (automatic only for large cells)
            err = band_rel_err(gpu_apply(plan, psi), ref)
            assert err <= TOL, "%s terms=%d gemm_sym=1: rel err %.3e" % (name, terms, err)
            plan.set_option("gemm_sym", 2)
    if nl_launches(plan, psi.shape[1]) == 1:
        # tiny cell: the runs above took the one-launch non-local kernel; the GEMM kernels (skinny GEMM-1 tiles) must agree
        for terms in (7, 4):
            plan.set_option("terms", terms)
            ref = oracle_apply(cfg, sph, psi, terms=terms, method=1 if name in ("c0", "aniso", "aniso8", "aniso5t") else 2)
            assert plan.apply_h(torch.as_tensor(psi, device="cuda")) is not None and plan.last_launches() == 2     # local term (or zero fill) + one launch
            plan.set_option("nl_tiny", 0)
            err = band_rel_err(gpu_apply(plan, psi), ref)
            assert err <= TOL, "%s terms=%d nl_tiny=0: rel err %.3e" % (name, terms, err)
            assert plan.last_launches() == 4
            plan.set_option("nl_tiny", 1)
    plan.destroy()


@pytest.mark.parametrize("name", ["c0", "c1m", "c4m", "aniso", "c3k2"])
def test_generic_fft_path_agrees(name):
    """Option fft_path=1 forces the generic shared-memory Stockham kernels (used for box lengths with no
    two-stage factorisation), 2 the register path without the TMA ring, 4 the five-pass path where the automatic choice
    would be the fused small-box kernel, 3 that kernel; all paths must match the oracle."""
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    ref = oracle_apply(cfg, sph, psi, method=1 if name in ("c0", "aniso") else 2)
    for path in (1, 2, 4, 0) + ((3,) if small_box_ok(plan) else ()):
        plan.set_option("fft_path", path)
        err = band_rel_err(gpu_apply(plan, psi), ref)
        assert err <= TOL, "%s fft_path=%d: rel err %.3e" % (name, path, err)
    plan.destroy()


@pytest.mark.parametrize("name", ["c1m", "c4m", "aniso", "c3k2"])
def test_both_gemm_variants_agree(name):
    """Option gemm_3m: 1 (default) = three real DMMA products per complex multiply-add (Gauss), 0 = four;
    both must match the oracle, with and without the non-local term's neighbours."""
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    for terms in (7, 4):
        ref = oracle_apply(cfg, sph, psi, terms=terms, method=1 if name == "aniso" else 2)
        plan.set_option("terms", terms)
        for sym in (0, 1):               # gemm_sym = 1 (default): at k = 0 both GEMMs are real GEMMs on the half sphere
            plan.set_option("gemm_sym", sym)
            for g3 in (0, 1):
                plan.set_option("gemm_3m", g3)
                err = band_rel_err(gpu_apply(plan, psi), ref)
                assert err <= TOL, "%s gemm_sym=%d gemm_3m=%d terms=%d: rel err %.3e" % (name, sym, g3, terms, err)
    plan.destroy()


@pytest.mark.parametrize("ngfft", [(20, 20, 180), (18, 20, 256), (20, 24, 128), (16, 20, 240), (15, 15, 225)])
def test_pass_c_barrier_domains(ngfft):
    """Option fft_c_split: the middle FFT pass (z . V . z^-1) with one barrier domain per CTA (0), two
    (1: each half of a 16-line tile with its own named barrier, V half-tile and pace) and the automatic choice (2: two where
    both radices of n3 are >= 12); z lengths 180 = 12 x 15, 256 = 16 x 16, 128 = 8 x 16, 240 = 15 x 16, 225 = 15 x 15, planes
    whose point count is not a multiple of the tile; against the oracle, and bit-identical to each other."""
    cfg, plan, sph = _setup("c0", ngfft=ngfft, nband=11)
    psi = synth.gen_psi(cfg, [sph[0][2]])
    plan.set_option("fft_path", 4)
    outs = []
    for terms in (2, 7):
        plan.set_option("terms", terms)
        ref = oracle_apply(cfg, sph, psi, terms=terms, method=2)
        for split in (0, 1, 2):
            plan.set_option("fft_c_split", split)
            for chunk in (0, 3):
                plan.set_option("band_chunk", chunk)
                got = gpu_apply(plan, psi)
                err = band_rel_err(got, ref)
                assert err <= TOL, "%s terms=%d fft_c_split=%d chunk=%d: %.3e" % (ngfft, terms, split, chunk, err)
                if terms == 2 and chunk == 0:
                    outs.append(got)
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    plan.destroy()


@pytest.mark.parametrize("ngfft", [(45, 54, 75), (54, 45, 135), (75, 45, 54)])
def test_box_lengths_45_54_75_135(ngfft):
    """Register path for the box lengths 45 = 5 x 9, 54 = 6 x 9, 75 = 5 x 15 and 135 = 9 x 15 on every axis in turn
    (all-terms H psi, local term alone, density) against the oracle."""
    cfg, plan, sph = _setup("c0", ngfft=ngfft, ecut=20.0, nband=5)
    psi = synth.gen_psi(cfg, [sph[0][2]])
    for terms in (7, 2):
        plan.set_option("terms", terms)
        ref = oracle_apply(cfg, sph, psi, terms=terms, method=2)
        for path in (0, 2, 1):
            plan.set_option("fft_path", path)
            err = band_rel_err(gpu_apply(plan, psi), ref)
            assert err <= TOL, "%s terms=%d fft_path=%d: %.3e" % (ngfft, terms, path, err)
    plan.set_option("fft_path", 0); plan.set_option("terms", 15)
    gpu_apply(plan, psi)
    assert plan.last_launches() == 5 + nl_launches(plan, 5)      # five passes
    w = np.linspace(0.5, 1.5, 5)[None]
    rho = plan.accumulate_density(torch.as_tensor(psi, device="cuda"), w).cpu().numpy()
    ref = oracle.density(cfg["ngfft"], sph[0][1], psi[0], w[0], method=2)
    assert np.max(np.abs(rho - ref)) <= 1e-12 * ref.max()
    plan.destroy()


@pytest.mark.parametrize("ngfft", [(200, 20, 24), (20, 216, 24), (20, 24, 270), (288, 20, 300), (24, 320, 20), (162, 20, 324),
                                   (20, 360, 24), (24, 20, 400), (384, 20, 24), (20, 432, 24), (24, 20, 480), (20, 576, 24)])
def test_box_lengths_with_radices_18_and_20(ngfft):
    """Register path for 162 = 9 x 18, 200 = 10 x 20, 216 = 12 x 18, 270 = 15 x 18, 288 = 16 x 18, 300 = 15 x 20,
    320 = 16 x 20, 324 = 18 x 18, 360 = 18 x 20, 400 = 20 x 20 and, with the radix 24 = 3 x 8, 384, 432, 480 and 576 on each axis (rows of more than 256 points take the plain
    kernels instead of the TMA ring): all-terms H psi and the local term alone against the oracle, the register path
    without the ring and the generic kernels too, the density, and two-component spinors (Pauli form where the z length
    needs a radix above 16)."""
    cfg, plan, sph = _setup("c0", ngfft=ngfft, nband=3)
    psi = synth.gen_psi(cfg, [sph[0][2]])
    for terms in (7, 2):
        plan.set_option("terms", terms)
        ref = oracle_apply(cfg, sph, psi, terms=terms, method=2)
        for path in (0, 2, 1):
            plan.set_option("fft_path", path)
            err = band_rel_err(gpu_apply(plan, psi), ref)
            assert err <= TOL, "%s terms=%d fft_path=%d: %.3e" % (ngfft, terms, path, err)
    plan.set_option("fft_path", 0); plan.set_option("terms", 15)
    w = np.linspace(0.5, 1.5, 3)[None]
    rho = plan.accumulate_density(torch.as_tensor(psi, device="cuda"), w).cpu().numpy()
    ref = oracle.density(cfg["ngfft"], sph[0][1], psi[0], w[0], method=2)
    assert np.max(np.abs(rho - ref)) <= 1e-12 * ref.max()
    v4, dspin = synth.spinor_inputs(cfg)
    plan.set_vloc_spinor(torch.as_tensor(v4, device="cuda"))
    plan.set_dij_spinor(dspin)
    sp = synth.gen_psi(cfg, [sph[0][2]], nband=4).reshape(1, 2, 2, plan.mpw)
    sref = oracle.apply_h_spinor(cfg, 0, *sph[0], sp[0], v4, dspin, method=2)
    out = plan.apply_h_spinor(torch.as_tensor(sp, device="cuda").contiguous())
    torch.cuda.synchronize()
    assert band_rel_err(out.cpu().numpy(), sref[None]) <= TOL
    plan.destroy()


def test_box_without_two_stage_factorisation():
    """Box 10 x 20 x 27: 10 and 27 have no two-stage factorisation (generic kernels), 20 = 4 x 5 has, so the
    passes of one transform mix both kernel families."""
    cfg, plan, sph = _setup("c0", ngfft=(10, 20, 27))
    psi = synth.gen_psi(cfg, [sph[0][2]])
    err = band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi, method=1))
    assert err <= TOL, err
    plan.destroy()


def test_c0_against_dense_h():
    """tier T0: explicit dense H_{GG'} on the tiny cell (north_star: 'brute-force dense H on the tiny cell')."""
    cfg, plan, sph = _setup("c0")
    kg, ig, kin = sph[0]
    psi = synth.gen_psi(cfg, [kin])
    H = oracle.dense_h(cfg, 0, kg, kin)
    ref = np.stack([oracle.dense_matvec(H, psi[0, b]) for b in range(psi.shape[1])])[None]
    err = band_rel_err(gpu_apply(plan, psi), ref)
    assert err <= TOL, err
    plan.destroy()


@pytest.mark.parametrize("nband", [1, 3, 64, 65])
def test_band_counts_and_chunking(nband):
    cfg, plan, sph = _setup("c1m")
    psi = synth.gen_psi(cfg, [s[2] for s in sph], nband=nband)
    ref = oracle_apply(cfg, sph, psi)
    for path, chunks in ((4, (0, 1, 7)), (0, (0,))):     # five-pass path in band chunks; fused small-box kernel (no chunks)
        plan.set_option("fft_path", path)
        for chunk in chunks:
            plan.set_option("band_chunk", chunk)
            err = band_rel_err(gpu_apply(plan, psi), ref)
            assert err <= TOL, "nband=%d path=%d chunk=%d: %.3e" % (nband, path, chunk, err)
    plan.destroy()


def test_projector_table_matches_oracle():
    for name in ("c0", "aniso", "c3k2"):
        cfg, plan, sph = _setup(name)
        for ik in range(plan.nkpt):
            ref = oracle.projector_table(cfg, ik, sph[ik][0])
            got = plan.get_projectors(ik)
            assert np.max(np.abs(got - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
            dev = plan.projectors_device(ik).cpu().numpy()            # device-to-device copy of the same table
            assert np.array_equal(dev[:, :got.shape[1]], got) and np.all(dev[:, got.shape[1]:] == 0)
        plan.destroy()


def test_tight_box_wraparound():
    """SURVEY.md 8(c) case (iii): a box that just holds the sphere (n_j = 2 m_max + 1 -> heavy aliasing wrap)."""
    cfg, plan, sph = _setup("c0", ngfft=(9, 9, 9))
    psi = synth.gen_psi(cfg, [sph[0][2]])
    err = band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi, method=1))
    assert err <= TOL, err
    plan.destroy()


SMALL_BOX_CASES = [("c0", {}), ("c3k2", {}), ("c1m", {}), ("c2m", {}), ("c4m", {}), ("aniso", {}), ("anisok3", {}),
                   ("c0", {"ngfft": (9, 9, 9)}), ("c0", {"ngfft": (18, 24, 16)}), ("c0", {"ngfft": (12, 10, 8), "ecut": 3.0})]


@pytest.mark.parametrize("name,over", SMALL_BOX_CASES, ids=lambda v: v if isinstance(v, str) else "x".join(map(str, v.get("ngfft", ()))))
def test_small_box_fused_kernel(name, over):
    """fft_path = 3: the whole local term in one kernel, one CTA per (k-point, band), the box in shared memory
    (SURVEY.md 7 step 4(e), 8(d)).  All-terms and local-only results against the oracle, pads zeroed, four launches
    per application (fused local term, GEMM-1, D_ij, GEMM-2), and the automatic choice picks it."""
    cfg, plan, sph = _setup(name, **over)
    assert small_box_ok(plan), "the small-box kernel should serve %s %s" % (name, over)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    method = 1 if name in ("c0", "aniso", "anisok3") else 2
    for path in (3, 5, 0):      # 3 / 0: compile-time-size kernel where the box has one; 5: the run-time-dispatched kernel
        plan.set_option("fft_path", path)
        for terms in (7, 2):
            plan.set_option("terms", terms)
            got = gpu_apply(plan, psi)
            assert plan.last_launches() == (1 + nl_launches(plan, psi.shape[1]) if terms == 7 else 1)
            err = band_rel_err(got, oracle_apply(cfg, sph, psi, terms=terms, method=method))
            assert err <= TOL, "%s fft_path=%d terms=%d: rel err %.3e" % (name, path, terms, err)
            for ik in range(plan.nkpt):
                assert np.all(got[ik][:, plan.npw[ik]:] == 0)
    plan.destroy()


@pytest.mark.parametrize("nband", [1, 3, 64, 65])
def test_small_box_band_counts(nband):
    cfg, plan, sph = _setup("c3k2")
    psi = synth.gen_psi(cfg, [s[2] for s in sph], nband=nband)
    ref = oracle_apply(cfg, sph, psi)
    for path in (3, 5):
        plan.set_option("fft_path", path)
        err = band_rel_err(gpu_apply(plan, psi), ref)
        assert err <= TOL, "nband=%d fft_path=%d: %.3e" % (nband, path, err)
    plan.destroy()


def test_small_box_refused_when_it_does_not_fit():
    """fft_path = 3 on a plan whose working set exceeds one SM's shared memory is DFT_ERR_UNSUPPORTED (no silent
    change of path); the automatic choice then keeps the five-pass kernels."""
    cfg, plan, sph = _setup("c1m", ngfft=(72, 72, 72))
    assert not small_box_ok(plan)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    assert band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi)) <= TOL
    assert plan.last_launches() == 8
    plan.destroy()


def test_set_dij_and_user_workspace_and_host_api():
    cfg, plan, sph = _setup("c1m")
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    d2 = cfg["dij"] * 0.5 + 0.1 * np.eye(cfg["nlmn_max"])[None]
    plan.set_dij(d2)
    plan.set_option("fft_path", 4)           # the five-pass path: the one that uses a workspace
    ws = torch.empty(plan.workspace_bytes_per_band * 2 + 256, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    plan.set_workspace(ws[off:off + plan.workspace_bytes_per_band * 2])
    ref = oracle_apply(cfg, sph, psi, dij=d2)
    assert band_rel_err(gpu_apply(plan, psi), ref) <= TOL
    got_host = plan.apply_h_host(psi)
    assert band_rel_err(got_host, ref) <= TOL
    plan.set_workspace(None)
    assert band_rel_err(gpu_apply(plan, psi), ref) <= TOL
    assert plan.last_launches() == 8
    plan.destroy()


@pytest.mark.parametrize("name", ["c1m", "c4m", "aniso", "c3k2"])
def test_overlap_operator_and_cprj(name):
    """dft_apply_s (S psi, PAPER.md :473) and dft_get_cprj (<p|psi>, :477) against the oracle, both GEMM variants."""
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    rng = np.random.default_rng(3)
    sij = rng.standard_normal(cfg["dij"].shape) * 0.3
    sij = 0.5 * (sij + sij.transpose(0, 2, 1))
    tpsi = torch.as_tensor(psi, device="cuda")
    ident = plan.apply_s(tpsi).cpu().numpy()                  # s_ij = 0 after plan creation: S = 1 on the sphere
    for ik, (kg, ig, kin) in enumerate(sph):
        assert np.array_equal(ident[ik][:, :len(ig)], psi[ik][:, :len(ig)]) and np.all(ident[ik][:, len(ig):] == 0)
    plan.set_sij(sij)
    for g3 in (1, 0, 2):
        plan.set_option("gemm_3m", g3 & 1)
        plan.set_option("gemm_sym", 1 if g3 == 2 else 0)      # last round: the real GEMMs at k = 0 (default for large cells)
        got = plan.apply_s(tpsi).cpu().numpy()
        cp = plan.get_cprj(tpsi).cpu().numpy()
        for ik, (kg, ig, kin) in enumerate(sph):
            ref = oracle.apply_s(cfg, ik, kg, psi[ik], sij)
            err = float(np.max(np.linalg.norm(got[ik] - ref, axis=1) / np.linalg.norm(ref, axis=1)))
            assert err <= TOL, "%s S psi gemm_3m=%d k=%d: %.3e" % (name, g3, ik, err)
            assert np.all(got[ik][:, len(ig):] == 0)
            cref = oracle.cprj(cfg, ik, kg, psi[ik][:, :len(ig)]).T          # [nband][nproj]
            cerr = float(np.max(np.linalg.norm(cp[ik] - cref, axis=1) / np.linalg.norm(cref, axis=1)))
            assert cerr <= TOL, "%s cprj gemm_3m=%d k=%d: %.3e" % (name, g3, ik, cerr)
    assert plan.last_launches() == (3 if name == "c4m" else 2)    # cprj: (split at k = 0,) GEMM-1, reduction
    plan.destroy()


@pytest.mark.parametrize("name", ["c1m", "c4m", "aniso", "c3k2"])
def test_apply_hs_one_set_of_projections(name):
    """dft_apply_hs: H psi and S psi from ONE GEMM-1 (PAPER.md :479-:485) must equal the separate applications' oracle
    results; at k = 0 (c4m) both with the real symmetric-table GEMMs (default) and with the complex kernels."""
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    rng = np.random.default_rng(5)
    sij = rng.standard_normal(cfg["dij"].shape) * 0.3
    sij = 0.5 * (sij + sij.transpose(0, 2, 1))
    plan.set_sij(sij)
    tpsi = torch.as_tensor(psi, device="cuda")
    href = oracle_apply(cfg, sph, psi, method=1 if name == "aniso" else 2)
    for sym in (1, 0):
        plan.set_option("gemm_sym", sym)
        h, s_ = plan.apply_hs(tpsi)
        torch.cuda.synchronize()
        assert band_rel_err(h.cpu().numpy(), href) <= TOL
        got = s_.cpu().numpy()
        for ik, (kg, ig, kin) in enumerate(sph):
            ref = oracle.apply_s(cfg, ik, kg, psi[ik], sij)
            err = float(np.max(np.linalg.norm(got[ik] - ref, axis=1) / np.linalg.norm(ref, axis=1)))
            assert err <= TOL, "%s S psi of apply_hs gemm_sym=%d k=%d: %.3e" % (name, sym, ik, err)
            assert np.all(got[ik][:, len(ig):] == 0)
    plan.destroy()


@pytest.mark.parametrize("name", ["c1m", "aniso", "c3k2", "c2m"])
def test_chebyshev_filter(name):
    """dft_chebyshev_filter (PAPER.md :458, :489) against the oracle's recurrence; T_n grows like cosh(n acosh x) outside
    [-1, 1], so the per-band relative error is what is bounded."""
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    kmax = max(float(s[2].max()) for s in sph)
    cen, e = 0.5 * kmax + 1.0, 0.5 * kmax + 0.5           # damp roughly [0.5, kmax + 1.5] Ha
    plan.set_option("gemm_sym", 1)                          # c2m (k = 0): force the real symmetric-table GEMMs (automatic only for large cells)
    for g3 in (1, 0):
        plan.set_option("gemm_3m", g3)
        for deg in (0, 1, 4, 7):
            t = torch.as_tensor(psi, device="cuda").clone()
            got = plan.chebyshev_filter(t, deg, cen, e).cpu().numpy()
            if plan.nkpt == 1:      # c2m is at k = 0: its GEMMs are the real ones, with a split and a recombination kernel
                assert plan.last_launches() == ((1 if small_box_ok(plan) else 5) + (5 if name == "c2m" else nl_launches(plan, psi.shape[1]))) * deg
            for ik, (kg, ig, kin) in enumerate(sph):
                ref = oracle.chebyshev_filter(cfg, ik, kg, ig, kin, psi[ik], deg, cen, e, method=1 if name == "aniso" else 2)
                npw = len(ig)
                err = float(np.max(np.linalg.norm(got[ik][:, :npw] - ref[:, :npw], axis=1) / np.linalg.norm(ref[:, :npw], axis=1)))
                assert err <= TOL, "%s deg=%d gemm_3m=%d k=%d: %.3e" % (name, deg, g3, ik, err)
                if deg > 0:
                    assert np.all(got[ik][:, npw:] == 0)
    plan.destroy()


@pytest.mark.parametrize("name", ["c1m", "aniso", "c3k2"])
def test_velocity_gauge_kinetic(name):
    """dft_set_vector_potential (PAPER.md :340): kinetic term 1/2|k+G+A|^2, everything else unchanged; switching it off
    restores the plain operator."""
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    a = np.array([0.35, -0.2, 0.15])
    plain = gpu_apply(plan, psi)
    plan.set_vector_potential(a)
    for terms in (7, 1):
        plan.set_option("terms", terms)
        got = gpu_apply(plan, psi)
        for ik, (kg, ig, kin) in enumerate(sph):
            ka = oracle.kin_vecpot(cfg["rprimd"], cfg["kpt"][ik], kg, a)
            ref = oracle.apply_h(cfg, ik, kg, ig, ka, psi[ik], method=1 if name == "aniso" else 2, terms=terms)
            npw = len(ig)
            err = float(np.max(np.linalg.norm(got[ik][:, :npw] - ref[:, :npw], axis=1) / np.linalg.norm(ref[:, :npw], axis=1)))
            assert err <= TOL, "%s terms=%d k=%d: %.3e" % (name, terms, ik, err)
    plan.set_option("terms", 7)
    plan.set_vector_potential(None)
    assert np.array_equal(gpu_apply(plan, psi), plain)
    plan.destroy()


@pytest.mark.parametrize("name,over,path", [("c0", {}, 0), ("c1m", {}, 0), ("aniso", {}, 0), ("c3k2", {}, 0), ("c1m", {}, 1),
                                            ("aniso", {"ngfft": (20, 27, 25)}, 0), ("c0", {"ngfft": (10, 20, 27)}, 0)],
                         ids=lambda v: v if isinstance(v, str) else ("x".join(map(str, v.get("ngfft", ()))) if isinstance(v, dict) else "path%d" % v))
def test_density_accumulation(name, over, path):
    """dft_accumulate_density (Eq. 6, :140) against the oracle, accumulating over k-points, in two calls
    (rho is added to), with a band chunk that leaves a ragged tail; register kernels, generic kernels (fft_path 1) and
    boxes that mix axis lengths with and without a two-radix factorisation (the generic density kernel)."""
    cfg, plan, sph = _setup(name, nband=7, **over)
    plan.set_option("fft_path", path)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    rng = np.random.default_rng(9)
    w = rng.uniform(0.1, 2.0, size=(plan.nkpt, 7))
    plan.set_option("band_chunk", 3)
    tpsi = torch.as_tensor(psi, device="cuda")
    rho = plan.accumulate_density(tpsi, w)
    rho = plan.accumulate_density(tpsi, 0.5 * w, rho)
    torch.cuda.synchronize()
    ref = np.zeros(rho.shape)
    for ik, (kg, ig, kin) in enumerate(sph):
        ref += 1.5 * oracle.density(cfg["ngfft"], ig, psi[ik], w[ik], method=1 if name in ("c0", "aniso") else 2)
    got = rho.cpu().numpy()
    assert np.max(np.abs(got - ref)) <= 1e-12 * ref.max(), np.max(np.abs(got - ref)) / ref.max()
    tau = plan.accumulate_density(tpsi, w, tau=True).cpu().numpy()          # kinetic-energy density of the same equation
    tref = np.zeros(tau.shape)
    for ik, (kg, ig, kin) in enumerate(sph):
        tref += oracle.tau_density(cfg, ik, kg, ig, psi[ik], w[ik], method=1 if name in ("c0", "aniso") else 2)
    assert np.max(np.abs(tau - tref)) <= 1e-12 * tref.max(), np.max(np.abs(tau - tref)) / tref.max()
    plan.destroy()


@pytest.mark.parametrize("name,over,path", [("c1m", {}, 0), ("aniso", {}, 0), ("c3k2", {}, 0), ("c1m", {}, 1),
                                            ("aniso", {"ngfft": (20, 27, 25)}, 4), ("c0", {"ngfft": (10, 20, 27)}, 4)],
                         ids=lambda v: v if isinstance(v, str) else ("x".join(map(str, v.get("ngfft", ()))) if isinstance(v, dict) else "path%d" % v))
def test_meta_gga_term(name, over, path):
    """dft_set_vtau (Eq. 8): the term alone (terms = 8), with everything else (15), and switched off again; on
    the automatic path, on the generic kernels (fft_path 1) and on boxes that mix lengths with and without a two-radix
    factorisation (27 and 10 have none), where the diagonal factors and the accumulation go through the generic passes."""
    cfg, plan, sph = _setup(name, **over)
    plan.set_option("fft_path", path)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    n = cfg["ngfft"]
    rng = np.random.default_rng(6)
    vt = 0.4 + 0.15 * rng.standard_normal((n[2], n[1], n[0]))
    plain = gpu_apply(plan, psi)
    plan.set_vtau(torch.as_tensor(vt, device="cuda"))
    m = 1 if name in ("aniso", "c0") else 2
    tau = np.zeros_like(psi)
    for ik, (kg, ig, kin) in enumerate(sph):
        tau[ik] = oracle.apply_mgga(cfg, ik, kg, ig, psi[ik], vt, method=m)
    plan.set_option("terms", 8)
    assert band_rel_err(gpu_apply(plan, psi), tau) <= TOL
    plan.set_option("terms", 15)
    ref = oracle_apply(cfg, sph, psi, method=m) + tau
    assert band_rel_err(gpu_apply(plan, psi), ref) <= TOL
    plan.set_vtau(None)
    assert np.array_equal(gpu_apply(plan, psi), plain)
    plan.destroy()


@pytest.mark.parametrize("name,nband", [("c4m", 7), ("c4m", 2), ("c4m", 65), ("c2m", 5), ("c0", 8)])
def test_strassen_level_on_the_real_gemms(name, nband):
    """gemm_strassen = 1 (seven half-size products per real GEMM, block tables with a short second half completed by the TMA
    zero fill): H psi with term isolations, S psi, cprj, H psi and S psi from one GEMM-1, and the Chebyshev recurrence."""
    cfg, plan, sph = _setup(name, nband=nband)
    kg, ig, kin = sph[0]
    psi = synth.gen_psi(cfg, [kin])
    tpsi = torch.as_tensor(psi, device="cuda")
    plan.set_option("gemm_sym", 1); plan.set_option("gemm_strassen", 1)
    m = 1 if name == "c0" else 2
    for terms in (7, 4, 5):
        plan.set_option("terms", terms)
        err = band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi, terms=terms, method=m))
        assert err <= TOL, "%s nband=%d terms=%d: %.3e" % (name, nband, terms, err)
    plan.set_option("terms", 7)
    assert plan.last_launches() > 12                         # 7 + 1 GEMM launches + combinations: the Strassen path did run
    merged = gpu_apply(plan, psi)
    plan.set_option("gemm2_merge", 0)                        # the seven back-projection products as seven launches
    separate = gpu_apply(plan, psi)
    assert plan.last_launches() > 20 and np.array_equal(merged, separate)
    plan.set_option("gemm2_merge", 1)
    sij = np.random.default_rng(4).standard_normal(cfg["dij"].shape) * 0.3
    sij = 0.5 * (sij + sij.transpose(0, 2, 1))
    plan.set_sij(sij)
    h, s_ = plan.apply_hs(tpsi)
    cp = plan.get_cprj(tpsi).cpu().numpy()[0]
    sref = oracle.apply_s(cfg, 0, kg, psi[0], sij)
    assert band_rel_err(h.cpu().numpy(), oracle_apply(cfg, sph, psi, method=m)) <= TOL
    assert band_rel_err(s_.cpu().numpy(), sref[None]) <= TOL
    assert band_rel_err(plan.apply_s(tpsi).cpu().numpy(), sref[None]) <= TOL
    cref = oracle.cprj(cfg, 0, kg, psi[0][:, :len(ig)]).T
    assert float(np.max(np.linalg.norm(cp - cref, axis=1) / np.linalg.norm(cref, axis=1))) <= TOL
    cen, e = 0.5 * float(kin.max()) + 1.0, 0.5 * float(kin.max()) + 0.5
    got = plan.chebyshev_filter(tpsi.clone(), 3, cen, e).cpu().numpy()
    ref = oracle.chebyshev_filter(cfg, 0, kg, ig, kin, psi[0], 3, cen, e, method=m)
    assert band_rel_err(got, ref[None]) <= TOL
    plan.destroy()


@pytest.mark.parametrize("nband", [1, 3, 65])
def test_symmetric_table_gemms_with_other_terms(nband):
    """gemm_sym = 1 (k = 0: real GEMMs on the half sphere) together with what else can change the operator: a vector
    potential (kinetic diagonal only; the projector symmetry is untouched), the meta-GGA term, odd band counts and a band
    count that spans two GEMM tiles; and after proj_mode went to 1 and back (the full table is rebuilt, the half table stays)."""
    cfg, plan, sph = _setup("c4m", nband=nband)
    kg, ig, kin = sph[0]
    psi = synth.gen_psi(cfg, [kin])
    plan.set_option("gemm_sym", 1)
    a = np.array([0.2, 0.1, -0.3])
    plan.set_vector_potential(a)
    n = cfg["ngfft"]
    vt = 0.4 + 0.15 * np.random.default_rng(8).standard_normal((n[2], n[1], n[0]))
    plan.set_vtau(torch.as_tensor(vt, device="cuda"))
    ka = oracle.kin_vecpot(cfg["rprimd"], cfg["kpt"][0], kg, a)
    ref = oracle.apply_h(cfg, 0, kg, ig, ka, psi[0]) + oracle.apply_mgga(cfg, 0, kg, ig, psi[0], vt)
    got = gpu_apply(plan, psi)
    assert band_rel_err(got, ref[None]) <= TOL
    plan.set_option("proj_mode", 1); plan.set_option("proj_mode", 0)
    assert band_rel_err(gpu_apply(plan, psi), ref[None]) <= TOL
    plan.set_vector_potential(None); plan.set_vtau(None)
    assert band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi)) <= TOL
    plan.destroy()


@pytest.mark.parametrize("name", ["c1m", "c4m", "c2m", "aniso", "aniso8", "c3k2", "aniso5t"])
def test_factorised_projectors(name):
    """Option proj_mode = 1 (PAPER.md :477 "computed on-the-fly"): p = FY . S evaluated inside both GEMMs instead of the
    materialised table; H psi, S psi and cprj must match the oracle as before.  Atoms with more than 8 projectors (Al: 9)
    are walked as two blocks of 8 rows; aniso5t has five atom types in mixed order whose 56 form-factor rows exceed what
    the kernels hold at once, so both GEMMs run once per group of types."""
    cfg, plan, sph = _setup(name)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    tpsi = torch.as_tensor(psi, device="cuda")
    plan.set_option("proj_mode", 1)
    m = 1 if name.startswith("aniso") else 2
    for terms in (15, 4):
        plan.set_option("terms", terms)
        ref = oracle_apply(cfg, sph, psi, terms=terms & 7, method=m)
        err = band_rel_err(gpu_apply(plan, psi), ref)
        assert err <= TOL, "%s terms=%d: %.3e" % (name, terms, err)
    cp = plan.get_cprj(tpsi).cpu().numpy()
    rng = np.random.default_rng(3)
    sij = rng.standard_normal(cfg["dij"].shape) * 0.3
    sij = 0.5 * (sij + sij.transpose(0, 2, 1))
    plan.set_sij(sij)
    got = plan.apply_s(tpsi).cpu().numpy()
    for ik, (kg, ig, kin) in enumerate(sph):
        cref = oracle.cprj(cfg, ik, kg, psi[ik][:, :len(ig)]).T
        assert float(np.max(np.linalg.norm(cp[ik] - cref, axis=1) / np.linalg.norm(cref, axis=1))) <= TOL
        sref = oracle.apply_s(cfg, ik, kg, psi[ik], sij)
        assert float(np.max(np.linalg.norm(got[ik] - sref, axis=1) / np.linalg.norm(sref, axis=1))) <= TOL
    plan.set_option("terms", 15)
    if name in ("aniso5t", "aniso"):     # the recurrence in the epilogue of the LAST group's GEMM-2 only
        kmax = max(float(s[2].max()) for s in sph)
        cen, e = 0.5 * kmax + 1.0, 0.5 * kmax + 0.5
        got = plan.chebyshev_filter(tpsi.clone(), 3, cen, e).cpu().numpy()
        for ik, (kg, ig, kin) in enumerate(sph):
            ref = oracle.chebyshev_filter(cfg, ik, kg, ig, kin, psi[ik], 3, cen, e, method=1)
            npw = len(ig)
            assert float(np.max(np.linalg.norm(got[ik][:, :npw] - ref[:, :npw], axis=1) / np.linalg.norm(ref[:, :npw], axis=1))) <= TOL
    plan.set_option("proj_mode", 0)
    assert band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi, method=m)) <= TOL
    plan.destroy()


def test_plan_created_in_factorised_mode_never_builds_the_table():
    """dft_plan_create_opts with proj_mode = 1: the [nproj][mpw] table is neither allocated nor filled (device memory in
    use grows by less than the table's size), H psi matches the oracle, reading the table back is refused, the radial-table
    range check still fires, an unknown key is refused without leaking a plan, and proj_mode = 0 later builds the table."""
    cfg = synth.make_config("c2m", ecut=4.0)
    torch.cuda.synchronize(); torch.cuda.empty_cache()
    free0 = torch.cuda.mem_get_info()[0]
    plan = make_plan(cfg, options=[("proj_mode", 1), ("terms", 15)])
    torch.cuda.synchronize()
    used = free0 - torch.cuda.mem_get_info()[0]
    tab = plan.nproj * plan.mpw * 16
    assert tab > (64 << 20), "the cell is too small for the memory check to mean anything"
    assert used < tab // 2, "plan took %d bytes, the table alone would be %d" % (used, tab)
    sph = lib_spheres(plan)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    assert band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi, method=2)) <= TOL
    with pytest.raises(dft.DftError):
        plan.get_projectors(0)
    plan.set_option("proj_mode", 0)
    assert band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi, method=2)) <= TOL
    assert plan.get_projectors(0).shape == (plan.nproj, plan.npw[0])
    plan.destroy()
    with pytest.raises(dft.DftError):
        make_plan(cfg, options={"proj_mode": 1, "no_such_option": 3})
    short = dict(cfg, types=[dict(t, nq=t["nq"] // 2, f=t["f"][:, :t["nq"] // 2].copy(), f2=t["f2"][:, :t["nq"] // 2].copy()) for t in cfg["types"]])
    with pytest.raises(dft.DftError) as ei:
        make_plan(short, options={"proj_mode": 1})
    assert ei.value.code == dft.DFT_ERR_TABLE_RANGE


def test_apply_h_is_cuda_graph_capturable():
    """dft_apply_h only enqueues (no allocation or synchronisation once scratch exists), so a launch-bound small cell
    can be captured into a CUDA graph and replayed."""
    cfg, plan, sph = _setup("c0")
    psi = torch.as_tensor(synth.gen_psi(cfg, [s[2] for s in sph]), device="cuda")
    out = torch.empty_like(psi)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        plan.apply_h(psi, out)                                  # warm-up: scratch allocation, kernel attributes
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    ref = out.clone()
    graph = torch.cuda.CUDAGraph()
    out.zero_()
    with torch.cuda.graph(graph):
        plan.apply_h(psi, out)
    out.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    psi.mul_(2.0)
    graph.replay()
    torch.cuda.synchronize()
    assert torch.allclose(out, 2.0 * ref, rtol=1e-13, atol=0)
    plan.destroy()


def test_degenerate_inputs():
    """Edge cases of the method: no bands, one plane wave (ecut below the first shell), a k-point whose sphere is empty,
    and error codes for bad arguments."""
    import paper_2507_08578_b200 as dft
    cfg, plan, sph = _setup("c0")
    empty = torch.zeros((1, 0, plan.mpw), dtype=torch.complex128, device="cuda")
    assert plan.apply_h(empty).shape == (1, 0, plan.mpw) and plan.last_launches() == 0
    assert plan.apply_s(empty).numel() == 0 and plan.get_cprj(empty).numel() == 0
    plan.chebyshev_filter(empty, 3, 1.0, 2.0)
    with pytest.raises(dft.DftError) as ei:
        plan.set_option("no_such_option", 1)
    assert ei.value.code == dft.DFT_ERR_INVALID_ARG
    with pytest.raises(dft.DftError):
        plan.chebyshev_filter(torch.zeros((1, 2, plan.mpw), dtype=torch.complex128, device="cuda"), 2, 0.0, 0.0)   # halfwidth must be > 0
    plan.destroy()
    # one plane wave at Gamma: H is the 1x1 matrix kin(0) + mean(V) + sum |p(0)|^2-terms; compare with the oracle
    cfg, plan, sph = _setup("c0", ecut=0.05)
    assert plan.npw[0] == 1
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    assert band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi, method=1)) <= TOL
    plan.destroy()
    # k = (1/2,1/2,1/2) of the FCC cell with a cutoff below its lowest |k+G|^2/2: the sphere is empty, nothing to do
    cfg = synth.make_config("c0", ecut=0.05, kpt=[[0.5, 0.5, 0.5]])
    okg, oig, okin = oracle.sphere(cfg["rprimd"], cfg["kpt"][0], cfg["ecut"], cfg["ngfft"])
    assert len(oig) == 0
    plan = make_plan(cfg)
    assert plan.npw[0] == 0 and plan.mpw == 0
    out = plan.apply_h(torch.zeros((1, 4, 0), dtype=torch.complex128, device="cuda"))
    assert out.numel() == 0
    plan.destroy()


def test_host_api_band_groups():
    """dft_apply_h_host cuts one k-point's bands into groups whose copies overlap the neighbours' kernels;
    the result must not depend on the grouping."""
    cfg, plan, sph = _setup("c1m", nband=200)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    ref = oracle_apply(cfg, sph, psi)
    plan.set_option("fft_path", 4)
    for groups in (3, 1, 4):
        plan.set_option("host_groups", groups)
        got = plan.apply_h_host(psi)
        assert band_rel_err(got, ref) <= TOL, groups
        assert plan.last_launches() == 8 * (2 if groups > 1 else 1)   # 200 bands -> groups of 128 and 72
    plan.destroy()


def test_multik_host_api_and_small_user_workspace():
    """Several k-points: the host API takes its single-copy path, and a caller-owned workspace too small for the
    all-k-points-per-launch FFT path makes the library fall back to one k-point per launch; same result either way."""
    cfg, plan, sph = _setup("c3k2")
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    ref = oracle_apply(cfg, sph, psi)
    plan.set_option("fft_path", 4)
    assert band_rel_err(gpu_apply(plan, psi), ref) <= TOL
    batched_launches = plan.last_launches()
    assert band_rel_err(plan.apply_h_host(psi), ref) <= TOL
    ws = torch.empty(plan.workspace_bytes_per_band + 256, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    plan.set_workspace(ws[off:off + plan.workspace_bytes_per_band])
    assert band_rel_err(gpu_apply(plan, psi), ref) <= TOL
    assert plan.last_launches() > batched_launches            # one band and one k-point per launch now
    plan.set_workspace(None)
    plan.destroy()


def test_host_api_uneven_groups():
    """With enough bands the first and last groups of dft_apply_h_host are one 64-band tile each (their copies are the
    only exposed ones): 520 bands, 4 groups -> 64, 256, 136, 64."""
    cfg, plan, sph = _setup("c1m", nband=520)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    plan.set_option("host_groups", 4)
    plan.set_option("fft_path", 4)
    got = plan.apply_h_host(psi)
    assert plan.last_launches() == 8 * 4
    ref = gpu_apply(plan, psi)
    assert band_rel_err(got, ref) <= 1e-13
    sample = [0, 63, 64, 319, 320, 455, 456, 519]
    oref = oracle_apply(cfg, sph, psi[:, sample])
    assert band_rel_err(got[:, sample], oref) <= TOL
    plan.destroy()


def test_host_api_ramped_groups():
    """Six groups and at least 128 bands per group: 64, 128, middle groups, 128, 64 (a group's copies run under its
    neighbours' kernels, and large groups next to the small first and last ones would outlast them): 800 bands ->
    64, 128, 256, 160, 128, 64."""
    cfg, plan, sph = _setup("c1m", nband=800)
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    plan.set_option("host_groups", 6)
    plan.set_option("fft_path", 4)
    got = plan.apply_h_host(psi)
    assert plan.last_launches() == 8 * 6
    ref = gpu_apply(plan, psi)
    assert band_rel_err(got, ref) <= 1e-13
    sample = [0, 63, 64, 191, 192, 447, 448, 607, 608, 735, 736, 799]       # both sides of every group boundary
    oref = oracle_apply(cfg, sph, psi[:, sample])
    assert band_rel_err(got[:, sample], oref) <= TOL
    plan.destroy()


def test_c1_full():
    cfg, plan, sph = _setup("c1")
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    err = band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi))
    assert err <= TOL, err
    plan.destroy()


def test_c3_full_multik_batch():
    cfg, plan, sph = _setup("c3")
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    err = band_rel_err(gpu_apply(plan, psi), oracle_apply(cfg, sph, psi))
    assert err <= TOL, err
    plan.destroy()


def _bench_launch_sample(plan, nband, per_tile, seed):
    """A seeded band sample that hits EVERY 64-band GEMM tile and every FFT band chunk of the bench launch configuration:
    first and last band of each tile plus per_tile - 2 seeded interior ones (the FFT chunk boundaries are added too)."""
    rng = np.random.default_rng(seed)
    sample = set()
    for t0 in range(0, nband, 64):
        t1 = min(nband, t0 + 64)
        sample.update((t0, t1 - 1))
        if t1 - t0 > 2 and per_tile > 2:
            sample.update(int(v) for v in rng.choice(np.arange(t0 + 1, t1 - 1), size=min(per_tile - 2, t1 - t0 - 2), replace=False))
    lo, full = plan.workspace_bytes(nband)
    chunk = max(1, min(nband, (8 << 30) // max(1, full // nband)))          # the library's default: about 8 GiB of scratch
    for b0 in range(0, nband, chunk):
        sample.update((b0, min(nband, b0 + chunk) - 1))
    return sorted(sample), chunk


def _sampled_full_size(name, per_tile, nvariant):
    """Full-size run in bench.py's launch configuration; the oracle computes a seeded sample of >= 64 bands one by
    one (bands are independent, PAPER.md :436; 'a seeded >= 64-band subset ... and say so')."""
    cfg, plan, sph = _setup(name)
    nband = cfg["nband"]
    sample, chunk = _bench_launch_sample(plan, nband, per_tile, 7)
    ntile, nchunk = (nband + 63) // 64, (nband + chunk - 1) // chunk
    assert len(sample) >= 64 and len({b // 64 for b in sample}) == ntile and len({b // chunk for b in sample}) == nchunk
    psi = synth.gen_psi_torch(cfg, [s[2] for s in sph], "cuda")
    out = plan.apply_h(psi)
    torch.cuda.synchronize()
    psi_s = psi[:, sample].cpu().numpy()
    got = out[:, sample].cpu().numpy()
    ref = oracle_apply(cfg, sph, psi_s)
    err = band_rel_err(got, ref)
    print("%s: %d of %d bands oracle-checked (all %d GEMM band tiles, all %d FFT chunks of %d bands): rel err %.2e"
          % (name, len(sample), nband, ntile, nchunk, chunk, err))
    assert err <= TOL, "%s %d sampled bands: %.3e" % (name, len(sample), err)
    # property at full size: Hermiticity <phi|H psi> = <H phi|psi> on two other bands
    a, b = 1, nband - 2
    lhs = torch.vdot(psi[0, a], out[0, b]); rhs = torch.vdot(out[0, a], psi[0, b])
    scale = torch.linalg.norm(psi[0, a]) * torch.linalg.norm(out[0, b])
    assert abs(lhs - rhs) <= 1e-11 * scale
    # the other GEMM variants at full size: 4-product table kernels and factorised projectors, on >= 16 of those bands
    # (one per GEMM band tile); every band of the 3M result is also compared with them (1e-12: same operator, other rounding)
    sub = sample[::max(1, len(sample) // max(nvariant, ntile))]
    pos = [sample.index(b) for b in sub]
    assert len(sub) >= 16 and len({b // 64 for b in sub}) == ntile
    # (the default at k = 0 is the symmetric-table real GEMMs with one Strassen level; gemm_strassen = 0 gives the plain real GEMMs,
    # gemm_sym = 0 the complex 3M kernels, then the others)
    for key, val in (("gemm_strassen", 0), ("gemm_sym", 0), ("gemm_3m", 0), ("proj_mode", 1)):
        plan.set_option(key, val)
        out2 = plan.apply_h(psi)
        torch.cuda.synchronize()
        err = band_rel_err(out2[:, sub].cpu().numpy(), ref[:, pos])
        assert err <= TOL, "%s %s=%d %d sampled bands: %.3e" % (name, key, val, len(sub), err)
        cross = float((torch.linalg.norm(out2 - out, dim=-1) / torch.linalg.norm(out, dim=-1)).max())
        assert cross <= 1e-12, "%s %s=%d vs default on all bands: %.3e" % (name, key, val, cross)
        del out2
    plan.destroy()
    del psi, out
    torch.cuda.empty_cache()


def test_c2_full_size_64_band_sample():
    _sampled_full_size("c2", 10, 16)      # 7 tiles x up to 10 bands = 68 of 432 bands


def test_c4_full_size_64_band_sample():
    _sampled_full_size("c4", 4, 16)       # 16 tiles x 4 bands (+ FFT chunk boundaries) = 64+ of 1024 bands


def test_multik_scratch_maxima_on_different_kpoints():
    """anisok3: the k-point with most columns (T1) is not the one with most planes (T2), so the all-k-points-per-launch
    path needs max_k t1 + max_k t2 per band and k-point, more than max_k (t1 + t2).  Run it in an exactly sized caller
    workspace with guard regions on both sides; the guards must stay untouched and the result must match the oracle."""
    cfg, plan, sph = _setup("anisok3")
    plan.set_option("fft_path", 4)
    geo = []
    n1, n2, n3 = cfg["ngfft"]
    for kg, ig, kin in sph:
        col = np.unique(ig // n1)
        geo.append(((len(col) * n1 * 16 + 255) // 256 * 256, (len(np.unique(col // n2)) * n2 * n1 * 16 + 255) // 256 * 256))
    assert max(range(3), key=lambda i: geo[i][0]) != max(range(3), key=lambda i: geo[i][1])
    nband = cfg["nband"]
    lo, full = plan.workspace_bytes(nband)
    assert lo == max(a + b for a, b in geo)
    assert full == (max(a for a, _ in geo) + max(b for _, b in geo)) * 3 * nband > lo * 3 * nband
    psi = synth.gen_psi(cfg, [s[2] for s in sph])
    ref = oracle_apply(cfg, sph, psi, method=1)
    guard = 4096
    buf = torch.full((full + 2 * guard + 256,), 0xA5, dtype=torch.uint8, device="cuda")
    off = (-buf.data_ptr()) % 256 + guard
    off += (-(buf.data_ptr() + off)) % 256
    plan.set_workspace(buf[off:off + full])
    got = gpu_apply(plan, psi)
    assert plan.last_launches() == 5 + nl_launches(plan, nband)   # one launch per pass over all three k-points
    assert band_rel_err(got, ref) <= TOL
    assert bool((buf[:off] == 0xA5).all()) and bool((buf[off + full:] == 0xA5).all()), "scratch written outside the workspace"
    # one byte less than the batched layout needs: the library must fall back to one k-point per launch, not overrun
    plan.set_workspace(buf[off:off + full - 256])
    got = gpu_apply(plan, psi)
    assert plan.last_launches() > 5 + nl_launches(plan, nband) and band_rel_err(got, ref) <= TOL
    assert bool((buf[:off] == 0xA5).all()) and bool((buf[off + full - 256:] == 0xA5).all())
    plan.set_workspace(None)
    plan.destroy()
