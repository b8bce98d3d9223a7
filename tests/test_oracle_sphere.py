"""Pins of the oracle's lattice algebra and G-sphere builder (SURVEY.md 8(c) readings 1-3)."""
import os

import numpy as np
import pytest

import oracle
import synth
from util import config, sphere


def _golden(path):
    out = {}
    for line in open(path):
        if line.strip() and not line.startswith("#"):
            t = line.split(); out[t[0]] = [int(v) for v in t[1:]]
    return out


def test_counts_match_survey_enumeration(golden_dir):
    for name, counts in _golden(os.path.join(golden_dir, "sphere_counts.txt")).items():
        c = synth.make_config(name, with_vloc=False)
        got = [len(oracle.sphere(c["rprimd"], k, c["ecut"], c["ngfft"])[0]) for k in c["kpt"]]
        assert got == counts, name


def test_geometry_matches_survey(golden_dir):
    for name, (mn, mx, ncol) in _golden(os.path.join(golden_dir, "sphere_geometry.txt")).items():
        kg, ig, _ = sphere(name)
        assert kg.min() == mn and kg.max() == mx
        assert len(np.unique(kg[:, 0] * 100000 + kg[:, 1])) == ncol
    c = config("c3")
    for ik in range(c["nkpt"]):
        kg, _, _ = sphere("c3", ik)
        assert 185 <= len(np.unique(kg[:, 0] * 1000 + kg[:, 1])) <= 189
        assert kg[:, 2].min() == -7 and kg[:, 2].max() == 7


@pytest.mark.parametrize("name", ["c0", "c1", "c3", "c2"])
def test_cubic_closed_form_and_independent_enumeration(name):
    """For cubic cells 1/2|k+G|^2 = (2 pi/L)^2 |k+m|^2/2; for the FCC cell use numpy's inverse.
    The set is re-enumerated with numpy over the whole box (different code path and formula)."""
    c = config(name)
    n1, n2, n3 = c["ngfft"]
    Bm = np.linalg.inv(c["rprimd"]).T
    for ik in range(min(c["nkpt"], 3)):
        kg, ig, kin = sphere(name, ik)
        k = c["kpt"][ik]
        m = [np.where(np.arange(n) <= (n - 1) // 2, np.arange(n), np.arange(n) - n) for n in (n1, n2, n3)]
        M3, M2, M1 = np.meshgrid(m[2], m[1], m[0], indexing="ij")
        t = np.stack([M1 + k[0], M2 + k[1], M3 + k[2]], -1)
        q = 2 * np.pi * t @ Bm
        e = 0.5 * np.sum(q * q, -1)
        inside = np.flatnonzero(e.ravel() <= c["ecut"])
        assert np.array_equal(inside, ig)
        np.testing.assert_allclose(kin, e.ravel()[inside], rtol=2e-15)
        # margin: no box point sits within rounding distance of the cutoff (reading 1)
        assert np.min(np.abs(e - c["ecut"])) / c["ecut"] > 1e-5


def test_continuum_estimate():
    """npw ~ Omega (2 ecut)^(3/2)/(6 pi^2), within the surface term."""
    for name in ("c0", "c1", "c2", "c4"):
        c = config(name) if name != "c4" else synth.make_config("c4", with_vloc=False)
        npw = len(oracle.sphere(c["rprimd"], c["kpt"][0], c["ecut"], c["ngfft"])[0])
        est = abs(np.linalg.det(c["rprimd"])) * (2 * c["ecut"]) ** 1.5 / (6 * np.pi ** 2)
        assert abs(npw - est) / est < 0.04, (name, npw, est)


def test_ordering_and_wrap():
    for name in ("c0", "c1", "aniso"):
        c = config(name); n = np.array(c["ngfft"])
        kg, ig, _ = sphere(name)
        assert np.all(np.diff(ig) > 0)                       # strictly increasing box index
        i1 = ig % n[0]; i2 = (ig // n[0]) % n[1]; i3 = ig // (n[0] * n[1])
        for i, col in zip((i1, i2, i3), range(3)):
            nn = n[col]
            m = np.where(i <= (nn - 1) // 2, i, i - nn)
            assert np.array_equal(m, kg[:, col])


def test_inversion_symmetry_at_gamma_and_k_shift():
    c = config("c0")
    kg, _, _ = sphere("c0")
    s = {tuple(v) for v in kg}
    assert all((-a, -b, -d) in s for a, b, d in s)
    # S_{k+integer} is S_k shifted by that integer
    c1 = config("c1")
    k = c1["kpt"][0]; sh = np.array([1, -1, 0])
    kgA, _, kinA = oracle.sphere(c1["rprimd"], k, c1["ecut"], c1["ngfft"])
    kgB, _, kinB = oracle.sphere(c1["rprimd"], k + sh, c1["ecut"], c1["ngfft"])
    A = {tuple(v) for v in kgA}; B = {tuple(v + sh) for v in kgB}
    assert A == B


def test_inclusive_boundary():
    """ecut := kin(m*) exactly as the rule computes it -> m* (and -m* at Gamma) are inside."""
    c = config("c0")
    for mstar in ([3, -1, 2], [4, 0, 0], [1, 1, 1]):
        e = oracle.kin_of(c["rprimd"], [0, 0, 0], mstar)
        kg, _, kin = oracle.sphere(c["rprimd"], [0, 0, 0], e, c["ngfft"])
        s = {tuple(v) for v in kg}
        assert tuple(mstar) in s and tuple(-np.array(mstar)) in s
        assert kin.max() == e
        kg2, _, _ = oracle.sphere(c["rprimd"], [0, 0, 0], np.nextafter(e, 0), c["ngfft"])
        assert tuple(mstar) not in {tuple(v) for v in kg2}


def test_lattice_duality_and_fit():
    rng = np.random.default_rng(5)
    for _ in range(5):
        A = rng.standard_normal((3, 3)) + 4 * np.eye(3)
        Bm, gm = oracle.lattice(A)
        np.testing.assert_allclose(A @ Bm.T, np.eye(3), atol=1e-14)
        np.testing.assert_allclose(gm, Bm @ Bm.T, atol=1e-15)
    c = config("c0")
    fits, mn, mx = oracle.sphere_extent(c["rprimd"], c["kpt"][0], c["ecut"], c["ngfft"])
    assert fits and list(mn) == [-4] * 3 and list(mx) == [4] * 3
    fits, _, _ = oracle.sphere_extent(c["rprimd"], c["kpt"][0], c["ecut"], (8, 20, 20))
    assert not fits
    # random triclinic lattice, random k: brute force over the box == bounded enumeration of the extent
    A = rng.standard_normal((3, 3)) + 6 * np.eye(3); k = rng.uniform(-.5, .5, 3)
    fits, mn, mx = oracle.sphere_extent(A, k, 3.0, (40, 40, 40))
    kg, _, _ = oracle.sphere(A, k, 3.0, (40, 40, 40))
    assert fits and np.array_equal(kg.min(0), mn) and np.array_equal(kg.max(0), mx)
