"""Whole-operator pins of the oracle (SURVEY.md 8(c) "Whole operator" row)."""
import numpy as np
import pytest

import oracle
import synth
from util import config, sphere, rel_err, rand_c


@pytest.mark.parametrize("name,ik", [("c0", 0), ("aniso", 0), ("c3k2", 1), ("c1m", 0), ("c2m", 0), ("c4m", 0)])
def test_dense_h_equals_fft_path_and_is_hermitian(name, ik):
    c = config(name); kg, ig, kin = sphere(name, ik)
    psi = synth.gen_psi(c, [sphere(name, j)[2] for j in range(c["nkpt"])])[ik]
    H = oracle.dense_h(c, ik, kg, kin)
    assert abs(H - H.conj().T).max() < 1e-13 * abs(H).max()
    ref = np.array([oracle.dense_matvec(H, p[:len(kg)]) for p in psi])
    for method in (1, 2):
        got = oracle.apply_h(c, ik, kg, ig, kin, psi, method=method)
        assert rel_err(got[:, :len(kg)], ref) < 1e-12
        assert np.all(got[:, len(kg):] == 0)


def test_hermiticity_linearity_permutation_batching():
    c = config("c1m"); kg, ig, kin = sphere("c1m")
    x = rand_c((4, len(kg)), 11)
    h = oracle.apply_h(c, 0, kg, ig, kin, x)
    # <phi|H psi> = <H phi|psi> = conj(<psi|H phi>)
    a = np.vdot(x[0], h[1]); b = np.vdot(h[0], x[1]); d = np.conj(np.vdot(x[1], h[0]))
    assert abs(a - b) < 1e-12 * abs(a) and abs(a - d) < 1e-12 * abs(a)
    lin = oracle.apply_h(c, 0, kg, ig, kin, (2.5 * x[0] - 1j * x[2])[None])[0]
    assert rel_err(lin, 2.5 * h[0] - 1j * h[2]) < 1e-13
    perm = [2, 0, 3, 1]
    assert rel_err(oracle.apply_h(c, 0, kg, ig, kin, x[perm]), h[perm]) < 1e-14
    assert rel_err(oracle.apply_h(c, 0, kg, ig, kin, x[1:2]), h[1:2]) < 1e-14


def test_translation_covariance():
    """Shift atoms and V by a grid vector tau, multiply c(m) by exp(-2 pi i (k+m).tau):
    (H psi)(m) picks up the same phase.  Exercises sphere, wrap, structure factors and D_ij at once."""
    c = dict(config("aniso")); kg, ig, kin = sphere("aniso")
    n1, n2, n3 = c["ngfft"]
    s = np.array([3, -5, 7]); tau = s / np.array([n1, n2, n3])
    psi = rand_c((2, len(kg)), 13)
    h = oracle.apply_h(c, 0, kg, ig, kin, psi)
    c2 = dict(c)
    c2["xred"] = c["xred"] + tau
    c2["vloc"] = np.roll(c["vloc"], shift=(s[2], s[1], s[0]), axis=(0, 1, 2))
    ph = np.exp(-2j * np.pi * ((kg + c["kpt"][0]) @ tau))
    h2 = oracle.apply_h(c2, 0, kg, ig, kin, psi * ph)
    assert rel_err(h2, h * ph) < 1e-13


def test_term_isolation_adds_up():
    c = config("c0"); kg, ig, kin = sphere("c0")
    x = rand_c((2, len(kg)), 17)
    parts = sum(oracle.apply_h(c, 0, kg, ig, kin, x, terms=t) for t in (oracle.KIN, oracle.LOC, oracle.NL))
    assert rel_err(parts, oracle.apply_h(c, 0, kg, ig, kin, x)) < 1e-14


def test_generator_is_chunk_independent():
    c = config("c0"); kg, ig, kin = sphere("c0")
    full = synth.gen_psi(c, [kin])
    some = synth.gen_psi(c, [kin], bands=[5, 2])
    assert np.array_equal(some[0, 0], full[0, 5]) and np.array_equal(some[0, 1], full[0, 2])
    assert abs(np.std(full.real * (1 + 2 * kin)) - 1) < 0.1
    d = c["dij"]
    assert np.array_equal(d, d.transpose(0, 2, 1))


def test_chebyshev_filter_pins():
    """The recurrence reproduces the Chebyshev polynomial of H: (i) free electron (V = 0, D = 0), H diagonal, so the
    result is numpy's chebval of (kin - c)/e times psi; (ii) c0 with every term, through the eigen-decomposition of the
    dense H (numpy eigh): V T_n((lambda - c)/e) V^H psi; (iii) degrees 0 and 1 by hand."""
    from numpy.polynomial import chebyshev as C
    import oracle
    from util import config, sphere, rand_c, rel_err
    c = config("c0"); kg, ig, kin = sphere("c0")
    psi = rand_c((2, len(kg)), 21)
    cen, e = 6.0, 5.0
    for deg in (2, 5, 10):
        coef = np.zeros(deg + 1); coef[deg] = 1.0
        got = oracle.chebyshev_filter(c, 0, kg, ig, kin, psi, deg, cen, e, terms=oracle.KIN)
        assert rel_err(got, C.chebval((kin - cen) / e, coef)[None, :] * psi) < 1e-12
    H = oracle.dense_h(c, 0, kg, kin)
    lam, V = np.linalg.eigh(H)
    cen, e = 0.5 * (lam[-1] + lam[4]), 0.5 * (lam[-1] - lam[4])          # damp everything above the 4 lowest states
    for deg in (3, 8):
        coef = np.zeros(deg + 1); coef[deg] = 1.0
        ref = (V @ (C.chebval((lam - cen) / e, coef)[:, None] * (V.conj().T @ psi.T))).T
        got = oracle.chebyshev_filter(c, 0, kg, ig, kin, psi, deg, cen, e, method=1)
        assert rel_err(got, ref) < 1e-11
    assert np.array_equal(oracle.chebyshev_filter(c, 0, kg, ig, kin, psi, 0, cen, e), psi)
    h1 = oracle.apply_h(c, 0, kg, ig, kin, psi)
    assert rel_err(oracle.chebyshev_filter(c, 0, kg, ig, kin, psi, 1, cen, e), (h1 - cen * psi) / e) < 1e-15


def test_velocity_gauge_kinetic_pins():
    """1/2|k+G+A|^2 (PAPER.md :340): A = 0 gives the sphere's kin; A = 2 pi Bm^T d for an integer triple d is the
    kinetic energy of the plane wave m + d (k shifted by a reciprocal vector); cubic closed form; and with V = 0,
    D = 0 the operator is that diagonal."""
    import oracle
    from util import config, sphere, rand_c, rel_err
    for name in ("c0", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        k = np.asarray(c["kpt"][0], float)
        assert np.max(np.abs(oracle.kin_vecpot(c["rprimd"], k, kg, [0, 0, 0]) - kin)) < 1e-13 * kin.max()
        bm, _ = oracle.lattice(c["rprimd"])
        d = np.array([1, -2, 3])
        a = 2 * np.pi * d @ bm
        ref = np.array([oracle.kin_of(c["rprimd"], k, m + d) for m in kg])
        assert np.max(np.abs(oracle.kin_vecpot(c["rprimd"], k, kg, a) - ref)) < 1e-12 * ref.max()
    c = config("c1m"); kg, ig, kin = sphere("c1m")
    L = c["rprimd"][0][0]; a = np.array([0.3, -0.1, 0.25])
    q = 2 * np.pi / L * (kg + np.asarray(c["kpt"][0])[None, :]) + a[None, :]
    ka = oracle.kin_vecpot(c["rprimd"], c["kpt"][0], kg, a)
    assert np.max(np.abs(ka - 0.5 * np.sum(q * q, axis=1))) < 1e-13 * ka.max()
    psi = rand_c((2, len(kg)), 4)
    out = oracle.apply_h(c, 0, kg, ig, ka, psi, terms=oracle.KIN)
    assert rel_err(out, ka[None, :] * psi) < 1e-15


def test_meta_gga_term_pins():
    """-1/2 div(v_tau grad) (Eq. 8): constant v_tau = c gives c * 1/2|k+G|^2 psi; the dense definition
    H_tau[m, m'] = 1/2 q(m).q(m') vt~[(m - m') mod n] built from the oracle's Fourier coefficients of v_tau;
    Hermiticity."""
    import oracle
    from util import config, sphere, rand_c, rel_err
    for name in ("c0", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        n = c["ngfft"]; npw = len(kg)
        psi = rand_c((2, npw), 17)
        const = np.full((n[2], n[1], n[0]), 0.37)
        assert rel_err(oracle.apply_mgga(c, 0, kg, ig, psi, const, method=1), 0.37 * kin[None, :] * psi) < 1e-12
        rng = np.random.default_rng(2)
        vt = 0.5 + 0.2 * rng.standard_normal((n[2], n[1], n[0]))
        got = oracle.apply_mgga(c, 0, kg, ig, psi, vt, method=1)
        vtil = oracle.vtilde(vt).reshape(-1)                       # [(d3*n2 + d2)*n1 + d1]
        bm, _ = oracle.lattice(c["rprimd"])
        q = 2 * np.pi * (kg + np.asarray(c["kpt"][0])[None, :]) @ bm
        d = (kg[:, None, :] - kg[None, :, :]) % np.array(n)[None, None, :]
        H = 0.5 * (q @ q.T) * vtil[(d[..., 2] * n[1] + d[..., 1]) * n[0] + d[..., 0]]
        assert rel_err(got, psi @ H.T) < 1e-12
        assert np.max(np.abs(H - H.conj().T)) < 1e-13 * np.max(np.abs(H))
