"""Pins of the oracle's projectors and non-local term (Eq. 26, PAPER.md :470; readings 6-11)."""
import numpy as np
import pytest

import oracle
import synth
from util import config, sphere, rel_err, rand_c


def test_spline_reproduces_a_cubic_exactly_and_the_recipe_closely():
    dq, nq = 0.01, 400
    q = dq * np.arange(nq)
    f = 1 + 2 * q - 3 * q ** 2 + 0.5 * q ** 3; f2 = -6 + 3 * q      # exact pair for a cubic
    for x in (0.0, 0.0049, 1.23456, 3.985, 3.99):
        assert abs(oracle.spline(f, f2, dq, x) - (1 + 2 * x - 3 * x * x + 0.5 * x ** 3)) < 1e-13
    t = config("c0")["types"][0]
    for r, (l, rc) in enumerate(zip(t["rad_l"], t["rad_rc"])):
        for x in (0.0, 0.123456, 1.0, 2.71828, 3.9):
            ref = x ** l * np.exp(-x * x * rc * rc / 2)
            assert abs(oracle.spline(t["f"][r], t["f2"][r], t["dq"], x) - ref) < 2e-9


def test_ylm_axis_values_orthonormality_addition_theorem():
    s3 = np.sqrt(3 / (4 * np.pi))
    assert abs(oracle.ylm(0, 0, [1, 2, 3]) - 1 / (2 * np.sqrt(np.pi))) < 1e-16
    # l=1 order m=-1,0,1 <-> (y, z, x), no Condon-Shortley sign
    for m, axis in ((-1, [0, 2.0, 0]), (0, [0, 0, 2.0]), (1, [2.0, 0, 0])):
        assert abs(oracle.ylm(1, m, axis) - s3) < 1e-15
        assert abs(oracle.ylm(1, m, [-a for a in axis]) + s3) < 1e-15
    assert abs(oracle.ylm(2, 0, [0, 0, 1]) - 0.5 * np.sqrt(5 / np.pi)) < 1e-15
    assert abs(oracle.ylm(2, 2, [1, 0, 0]) - 0.25 * np.sqrt(15 / np.pi)) < 1e-15
    assert abs(oracle.ylm(2, -2, [1, 1, 0]) - 0.25 * np.sqrt(15 / np.pi)) < 1e-15
    assert abs(oracle.ylm(2, -1, [0, 1, 1]) - 0.25 * np.sqrt(15 / np.pi)) < 1e-15
    assert abs(oracle.ylm(2, 1, [1, 0, 1]) - 0.25 * np.sqrt(15 / np.pi)) < 1e-15
    assert oracle.ylm(1, 0, [0, 0, 0]) == 0.0 and oracle.ylm(2, 1, [0, 0, 0]) == 0.0
    # orthonormality on a Gauss-Legendre x uniform-phi quadrature
    x, w = np.polynomial.legendre.leggauss(16)
    phi = 2 * np.pi * (np.arange(32) + 0.5) / 32
    lm = [(l, m) for l in range(3) for m in range(-l, l + 1)]
    Y = np.array([[[oracle.ylm(l, m, [np.sqrt(1 - c * c) * np.cos(p), np.sqrt(1 - c * c) * np.sin(p), c])
                    for p in phi] for c in x] for l, m in lm])
    G = np.einsum("aij,bij,i->ab", Y, Y, w) * (2 * np.pi / 32)
    np.testing.assert_allclose(G, np.eye(9), atol=1e-14)
    # addition theorem (independent of sign/order conventions)
    rng = np.random.default_rng(0)
    P = [lambda t: 1.0, lambda t: t, lambda t: 1.5 * t * t - 0.5]
    for _ in range(5):
        a = rng.standard_normal(3); b = rng.standard_normal(3)
        ct = a @ b / np.linalg.norm(a) / np.linalg.norm(b)
        for l in range(3):
            s = sum(oracle.ylm(l, m, a) * oracle.ylm(l, m, b) for m in range(-l, l + 1))
            assert abs(s - (2 * l + 1) / (4 * np.pi) * P[l](ct)) < 1e-15


def test_projector_table_against_recipe_written_in_numpy():
    """p = q^l exp(-q^2 rc^2/2) Y_lm(q^) exp(-i (k+G).R) (BASELINE.json), to the spline accuracy."""
    for name in ("c0", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        P = oracle.projector_table(c, 0, kg)
        Bm = np.linalg.inv(c["rprimd"]).T
        t = kg + c["kpt"][0]
        q = 2 * np.pi * t @ Bm; qn = np.linalg.norm(q, axis=1)
        np.testing.assert_allclose(0.5 * qn ** 2, kin, rtol=1e-13)
        row = 0
        for a in range(c["natom"]):
            T = c["types"][c["typat"][a]]
            R = c["xred"][a] @ c["rprimd"]
            phase = np.exp(-1j * (q @ R))
            for i in range(T["nlmn"]):
                l, m, ir = T["l"][i], T["m"][i], T["irad"][i]
                rc = T["rad_rc"][ir]
                Y = np.array([oracle.ylm(l, m, v) for v in q])
                ref = qn ** l * np.exp(-qn ** 2 * rc * rc / 2) * Y * phase
                np.testing.assert_allclose(P[row], ref, atol=5e-9)
                row += 1
        assert row == c["nproj"]
        assert oracle.max_q(c, 0, kg) == pytest.approx(qn.max(), rel=1e-14)


def test_nonlocal_equals_numpy_reduction_and_cprj():
    for name in ("c0", "aniso", "c4m"):
        c = config(name); kg, ig, kin = sphere(name)
        psi = rand_c((3, len(kg)), 7)
        P = oracle.projector_table(c, 0, kg)
        D = np.zeros((c["nproj"], c["nproj"]))
        r = 0
        for a in range(c["natom"]):
            nl = c["types"][c["typat"][a]]["nlmn"]
            D[r:r + nl, r:r + nl] = c["dij"][a, :nl, :nl]; r += nl
        out, cp = oracle.nonlocal_apply(c, 0, kg, psi, want_cprj=True)
        cref = P.conj() @ psi.T
        assert rel_err(cp.T, cref.T) < 1e-13
        assert rel_err(out, (P.T @ (D @ cref)).T) < 1e-13
        Hnl = oracle.dense_h(c, 0, kg, kin, terms=oracle.NL)
        assert rel_err(psi @ Hnl.T, out) < 1e-13
        assert abs(Hnl - Hnl.conj().T).max() < 1e-14 * abs(Hnl).max()


def test_single_s_projector_rank_and_zero_d():
    c = dict(config("c0"))
    kg, ig, kin = sphere("c0")
    c["natom"] = 1; c["xred"] = np.zeros((1, 3)); c["typat"] = np.zeros(1, np.int32); c["nproj"] = 8
    d = np.zeros((1, 8, 8)); d[0, 0, 0] = 0.7
    P = oracle.projector_table(c, 0, kg)
    p = P[0]
    out = oracle.nonlocal_apply(c, 0, kg, p[None], dij=d)[0]
    np.testing.assert_allclose(out, 0.7 * np.vdot(p, p) * p, rtol=1e-13)       # V_nl p = D <p|p> p
    c = config("c0")
    P = oracle.projector_table(c, 0, kg)
    x = rand_c(len(kg), 1)
    Q, _ = np.linalg.qr(P.T)                                                   # span of projectors
    x = x - Q @ (Q.conj().T @ x)
    out = oracle.nonlocal_apply(c, 0, kg, x[None])[0]
    assert np.linalg.norm(out) < 1e-12 * np.linalg.norm(x)                     # rank(V_nl) <= nproj
    assert np.linalg.matrix_rank(oracle.dense_h(c, 0, kg, kin, terms=oracle.NL), tol=1e-10) <= c["nproj"]
    assert np.all(oracle.nonlocal_apply(c, 0, kg, rand_c((2, len(kg)), 3), dij=np.zeros_like(c["dij"])) == 0)


def test_overlap_operator_pins():
    """S = 1 + sum |p> s <p| (PAPER.md :473): numpy reduction I + P^T s conj(P), closed form on one projector,
    Hermiticity, s = 0 -> identity, and pad columns returned as zero."""
    for name in ("c0", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        npw = len(kg)
        rng = np.random.default_rng(5)
        sij = rng.standard_normal(c["dij"].shape) * 0.3
        sij = 0.5 * (sij + sij.transpose(0, 2, 1))
        psi = rand_c((3, npw + 2), 11)
        out = oracle.apply_s(c, 0, kg, psi, sij)
        P = oracle.projector_table(c, 0, kg)
        Sm = np.zeros((c["nproj"], c["nproj"]))
        r = 0
        for a in range(c["natom"]):
            nl = c["types"][c["typat"][a]]["nlmn"]
            Sm[r:r + nl, r:r + nl] = sij[a, :nl, :nl]; r += nl
        x = psi[:, :npw]
        ref = x + (P.T @ (Sm @ (P.conj() @ x.T))).T
        assert rel_err(out[:, :npw], ref) < 1e-13
        assert np.all(out[:, npw:] == 0)
        phi = rand_c((1, npw), 12)
        sphi = oracle.apply_s(c, 0, kg, phi, sij)
        lhs = np.vdot(phi[0], out[0, :npw]); rhs = np.vdot(sphi[0], x[0])
        assert abs(lhs - rhs) < 1e-12 * abs(lhs)                              # <phi|S psi> = <S phi|psi>
        assert rel_err(oracle.apply_s(c, 0, kg, x, np.zeros_like(sij)), x) == 0.0
        assert rel_err(oracle.cprj(c, 0, kg, x).T, (P.conj() @ x.T).T) < 1e-13
    c = dict(config("c0")); kg, ig, kin = sphere("c0")
    c["natom"] = 1; c["xred"] = np.zeros((1, 3)); c["typat"] = np.zeros(1, np.int32); c["nproj"] = 8
    s1 = np.zeros((1, 8, 8)); s1[0, 0, 0] = 0.4
    p = oracle.projector_table(c, 0, kg)[0]
    np.testing.assert_allclose(oracle.apply_s(c, 0, kg, p[None], s1)[0], (1 + 0.4 * np.vdot(p, p).real) * p, rtol=1e-13)
