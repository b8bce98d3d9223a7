"""Pins of the NEXT-row-4 oracle restatements: Gamma-point real-symmetry storage (PAPER.md :407)
and two-component spinors (PAPER.md :448).  Each pin is something other than the function itself: golden counts,
reality of psi(r), the full-sphere operator, closed forms, Hermiticity, spin-rotation covariance."""
import os

import numpy as np
import pytest

import oracle
import synth
from util import config, sphere, rel_err, rand_c


def _golden_counts(golden_dir):
    out = {}
    with open(os.path.join(golden_dir, "sphere_counts.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                t = line.split()
                out[t[0]] = [int(v) for v in t[1:]]
    return out


# ------------------------------------------------------------------------------------------------ Gamma storage
@pytest.mark.parametrize("name", ["c0", "c2m", "c4m"])
def test_gamma_half_counts_and_pairing(name, golden_dir):
    """nhalf = (npw + 1)/2 against the survey's golden counts; every G is kept or its partner is, never both (but 0)."""
    kg, ig, kin = sphere(name)
    ih, ineg = oracle.gamma_half(kg)
    npw = _golden_counts(golden_dir)[name][0]
    assert len(kg) == npw and len(ih) == (npw + 1) // 2
    assert np.array_equal(kg[ineg], -kg[ih])
    both = np.intersect1d(ih, ineg)
    assert len(both) == 1 and np.all(kg[both[0]] == 0) and ih[0] == both[0]      # G = 0 is stored first
    assert len(np.union1d(ih, ineg)) == npw
    assert np.all(np.diff(ih) > 0)                                              # order of the full list
    assert np.array_equal(kin[ih].view(np.int64), kin[ineg].view(np.int64))     # |G| = |-G| bit for bit at k = 0


def test_gamma_counts_of_the_large_cells(golden_dir):
    """(npw + 1)/2 for c2 and c4 from the golden counts: 62 145 and 147 834 (sizes the GPU tests assert)."""
    g = _golden_counts(golden_dir)
    assert (g["c2"][0] + 1) // 2 == 62145 and (g["c4"][0] + 1) // 2 == 147834 and (g["c0"][0] + 1) // 2 == 142


@pytest.mark.parametrize("name", ["c0", "c4m"])
def test_gamma_expand_gives_a_real_field(name):
    """The symmetric vector is exactly the one whose psi(r) is real (pins the -G map and the conjugation)."""
    c = config(name); kg, ig, kin = sphere(name)
    ih, _ = oracle.gamma_half(kg)
    half = rand_c((1, len(ih)), 5)
    full = oracle.gamma_expand(kg, half)
    box = oracle.g2r(c["ngfft"], ig, full[0], 1 if name == "c0" else 2)
    assert np.max(np.abs(box.imag)) < 1e-13 * np.max(np.abs(box.real))
    assert full[0, ih[0]].imag == 0.0
    # and a generic (unsymmetric) vector does not
    box2 = oracle.g2r(c["ngfft"], ig, rand_c((len(kg),), 6), 1 if name == "c0" else 2)
    assert np.max(np.abs(box2.imag)) > 1e-2 * np.max(np.abs(box2.real))


def test_gamma_dot_is_the_full_inner_product():
    kg, ig, kin = sphere("c2m")
    ih, _ = oracle.gamma_half(kg)
    a = rand_c((3, len(ih)), 7); b = rand_c((3, len(ih)), 8)
    fa = oracle.gamma_expand(kg, a); fb = oracle.gamma_expand(kg, b)
    full = np.array([np.vdot(fa[i], fb[i]) for i in range(3)])
    assert np.max(np.abs(full.imag)) < 1e-12 * np.max(np.abs(full.real))
    assert np.allclose(oracle.gamma_dot(a, b, len(ih)), full.real, rtol=1e-13, atol=0)


@pytest.mark.parametrize("name", ["c0", "c2m"])
def test_gamma_operator_closed_forms_and_hermiticity(name):
    c = dict(config(name)); kg, ig, kin = sphere(name)
    ih, _ = oracle.gamma_half(kg)
    nh = len(ih)
    x = rand_c((3, nh), 9)
    m = 1 if name == "c0" else 2
    # constant V0, D = 0: (kin + V0) c on the stored half, Im (Hc)(0) = 0
    got = oracle.apply_h_gamma(c, kg, ig, kin, x, method=m, vloc=np.full_like(c["vloc"], 0.37), dij=np.zeros_like(c["dij"]))
    ref = (kin[ih] + 0.37)[None, :] * x
    ref[:, 0] = ref[:, 0].real
    assert rel_err(got, ref) < 1e-13 and np.all(got[:, 0].imag == 0)
    # whole operator with a time-reversal-compatible D: Hermitian in the real inner product of the storage
    d = synth.gamma_dij(c)
    h = oracle.apply_h_gamma(c, kg, ig, kin, x, method=m, dij=d)
    lhs = oracle.gamma_dot(x[0], h[1], nh); rhs = oracle.gamma_dot(h[0], x[1], nh)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    # real-linear: H(2 a - 3 b) = 2 Ha - 3 Hb  (complex scalars would leave the symmetric subspace)
    lin = oracle.apply_h_gamma(c, kg, ig, kin, (2.0 * x[0] - 3.0 * x[2])[None], method=m, dij=d)[0]
    assert rel_err(lin, 2.0 * h[0] - 3.0 * h[2]) < 1e-13


def test_gamma_storage_refuses_a_d_that_breaks_time_reversal():
    """With the random dense D_ij of the recipe (s and p projectors coupled) H psi of a real psi(r) is not real:
    the storage is not closed and the oracle says so; the parity-masked D passes (previous test)."""
    c = config("c0"); kg, ig, kin = sphere("c0")
    ih, _ = oracle.gamma_half(kg)
    x = rand_c((1, len(ih)), 10)
    with pytest.raises(ValueError, match="time reversal"):
        oracle.apply_h_gamma(c, kg, ig, kin, x, method=1)


def test_gamma_projections_are_real_up_to_i_power_l():
    """<p_i|psi> of a symmetric vector is real for even l and purely imaginary for odd l (p(-G) = (-1)^l conj p(G)):
    the identity behind a real-GEMM formulation."""
    c = config("c2m"); kg, ig, kin = sphere("c2m")
    ih, _ = oracle.gamma_half(kg)
    full = oracle.gamma_expand(kg, rand_c((2, len(ih)), 12))
    cp = oracle.cprj(c, 0, kg, full)                     # [nproj][nband]
    l = synth.projector_l(c)
    scale = np.max(np.abs(cp))
    assert np.max(np.abs(cp[l % 2 == 0].imag)) < 1e-13 * scale
    assert np.max(np.abs(cp[l % 2 == 1].real)) < 1e-13 * scale
    assert np.max(np.abs(cp[l % 2 == 1].imag)) > 1e-3 * scale


def test_gamma_chebyshev_closed_form_and_full_sphere_agreement():
    """Diagonal H (constant V, D = 0): T_n((kin + V0 - c)/e) c on the stored half, by numpy's chebval; and for the whole
    operator the Gamma recurrence equals the (pinned) full-sphere recurrence on the expanded vectors."""
    c = dict(config("c2m")); kg, ig, kin = sphere("c2m")
    ih, _ = oracle.gamma_half(kg)
    x = rand_c((2, len(ih)), 31)
    cen, e = 0.5 * kin.max() + 1.0, 0.5 * kin.max() + 0.5
    v0 = 0.37
    for deg in (0, 1, 5):
        got = oracle.chebyshev_filter_gamma(c, kg, ig, kin, x, deg, cen, e, vloc=np.full_like(c["vloc"], v0), dij=np.zeros_like(c["dij"]))
        coef = np.zeros(deg + 1); coef[deg] = 1.0
        x0 = x.copy()
        if deg > 0:
            x0[:, 0] = x0[:, 0].real
        ref = np.polynomial.chebyshev.chebval((kin[ih] + v0 - cen) / e, coef)[None, :] * x0
        assert rel_err(got, ref) < 1e-12
    d = synth.gamma_dij(c)
    got = oracle.chebyshev_filter_gamma(c, kg, ig, kin, x, 4, cen, e, dij=d)
    full = oracle.chebyshev_filter(c, 0, kg, ig, kin, oracle.gamma_expand(kg, x), 4, cen, e, dij=d)
    assert rel_err(got[:, 1:], full[:, ih][:, 1:]) < 1e-12 and np.max(np.abs(got[:, 0].imag)) == 0


# ------------------------------------------------------------------------------------------------ spinors
def _spin_diag(c):
    v4 = np.stack([c["vloc"], c["vloc"], np.zeros_like(c["vloc"]), np.zeros_like(c["vloc"])])
    d = np.zeros((c["natom"], 2, 2, c["nlmn_max"], c["nlmn_max"]), np.complex128)
    d[:, 0, 0] = c["dij"]; d[:, 1, 1] = c["dij"]
    return v4, d


@pytest.mark.parametrize("name", ["c0", "aniso"])
def test_spinor_reduces_to_two_scalar_applications(name):
    """Spin-diagonal V and D: the spinor operator is the (pinned) scalar operator on each component."""
    c = config(name); kg, ig, kin = sphere(name)
    psi = rand_c((2, 2, len(kg) + 3), 21)
    v4, d = _spin_diag(c)
    for terms in (oracle.ALL, oracle.KIN, oracle.LOC, oracle.NL):
        got = oracle.apply_h_spinor(c, 0, kg, ig, kin, psi, v4, d, method=1, terms=terms)
        for s in range(2):
            ref = oracle.apply_h(c, 0, kg, ig, kin, psi[:, s], method=1, terms=terms)
            assert rel_err(got[:, s], ref) < 1e-13
        assert np.all(got[:, :, len(kg):] == 0)


def test_spinor_uniform_field_closed_form():
    """Constant 2x2 V, D = 0: (H psi)_s(G) = kin psi_s + sum_s' V^{ss'} psi_s'(G); V_updn = Bx - i By decides the sign
    convention of the fourth field."""
    c = config("c0"); kg, ig, kin = sphere("c0")
    psi = rand_c((1, 2, len(kg)), 22)
    one = np.ones_like(c["vloc"])
    vuu, vdd, vre, vim = 0.3, -0.2, 0.11, 0.07
    v4 = np.stack([vuu * one, vdd * one, vre * one, vim * one])
    d = np.zeros((c["natom"], 2, 2, c["nlmn_max"], c["nlmn_max"]), np.complex128)
    got = oracle.apply_h_spinor(c, 0, kg, ig, kin, psi, v4, d, method=1)
    vud = vre + 1j * vim
    ref = np.empty_like(psi)
    ref[:, 0] = kin * psi[:, 0] + vuu * psi[:, 0] + vud * psi[:, 1]
    ref[:, 1] = kin * psi[:, 1] + np.conj(vud) * psi[:, 0] + vdd * psi[:, 1]
    assert rel_err(got.reshape(1, -1), ref.reshape(1, -1)) < 1e-13


@pytest.mark.parametrize("name", ["c0", "c3k2"])
def test_spinor_hermiticity_and_spin_rotation_covariance(name):
    c = config(name); ik = c["nkpt"] - 1
    kg, ig, kin = sphere(name, ik)
    v4, d = synth.spinor_inputs(c)
    psi = rand_c((2, 2, len(kg)), 23)
    m = 1 if name == "c0" else 2
    h = oracle.apply_h_spinor(c, ik, kg, ig, kin, psi, v4, d, method=m)
    a = np.vdot(psi[0], h[1]); b = np.vdot(h[0], psi[1])
    assert abs(a - b) < 1e-12 * abs(a)
    # global SU(2) rotation U: psi -> U psi, V -> U V U^+, D -> U D U^+  =>  H psi -> U H psi (pins the s, s' order of
    # v4 and dspin against each other and against psi's component order)
    th, ph = 0.7, 1.9
    U = np.array([[np.cos(th / 2), -np.exp(-1j * ph) * np.sin(th / 2)], [np.exp(1j * ph) * np.sin(th / 2), np.cos(th / 2)]])
    V = np.empty((2, 2) + v4.shape[1:], np.complex128)
    V[0, 0] = v4[0]; V[1, 1] = v4[1]; V[0, 1] = v4[2] + 1j * v4[3]; V[1, 0] = v4[2] - 1j * v4[3]
    Vr = np.einsum("ab,bc...,dc->ad...", U, V, U.conj())
    assert np.max(np.abs(Vr[0, 0].imag)) < 1e-14 and np.max(np.abs(Vr[1, 0] - Vr[0, 1].conj())) < 1e-14
    v4r = np.stack([Vr[0, 0].real, Vr[1, 1].real, Vr[0, 1].real, Vr[0, 1].imag])
    dr = np.einsum("ab,xbcij,dc->xadij", U, d, U.conj())
    psir = np.einsum("ab,nbg->nag", U, psi)
    hr = oracle.apply_h_spinor(c, ik, kg, ig, kin, psir, v4r, dr, method=m)
    assert rel_err(hr.reshape(2, -1), np.einsum("ab,nbg->nag", U, h).reshape(2, -1)) < 1e-12
