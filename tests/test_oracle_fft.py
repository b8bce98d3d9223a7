"""Pins of the oracle's transforms and local term (SURVEY.md 8(c) readings 4-5)."""
import numpy as np
import pytest

import oracle
from util import config, sphere, rel_err, rand_c


@pytest.mark.parametrize("n", [1, 2, 7, 20, 30, 32, 36, 72, 128, 180])
def test_dft1d_against_definition_and_numpy(n):
    x = rand_c(n, n)
    j = np.arange(n)
    for sign in (+1, -1):
        W = np.exp(sign * 2j * np.pi * np.outer(j, j) / n)         # the definition, written out
        ref = W @ x
        for method in (1, 2):
            assert rel_err(oracle.dft1d(x, sign, method), ref) < 1e-13
    assert rel_err(oracle.dft1d(x, -1, 2), np.fft.fft(x)) < 1e-13   # library reduction
    assert rel_err(oracle.dft1d(x, +1, 2), np.fft.ifft(x) * n) < 1e-13


@pytest.mark.parametrize("shape", [(5, 4, 6), (20, 24, 30), (32, 32, 32)])
def test_dft3d_against_numpy(shape):
    x = rand_c(shape, 3)
    for method in (1, 2):
        assert rel_err(oracle.dft3d(x, -1, method).ravel(), np.fft.fftn(x).ravel()) < 1e-13
        assert rel_err(oracle.dft3d(x, +1, method).ravel(), (np.fft.ifftn(x) * x.size).ravel()) < 1e-13
    # axis order: a delta along the fastest axis (n1 = shape[2]) gives a phase along that axis only
    d = np.zeros(shape, complex); d[0, 0, 1] = 1
    out = oracle.dft3d(d, +1, 2)
    np.testing.assert_allclose(out[2, 3, :], np.exp(2j * np.pi * np.arange(shape[2]) / shape[2]), atol=1e-14)


def test_parseval_and_expectation_value():
    c = config("c0"); kg, ig, kin = sphere("c0")
    psi = rand_c(len(kg), 1)
    box = oracle.g2r(c["ngfft"], ig, psi)
    N = box.size
    assert abs(np.sum(abs(psi) ** 2) - np.sum(abs(box) ** 2) / N) < 1e-12 * np.sum(abs(psi) ** 2)
    h = oracle.apply_h(c, 0, kg, ig, kin, psi[None], terms=oracle.LOC)[0]
    ev = np.vdot(psi, h)
    ref = np.sum(c["vloc"] * abs(box) ** 2) / N
    assert abs(ev - ref) < 1e-12 * abs(ref) and abs(ev.imag) < 1e-12 * abs(ref)


def test_constant_potential_single_plane_wave_eigenvalue():
    """BASELINE.json pin: a single plane wave under constant V has eigenvalue 1/2|k+G|^2 + V0."""
    for name in ("c0", "c1m", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        V0 = -0.37
        V = np.full(c["vloc"].shape, V0)
        for ipw in (0, len(kg) // 3, len(kg) - 1):
            e = np.zeros((1, len(kg)), complex); e[0, ipw] = 1.0
            h = oracle.apply_h(c, 0, kg, ig, kin, e, terms=oracle.KIN | oracle.LOC, vloc=V)
            np.testing.assert_allclose(h[0], (kin[ipw] + V0) * e[0], atol=1e-13)


def test_free_electron():
    c = config("c1m"); kg, ig, kin = sphere("c1m")
    psi = rand_c((3, len(kg)), 2)
    h = oracle.apply_h(c, 0, kg, ig, kin, psi, vloc=np.zeros(c["vloc"].shape), dij=np.zeros_like(c["dij"]))
    np.testing.assert_allclose(h, kin * psi, atol=1e-13)
    L = c["rprimd"][0, 0]                                            # cubic closed form
    np.testing.assert_allclose(kin, 0.5 * (2 * np.pi / L) ** 2 * np.sum((kg + c["kpt"][0]) ** 2, 1), rtol=1e-14)


def test_cosine_potential_is_a_pure_shift():
    """V(r) = 2v cos(2 pi g0.j/n + phi): H_loc delta_{m0} = v e^{+i phi} delta_{m0+g0} + v e^{-i phi} delta_{m0-g0}
    restricted to the sphere; phi != 0 distinguishes +g0 from -g0 (sign/axis/wrap of the transforms)."""
    c = config("aniso"); kg, ig, kin = sphere("aniso")
    n1, n2, n3 = c["ngfft"]
    v, phi = 0.8, 0.6
    index = {tuple(m): i for i, m in enumerate(kg)}
    j3, j2, j1 = np.meshgrid(np.arange(n3), np.arange(n2), np.arange(n1), indexing="ij")
    for g0 in ([1, 0, 0], [0, 2, 0], [0, 0, -3], [1, -2, 1]):
        V = 2 * v * np.cos(2 * np.pi * (g0[0] * j1 / n1 + g0[1] * j2 / n2 + g0[2] * j3 / n3) + phi)
        for m0 in ([0, 0, 0], [1, -1, 2], [-2, 1, 0]):
            e = np.zeros((1, len(kg)), complex); e[0, index[tuple(m0)]] = 1.0
            ref = np.zeros(len(kg), complex)
            p = tuple(np.add(m0, g0)); q = tuple(np.subtract(m0, g0))
            if p in index: ref[index[p]] += v * np.exp(1j * phi)
            if q in index: ref[index[q]] += v * np.exp(-1j * phi)
            for method in (1, 2):
                h = oracle.apply_h(c, 0, kg, ig, kin, e, method=method, terms=oracle.LOC, vloc=V)[0]
                np.testing.assert_allclose(h, ref, atol=1e-14)


def test_tiers_agree_dense_convolution_vs_dft_vs_fft_vs_numpy():
    for name in ("c0", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        psi = rand_c((2, len(kg)), 4)
        Hloc = oracle.dense_h(c, 0, kg, kin, terms=oracle.LOC)      # T0: V~[(m-m') mod n]
        t0 = psi @ Hloc.T
        t1 = oracle.apply_h(c, 0, kg, ig, kin, psi, method=1, terms=oracle.LOC)
        t2 = oracle.apply_h(c, 0, kg, ig, kin, psi, method=2, terms=oracle.LOC)
        assert rel_err(t1, t0) < 1e-13 and rel_err(t2, t1) < 1e-13
        n1, n2, n3 = c["ngfft"]                                     # numpy library reduction
        box = np.zeros((2, n3 * n2 * n1), complex); box[:, ig] = psi
        r = np.fft.ifftn(box.reshape(2, n3, n2, n1), axes=(1, 2, 3)) * (n1 * n2 * n3)
        back = np.fft.fftn(r * c["vloc"], axes=(1, 2, 3)).reshape(2, -1)[:, ig] / (n1 * n2 * n3)
        assert rel_err(t2, back) < 1e-13
        # V~ itself against numpy
        assert rel_err(oracle.vtilde(c["vloc"]).ravel(), (np.fft.fftn(c["vloc"]) / c["vloc"].size).ravel()) < 1e-13


def test_tight_box_heavy_wraparound():
    """Box that just holds the sphere (n_j = 2 m_max + 1): result still equals the cyclic convolution."""
    from util import config_over
    c = config_over("c0", ngfft=(9, 9, 9))
    kg, ig, kin = oracle.sphere(c["rprimd"], c["kpt"][0], c["ecut"], c["ngfft"])
    assert len(kg) == 283
    psi = rand_c((2, len(kg)), 6)
    t0 = psi @ oracle.dense_h(c, 0, kg, kin, terms=oracle.LOC).T
    t2 = oracle.apply_h(c, 0, kg, ig, kin, psi, terms=oracle.LOC)
    assert rel_err(t2, t0) < 1e-13


def test_density_pins():
    """n(r) = sum_b w_b |psi_b(r)|^2 (Eq. 6, :140): Parseval (mean over the box = sum_b w_b <psi_b|psi_b>),
    one plane wave -> constant w, two plane waves -> w (|a|^2 + |b|^2 + 2 Re(conj(a) b e^{2 pi i (m_b - m_a).j/n})),
    and the numpy ifftn reduction."""
    import oracle
    from util import config, sphere, rand_c
    for name in ("c0", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        n = c["ngfft"]; N = int(np.prod(n)); npw = len(ig)
        psi = rand_c((3, npw), 31); w = np.array([0.7, 1.3, 2.0])
        rho = oracle.density(n, ig, psi, w, method=1)
        assert rho.shape == (n[2], n[1], n[0]) and rho.min() >= 0
        assert abs(rho.sum() / N - np.sum(w * np.sum(np.abs(psi) ** 2, axis=1))) < 1e-12 * rho.sum() / N
        ref = np.zeros_like(rho)
        for cb, wb in zip(psi, w):
            box = np.zeros(N, complex); box[ig] = cb
            r = np.fft.ifftn(box.reshape(n[2], n[1], n[0])) * N
            ref += wb * np.abs(r) ** 2
        assert np.max(np.abs(rho - ref)) < 1e-12 * ref.max()
        assert np.max(np.abs(oracle.density(n, ig, psi, w, method=2) - rho)) < 1e-12 * rho.max()
        one = np.zeros((1, npw), complex); one[0, 5] = 0.6 - 0.8j
        assert np.max(np.abs(oracle.density(n, ig, one, [2.5]) - 2.5)) < 1e-13
        two = np.zeros((1, npw), complex); a, b = 0.5 + 0.2j, -0.3 + 0.9j
        two[0, 3] = a; two[0, 11] = b
        dm = kg[11] - kg[3]
        j3, j2, j1 = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
        ph = np.exp(2j * np.pi * (dm[0] * j1 / n[0] + dm[1] * j2 / n[1] + dm[2] * j3 / n[2]))
        ref2 = 1.5 * (abs(a) ** 2 + abs(b) ** 2 + 2 * np.real(np.conj(a) * b * ph))
        assert np.max(np.abs(oracle.density(n, ig, two, [1.5]) - ref2)) < 1e-13


def test_tau_density_pins():
    """tau(r) = 1/2 sum w |grad psi|^2 (Eq. 6): one plane wave -> the constant w * 1/2|k+G|^2; the box mean is
    sum_b w_b sum_G 1/2|k+G|^2 |c_b(G)|^2 (Parseval per gradient component)."""
    import oracle
    from util import config, sphere, rand_c
    for name in ("c0", "aniso"):
        c = config(name); kg, ig, kin = sphere(name)
        npw = len(ig); N = int(np.prod(c["ngfft"]))
        one = np.zeros((1, npw), complex); one[0, 7] = 0.6 - 0.8j
        assert np.max(np.abs(oracle.tau_density(c, 0, kg, ig, one, [2.0], method=1) - 2.0 * kin[7])) < 1e-12 * (1 + kin[7])
        psi = rand_c((3, npw), 41); w = np.array([0.4, 1.1, 0.9])
        tau = oracle.tau_density(c, 0, kg, ig, psi, w, method=1)
        ref = np.sum(w * np.sum(kin[None, :] * np.abs(psi) ** 2, axis=1))
        assert tau.min() >= 0 and abs(tau.sum() / N - ref) < 1e-12 * ref
