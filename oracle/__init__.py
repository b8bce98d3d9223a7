"""ctypes wrapper of the CPU oracle (oracle/oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference`
legs may import this package.  It imports nothing from paper_2507_08578_b200 and the
product never imports it.  The arithmetic of the hot path (sphere, FFT tiers, projector table, non-local loops, dense H) is in oracle.c and this
file marshals numpy arrays for it; the restatements of the NEXT rows (kin_vecpot, density, tau_density, apply_mgga,
chebyshev_filter, apply_s, cprj, and the Gamma-storage / spinor functions) are plain numpy in this file, each with its own pin in tests/.

`cfg` arguments are the dicts of synth.make_config (input data only).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
BUILD_CMD = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
             _SRC, "-o", _LIB, "-lm"]


def build(force=False):
    """Compile oracle.c -> liboracle.so (in-tree, git-ignored) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        cmd = list(BUILD_CMD)
        cmd[cmd.index(_LIB)] = tmp
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_sphere.restype = C.c_int64
        _lib.orc_kin.restype = C.c_double
        _lib.orc_spline.restype = C.c_double
        _lib.orc_ylm.restype = C.c_double
        _lib.orc_max_q.restype = C.c_double
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _i(a):
    return a.ctypes.data_as(_ip) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def num_threads():
    return lib().orc_num_threads()


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))


# ---------------------------------------------------------------- lattice / sphere
def lattice(rprimd):
    bm = np.zeros(9); gm = np.zeros(9)
    lib().orc_lattice(_d(_f64(rprimd).ravel()), _d(bm), _d(gm))
    return bm.reshape(3, 3), gm.reshape(3, 3)


def kin_of(rprimd, k, m):
    _, gm = lattice(rprimd)
    return lib().orc_kin(_d(gm.ravel()), _d(_f64(k)), C.c_int(int(m[0])), C.c_int(int(m[1])), C.c_int(int(m[2])))


def sphere(rprimd, k, ecut, ngfft):
    """Brute-force sphere: returns (kg[npw,3] int32, igfft[npw] int32, kin[npw] float64)."""
    r = _f64(rprimd).ravel(); kk = _f64(k); n = _i32(ngfft)
    npw = lib().orc_sphere(_d(r), _d(kk), C.c_double(ecut), _i(n), None, None, None, C.c_int64(0))
    kg = np.zeros((npw, 3), np.int32); ig = np.zeros(npw, np.int32); kin = np.zeros(npw)
    lib().orc_sphere(_d(r), _d(kk), C.c_double(ecut), _i(n), _i(kg), _i(ig), _d(kin), C.c_int64(npw))
    return kg, ig, kin


def sphere_extent(rprimd, k, ecut, ngfft):
    mn = np.zeros(3, np.int32); mx = np.zeros(3, np.int32)
    fits = lib().orc_sphere_extent(_d(_f64(rprimd).ravel()), _d(_f64(k)), C.c_double(ecut), _i(_i32(ngfft)), _i(mn), _i(mx))
    return bool(fits), mn, mx


# ---------------------------------------------------------------- transforms
def dft1d(x, sign, method):
    x = np.ascontiguousarray(x, np.complex128); out = np.zeros_like(x)
    lib().orc_dft1d(C.c_int(len(x)), C.c_int(sign), C.c_int(method), _d(x.view(np.float64)), _d(out.view(np.float64)))
    return out


def dft3d(box, sign, method):
    """box[n3][n2][n1] complex -> transformed copy (no scaling)."""
    b = np.array(box, dtype=np.complex128, order="C")
    n = _i32(b.shape[::-1])
    lib().orc_dft3d(_i(n), C.c_int(sign), C.c_int(method), _d(b.view(np.float64)))
    return b


def g2r(ngfft, igfft, c, method=2):
    n = _i32(ngfft); c = np.ascontiguousarray(c, np.complex128)
    box = np.zeros((n[2], n[1], n[0]), np.complex128)
    lib().orc_g2r(_i(n), C.c_int64(len(igfft)), _i(_i32(igfft)), _d(c.view(np.float64)), C.c_int(method), _d(box.view(np.float64)))
    return box


def vtilde(V):
    V = _f64(V); n = _i32(V.shape[::-1]); out = np.zeros(V.shape, np.complex128)
    lib().orc_vtilde(_i(n), _d(V), _d(out.view(np.float64)))
    return out


# ---------------------------------------------------------------- projectors
def spline(f, f2, dq, q):
    f = _f64(f); f2 = _f64(f2)
    return lib().orc_spline(C.c_int(len(f)), C.c_double(dq), _d(f), _d(f2), C.c_double(q))


def ylm(l, m, v):
    return lib().orc_ylm(C.c_int(l), C.c_int(m), C.c_double(v[0]), C.c_double(v[1]), C.c_double(v[2]))


class _Proj:
    """Flattened per-type projector metadata in the padded layout oracle.c expects."""

    def __init__(self, cfg, ik):
        ty = cfg["types"]
        self.keep = []
        self.lmax = cfg["nlmn_max"]; self.ntypat = len(ty)
        self.nrad_max = max(t["nrad"] for t in ty); self.nq_max = max(t["nq"] for t in ty)
        self.nlmn = _i32([t["nlmn"] for t in ty])
        self.l = np.zeros((self.ntypat, self.lmax), np.int32); self.m = self.l.copy(); self.ir = self.l.copy()
        self.f = np.zeros((self.ntypat, self.nrad_max, self.nq_max)); self.f2 = self.f.copy()
        for t, T in enumerate(ty):
            self.l[t, :T["nlmn"]] = T["l"]; self.m[t, :T["nlmn"]] = T["m"]; self.ir[t, :T["nlmn"]] = T["irad"]
            self.f[t, :T["nrad"], :T["nq"]] = T["f"]; self.f2[t, :T["nrad"], :T["nq"]] = T["f2"]
        self.nq = _i32([t["nq"] for t in ty]); self.dq = _f64([t["dq"] for t in ty])
        self.rprimd = _f64(cfg["rprimd"]).ravel(); self.k = _f64(cfg["kpt"][ik])
        self.typat = _i32(cfg["typat"]); self.xred = _f64(cfg["xred"]).ravel()
        self.natom = cfg["natom"]

    def args(self):
        return (_d(self.rprimd), _d(self.k), C.c_int(self.natom), _i(self.typat), _d(self.xred),
                C.c_int(self.ntypat), C.c_int(self.lmax), _i(self.nlmn), _i(self.l), _i(self.m), _i(self.ir),
                C.c_int(self.nrad_max), C.c_int(self.nq_max), _i(self.nq), _d(self.dq), _d(self.f), _d(self.f2))


def projector_table(cfg, ik, kg):
    """P[nproj][npw] complex128 (materialised; small cases only)."""
    P = _Proj(cfg, ik); kg = _i32(kg)
    out = np.zeros((cfg["nproj"], len(kg)), np.complex128)
    lib().orc_projector_table(*P.args(), C.c_int64(len(kg)), _i(kg), _d(out.view(np.float64)))
    return out


def max_q(cfg, ik, kg):
    kg = _i32(kg)
    return lib().orc_max_q(_d(_f64(cfg["rprimd"]).ravel()), _d(_f64(cfg["kpt"][ik])), C.c_int64(len(kg)), _i(kg))


def nonlocal_apply(cfg, ik, kg, psi, dij=None, want_cprj=False):
    """V_nl psi for psi[nband][npw]; returns out (and cprj[nproj][nband] if asked)."""
    P = _Proj(cfg, ik); kg = _i32(kg)
    psi = np.ascontiguousarray(psi, np.complex128); nb, ld = psi.shape
    out = np.zeros_like(psi)
    dij = _f64(cfg["dij"] if dij is None else dij)
    cp = np.zeros((cfg["nproj"], nb), np.complex128) if want_cprj else None
    lib().orc_nonlocal_apply(*P.args(), _d(dij), C.c_int64(len(kg)), _i(kg), C.c_int(nb), C.c_int64(ld),
                             _d(psi.view(np.float64)), _d(out.view(np.float64)),
                             _d(cp.view(np.float64)) if want_cprj else None)
    return (out, cp) if want_cprj else out


def kin_vecpot(rprimd, k, kg, a_cart):
    """1/2 |k + G + A|^2 per plane wave (PAPER.md :340, velocity gauge: -i grad -> -i grad + A): q = 2 pi (k + m) Bm
    Cartesian (reading 1), A Cartesian in atomic units.  Plain numpy; pass the result to apply_h as `kin`."""
    bm, _ = lattice(rprimd)
    q = 2.0 * np.pi * (np.asarray(kg, float) + np.asarray(k, float)[None, :]) @ np.asarray(bm, float).reshape(3, 3)
    q = q + np.asarray(a_cart, float)[None, :]
    return 0.5 * np.sum(q * q, axis=1)


def density(ngfft, igfft, psi, weights, method=2):
    """sum_b weights[b] |psi_b(r_j)|^2 on the FFT box, [n3][n2][n1] (Eq. 6, :140), with
    psi_b(r_j) = sum_G c_b(G) exp(+2 pi i G.r_j) by the oracle's own G->r transform (orc_g2r: scatter + T1/T2 DFT)."""
    n1, n2, n3 = [int(v) for v in ngfft]
    rho = np.zeros((n3, n2, n1))
    npw = len(igfft)
    for c, w in zip(np.asarray(psi, np.complex128), np.asarray(weights, float)):
        box = g2r(ngfft, igfft, c[:npw], method)
        rho += w * (box.real ** 2 + box.imag ** 2)
    return rho


def apply_mgga(cfg, ik, kg, igfft, psi, vtau, method=2):
    """Meta-GGA term of Eq. 8 (PAPER.md :152), -1/2 div(v_tau grad psi), on the plane-wave coefficients of
    psi(r) = sum_G c(G) e^{i(k+G).r}: grad -> i q with q = k + G Cartesian (2 pi (k + m) Bm, reading 1), so
    (H_tau c)(G) = 1/2 sum_d q_d(G) [Loc_{v_tau} (q_d c)](G), Loc_v = the local operator of reading 4 with V := v_tau
    (the oracle's own scatter / DFT / multiply / DFT / gather, orc_apply_h with terms = LOC)."""
    psi = np.ascontiguousarray(psi, np.complex128)
    npw = len(kg)
    bm, _ = lattice(cfg["rprimd"])
    q = 2.0 * np.pi * (np.asarray(kg, float) + np.asarray(cfg["kpt"][ik], float)[None, :]) @ np.asarray(bm, float).reshape(3, 3)
    out = np.zeros_like(psi)
    zero = np.zeros(npw)
    for d in range(3):
        x = psi.copy(); x[:, :npw] *= q[None, :, d]
        y = apply_h(cfg, ik, kg, igfft, zero, x, method=method, terms=LOC, vloc=vtau)
        out[:, :npw] += 0.5 * q[None, :, d] * y[:, :npw]
    return out


def tau_density(cfg, ik, kg, igfft, psi, weights, method=2):
    """Kinetic-energy density of PAPER.md Eq. 6 (:140): tau(r_j) = 1/2 sum_b w_b sum_d |d_d psi_b(r_j)|^2 with
    d_d psi(r) = sum_G i q_d(G) c(G) e^{i(k+G).r}, q = k + G Cartesian; |.|^2 drops the factor i and the Bloch phase, so
    each gradient component is a density() of the coefficients q_d c with weight w/2."""
    bm, _ = lattice(cfg["rprimd"])
    npw = len(kg)
    q = 2.0 * np.pi * (np.asarray(kg, float) + np.asarray(cfg["kpt"][ik], float)[None, :]) @ np.asarray(bm, float).reshape(3, 3)
    psi = np.asarray(psi, np.complex128)[:, :npw]
    out = 0.0
    for d in range(3):
        out = out + density(cfg["ngfft"], igfft, psi * q[None, :, d], 0.5 * np.asarray(weights, float), method)
    return out


def cprj(cfg, ik, kg, psi):
    """<p_a,i|psi_b> (PAPER.md :477 "coefficients c_a,i,n,k"), [nproj][nband] complex: step 1 of Eq. 26 (:470),
    as the streamed loops of orc_nonlocal_apply compute it."""
    return nonlocal_apply(cfg, ik, kg, psi, dij=np.zeros_like(_f64(cfg["dij"])), want_cprj=True)[1]


def apply_s(cfg, ik, kg, psi, sij):
    """S psi = psi + sum_a sum_ij |p_a,i> s^a_ij <p_a,j|psi>: PAPER.md :473, "the overlap operator S ... has the same
    structure" as the non-local operator of Eq. 26, so it is the definition's unit term plus orc_nonlocal_apply with
    s_ij in the place of D_ij.  psi [nband][ld >= npw]; columns >= npw are returned as 0."""
    psi = np.ascontiguousarray(psi, np.complex128)
    out = nonlocal_apply(cfg, ik, kg, psi, dij=sij)
    npw = len(kg)
    out[:, :npw] += psi[:, :npw]
    return out


# ---------------------------------------------------------------- whole operator
KIN, LOC, NL, ALL = 1, 2, 4, 7


def apply_h(cfg, ik, kg, igfft, kin, psi, method=2, terms=ALL, vloc=None, dij=None):
    """H psi for psi[nband][ld] (ld >= npw; columns >= npw ignored and returned as 0)."""
    P = _Proj(cfg, ik); kg = _i32(kg); igfft = _i32(igfft); kin = _f64(kin)
    psi = np.ascontiguousarray(psi, np.complex128); nb, ld = psi.shape
    V = _f64(cfg["vloc"] if vloc is None else vloc)
    dij = _f64(cfg["dij"] if dij is None else dij)
    n = _i32(cfg["ngfft"]); out = np.zeros_like(psi)
    lib().orc_apply_h(*P.args(), _d(dij), _i(n), _d(V), C.c_int64(len(kg)), _i(kg), _i(igfft), _d(kin),
                      C.c_int(nb), C.c_int64(ld), _d(psi.view(np.float64)), _d(out.view(np.float64)),
                      C.c_int(method), C.c_int(terms))
    return out


def chebyshev_filter(cfg, ik, kg, igfft, kin, psi, degree, center, halfwidth, method=2, terms=ALL, vloc=None, dij=None):
    """T_degree((H - center)/halfwidth) psi by the three-term recurrence, one apply_h per degree (PAPER.md :458
    "Chebyshev filtering algorithm", :489 mdeg_filter; the paper prints no formula -- DESIGN.md reading 21):
    T_0 = psi, T_1 = (H - c) T_0 / e, T_{j+1} = 2 (H - c) T_j / e - T_{j-1}."""
    psi = np.ascontiguousarray(psi, np.complex128)
    H = lambda x: apply_h(cfg, ik, kg, igfft, kin, x, method=method, terms=terms, vloc=vloc, dij=dij)
    npw = len(kg)
    t_prev = psi.copy(); t_prev[:, npw:] = 0
    if degree == 0:
        return psi.copy()
    t_cur = (H(t_prev) - center * t_prev) / halfwidth
    for _ in range(1, degree):
        t_next = 2.0 * (H(t_cur) - center * t_cur) / halfwidth - t_prev
        t_prev, t_cur = t_cur, t_next
    return t_cur


# ---------------------------------------------------------------- NEXT row 4: Gamma-point real-symmetry storage
# PAPER.md :407 ("time-reversal symmetry ... real-valued wave functions at the Gamma point"), SURVEY.md 8(f) 4.
# At k = 0 a psi(r) that is real has c(-G) = conj(c(G)), so only one of every pair +-G is stored (reading 26):
#   kept:  m3 > 0, or m3 = 0 and m2 > 0, or m3 = m2 = 0 and m1 >= 0   (in the order of the full list: ascending box index)
#   c(0) is real: the imaginary part of the stored c(0) is ignored on input and returned as 0.
# The operator in this storage is, by definition, the full operator applied to the symmetric vector and restricted again.
# It maps symmetric vectors to symmetric vectors only if H commutes with time reversal: V real (always) and, with
# the projector convention of reading 6 (no (-i)^l factor: p(-G) = (-1)^l conj(p(G))), D_ij = 0 whenever l_i + l_j is odd.
def gamma_half(kg):
    """(ih, ineg): positions in the full plane-wave list of the kept G and of their partners -G."""
    kg = np.asarray(kg, np.int64)
    keep = (kg[:, 2] > 0) | ((kg[:, 2] == 0) & (kg[:, 1] > 0)) | ((kg[:, 2] == 0) & (kg[:, 1] == 0) & (kg[:, 0] >= 0))
    ih = np.nonzero(keep)[0]
    pos = {tuple(m): i for i, m in enumerate(kg.tolist())}
    try:
        ineg = np.array([pos[(-m[0], -m[1], -m[2])] for m in kg[ih].tolist()], np.int64)
    except KeyError:
        raise ValueError("Gamma storage needs a sphere that holds -G for every G (k = 0, no unpaired Nyquist index)")
    return ih, ineg


def gamma_expand(kg, c_half):
    """c_half [nband][>= nhalf] -> the symmetric full vector [nband][npw]: c(G) = c_half, c(-G) = conj(c_half), c(0) real."""
    ih, ineg = gamma_half(kg)
    c_half = np.atleast_2d(np.asarray(c_half, np.complex128))
    full = np.zeros((c_half.shape[0], len(kg)), np.complex128)
    full[:, ineg] = np.conj(c_half[:, :len(ih)])
    full[:, ih] = c_half[:, :len(ih)]
    self_conj = ih[ih == ineg]                       # G = 0 (its own partner)
    full[:, self_conj] = full[:, self_conj].real
    return full


def gamma_dot(a_half, b_half, nhalf):
    """<a|b> of the two symmetric full vectors, from the stored halves: 2 Re sum_{G != 0, kept} conj(a) b + a(0) b(0)
    with the real parts of the stored a(0), b(0) (G = 0 is stored first: it has the smallest box index)."""
    a = np.asarray(a_half, np.complex128)[..., :nhalf]; b = np.asarray(b_half, np.complex128)[..., :nhalf]
    return 2.0 * np.sum((np.conj(a[..., 1:]) * b[..., 1:]).real, axis=-1) + a[..., 0].real * b[..., 0].real


def apply_h_gamma(cfg, kg, igfft, kin, psi_half, method=2, terms=ALL, vloc=None, dij=None, sym_tol=1e-12):
    """H psi in Gamma storage: psi_half [nband][ld >= nhalf] -> [nband][ld] (columns >= nhalf returned as 0).
    The definition: expand to the symmetric full vector, apply the full-sphere operator (apply_h), check that the
    result is symmetric (else H does not commute with time reversal and the storage is not closed), restrict."""
    if np.any(np.asarray(cfg["kpt"][0], float) != 0.0):
        raise ValueError("Gamma storage needs k = 0")
    ih, ineg = gamma_half(kg)
    psi_half = np.atleast_2d(np.asarray(psi_half, np.complex128))
    full = gamma_expand(kg, psi_half)
    out = apply_h(cfg, 0, kg, igfft, kin, full, method=method, terms=terms, vloc=vloc, dij=dij)
    asym = np.max(np.abs(out[:, ineg] - np.conj(out[:, ih]))) if len(ih) else 0.0
    if asym > sym_tol * max(1.0, np.max(np.abs(out))):
        raise ValueError("H does not commute with time reversal (D_ij couples projectors of different l-parity?): "
                         "asymmetry %.3e" % asym)
    res = np.zeros_like(psi_half)
    res[:, :len(ih)] = out[:, ih]
    res[:, 0] = res[:, 0].real          # G = 0: the symmetric result is real there (rounding residue dropped)
    return res


def chebyshev_filter_gamma(cfg, kg, igfft, kin, psi_half, degree, center, halfwidth, method=2, vloc=None, dij=None):
    """The recurrence of chebyshev_filter (reading 21) with apply_h_gamma as H; Im psi(0) of the input is
    ignored (reading 26), i.e. T_0 is the symmetric vector itself."""
    psi = np.array(np.atleast_2d(psi_half), np.complex128)
    if degree == 0:
        return psi
    ih, _ = gamma_half(kg)
    psi[:, len(ih):] = 0
    psi[:, 0] = psi[:, 0].real
    H = lambda x: apply_h_gamma(cfg, kg, igfft, kin, x, method=method, vloc=vloc, dij=dij)
    t_prev = psi
    t_cur = (H(t_prev) - center * t_prev) / halfwidth
    for _ in range(1, degree):
        t_prev, t_cur = t_cur, 2.0 * (H(t_cur) - center * t_cur) / halfwidth - t_prev
    return t_cur


# ---------------------------------------------------------------- NEXT row 4: two-component spinors
# PAPER.md :448 ("all types of magnetism": non-collinear magnetism, spin-orbit coupling); DESIGN.md
# reading 27.  psi = (psi_up, psi_dn), each a plane-wave vector on the same sphere.
#   H = kin (x) 1  +  FFT^-1[ V^{ss'}(r) FFT[psi_s'] ]  +  sum_a sum_ij sum_ss' |p_a,i> D^{a,ss'}_ij <p_a,j|
# V^{ss'}(r) is a Hermitian 2x2 matrix per grid point, given as four real fields v4 = (V_upup, V_dndn, Re V_updn,
# Im V_updn), V_dnup = conj(V_updn); D^{a,ss'}_ij is complex, [natom][2][2][lm][lm], Hermitian in ((s,i),(s',j)).
def apply_h_spinor(cfg, ik, kg, igfft, kin, psi, v4, dspin, method=2, terms=ALL):
    """psi [nband][2][ld >= npw] -> H psi, same shape; every step is the definition written out with the oracle's own
    scatter / DFT (g2r, dft3d), the materialised projector table (projector_table) and numpy contractions."""
    psi = np.ascontiguousarray(psi, np.complex128)
    nb, two, ld = psi.shape
    assert two == 2
    npw = len(kg)
    n1, n2, n3 = [int(v) for v in cfg["ngfft"]]
    N = n1 * n2 * n3
    out = np.zeros_like(psi)
    v4 = np.asarray(v4, float)
    vud = v4[2] + 1j * v4[3]
    if terms & KIN:
        out[:, :, :npw] += np.asarray(kin, float)[None, None, :] * psi[:, :, :npw]
    if terms & LOC:
        ig = np.asarray(igfft, np.int64)
        for b in range(nb):
            up = g2r(cfg["ngfft"], igfft, psi[b, 0, :npw], method)
            dn = g2r(cfg["ngfft"], igfft, psi[b, 1, :npw], method)
            phi_up = v4[0] * up + vud * dn
            phi_dn = np.conj(vud) * up + v4[1] * dn
            out[b, 0, :npw] += dft3d(phi_up, -1, method).reshape(-1)[ig] / N
            out[b, 1, :npw] += dft3d(phi_dn, -1, method).reshape(-1)[ig] / N
    if (terms & NL) and cfg["nproj"] > 0:
        P = projector_table(cfg, ik, kg)                                    # [nproj][npw]
        dspin = np.asarray(dspin, np.complex128)
        first = np.concatenate([[0], np.cumsum([cfg["types"][t]["nlmn"] for t in cfg["typat"]])])
        for b in range(nb):
            cp = np.stack([P.conj() @ psi[b, s, :npw] for s in range(2)])   # <p|psi_s>, [2][nproj]
            cq = np.zeros_like(cp)
            for a in range(cfg["natom"]):
                lo, hi = first[a], first[a + 1]
                nl = hi - lo
                for s in range(2):
                    for s2 in range(2):
                        cq[s, lo:hi] += dspin[a, s, s2, :nl, :nl] @ cp[s2, lo:hi]
            for s in range(2):
                out[b, s, :npw] += P.T @ cq[s]
    return out


def dense_h(cfg, ik, kg, kin, terms=ALL, vloc=None, dij=None):
    """T0: explicit H[npw][npw] complex128 in the plane-wave basis."""
    P = _Proj(cfg, ik); kg = _i32(kg); kin = _f64(kin)
    V = _f64(cfg["vloc"] if vloc is None else vloc)
    dij = _f64(cfg["dij"] if dij is None else dij)
    n = _i32(cfg["ngfft"]); npw = len(kg)
    H = np.zeros((npw, npw), np.complex128)
    lib().orc_dense_h(*P.args(), _d(dij), _i(n), _d(V), C.c_int64(npw), _i(kg), _d(kin), C.c_int(terms),
                      _d(H.view(np.float64)))
    return H


def dense_matvec(H, x):
    H = np.ascontiguousarray(H, np.complex128); x = np.ascontiguousarray(x, np.complex128)
    y = np.zeros_like(x)
    lib().orc_dense_matvec(C.c_int64(len(x)), _d(H.view(np.float64)), _d(x.view(np.float64)), _d(y.view(np.float64)))
    return y
