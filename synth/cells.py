"""The five BASELINE.json cells (c0..c4) plus the small parity cells of SURVEY.md 8(c).

Everything here is *input data*: lattices, atoms, k-points, radial tables,
D_ij, V_loc(r) and the psi coefficients.  The plane-wave sphere, the kinetic
energies and everything downstream are computed by the oracle and by the CUDA
library independently; `gen_psi` therefore takes `kin` (1/2|k+G|^2 per plane
wave, in the caller's plane-wave order) as an argument.

Readings of BASELINE.json that this file fixes (all listed in DESIGN.md):
  * V_loc noise: nu(G) = amp*exp(-|G|^2/4)*xi(G), xi = N^-1/2 * DFT of a white
    N(0,1) field on the box (the "literal" reading of SURVEY.md 8(d)).
  * "width" w of the Gaussians is the denominator: depth*exp(-|r-R|^2/w).
  * radial tables: F(q) = q^l exp(-q^2 rc^2/2) on a uniform grid dq = 0.01 with
    the analytic second derivative (SURVEY.md 8(c) reading 7).
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from . import rng

BASE_SEED = 20250708
STREAM_PSI, STREAM_VNOISE, STREAM_DIJ = 1, 2, 3

CONFIG_NAMES = ("c0", "c1", "c2", "c3", "c4",
                "c1m", "c2m", "c4m", "aniso", "c3k2", "aniso8", "anisok3", "aniso5t")

_DIAMOND_SITES = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                           [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]])
# order of SURVEY.md 8(d): the 4 FCC sites, each followed by its (1/4,1/4,1/4) partner
_DIAMOND_SITES = _DIAMOND_SITES[[0, 4, 1, 5, 2, 6, 3, 7]]
_FCC_SITES = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])


def config_seed(name):
    """seed = 20250708 + config number; variants get their own."""
    return BASE_SEED + CONFIG_NAMES.index(name)


# ----------------------------------------------------------------------------
# projector "pseudopotential" tables (per atom type)
# ----------------------------------------------------------------------------
def _radial(l, rc, q):
    """F(q) = q^l exp(-alpha q^2), alpha = rc^2/2, and d2F/dq2 (analytic)."""
    al = 0.5 * rc * rc
    e = np.exp(-al * q * q)
    if l == 0:
        return e, (4 * al * al * q * q - 2 * al) * e
    if l == 1:
        return q * e, (4 * al * al * q ** 3 - 6 * al * q) * e
    if l == 2:
        return q * q * e, (2 - 10 * al * q * q + 4 * al * al * q ** 4) * e
    raise ValueError(l)


def _proj_type(kind, qmax, dq=0.01):
    """One atom type: (l, m, irad) per projector and the radial tables."""
    if kind == "Si":          # l=0,1 x 2 radial (rc 1.0, 0.7) -> 8 projectors
        rads = [(0, 1.0), (0, 0.7), (1, 1.0), (1, 0.7)]
        lmn = [(0, 0, 0), (0, 0, 1)] + [(1, m, 2) for m in (-1, 0, 1)] + [(1, m, 3) for m in (-1, 0, 1)]
    elif kind == "Al":        # l=0,1,2 x 1 radial (rc 1.2) -> 9 projectors
        rads = [(0, 1.2), (1, 1.2), (2, 1.2)]
        lmn = [(0, 0, 0)] + [(1, m, 1) for m in (-1, 0, 1)] + [(2, m, 2) for m in (-2, -1, 0, 1, 2)]
    elif kind == "Sip":       # test-only second light type: l=0 (rc 0.9), l=1 (rc 0.8) -> 4 projectors
        rads = [(0, 0.9), (1, 0.8)]
        lmn = [(0, 0, 0)] + [(1, m, 1) for m in (-1, 0, 1)]
    else:
        raise ValueError(kind)
    nq = int(np.ceil(1.05 * qmax / dq)) + 2
    q = dq * np.arange(nq)
    f = np.empty((len(rads), nq))
    f2 = np.empty((len(rads), nq))
    for r, (l, rc) in enumerate(rads):
        f[r], f2[r] = _radial(l, rc, q)
    return dict(kind=kind, nlmn=len(lmn),
                l=np.array([t[0] for t in lmn], np.int32),
                m=np.array([t[1] for t in lmn], np.int32),
                irad=np.array([t[2] for t in lmn], np.int32),
                nrad=len(rads), nq=nq, dq=dq, f=f, f2=f2,
                rad_l=[r[0] for r in rads], rad_rc=[r[1] for r in rads])


# ----------------------------------------------------------------------------
# V_loc(r)
# ----------------------------------------------------------------------------
def _vloc_gauss(rprimd, ngfft, xred, depth, w):
    n1, n2, n3 = ngfft
    A = np.asarray(rprimd, float)
    diag = np.allclose(A, np.diag(np.diag(A)), atol=0, rtol=0)
    if diag:                                   # separable product of 1-D image sums
        g = []
        for c, n in enumerate((n1, n2, n3)):
            d = np.arange(n)[None, :] / n - xred[:, c][:, None]
            d = d - np.floor(d + 0.5)           # wrap to [-1/2, 1/2)
            s = sum(np.exp(-((A[c, c] * (d + t)) ** 2) / w) for t in (-1, 0, 1))
            g.append(s)                         # [natom][n_c]
        gx, gy, gz = g
        yx = (gy[:, :, None] * gx[:, None, :]).reshape(len(xred), n2 * n1)
        return depth * (gz.T @ yx).reshape(n3, n2, n1)
    V = np.zeros((n3, n2, n1))
    j3, j2, j1 = np.meshgrid(np.arange(n3) / n3, np.arange(n2) / n2, np.arange(n1) / n1, indexing="ij")
    for x in xred:
        d = np.stack([j1 - x[0], j2 - x[1], j3 - x[2]], axis=-1)
        d = d - np.floor(d + 0.5)
        for t1 in (-1, 0, 1):
            for t2 in (-1, 0, 1):
                for t3 in (-1, 0, 1):
                    r = (d + np.array([t1, t2, t3])) @ A      # Cartesian = reduced . rows a_i
                    V += depth * np.exp(-np.sum(r * r, axis=-1) / w)
    return V


def _vloc_noise(rprimd, ngfft, amp, seed):
    n1, n2, n3 = ngfft
    N = n1 * n2 * n3
    wn = rng.normals(seed, STREAM_VNOISE, np.arange(N, dtype=np.uint64)).reshape(n3, n2, n1)
    xi = np.fft.fftn(wn) / np.sqrt(N)
    Bm = np.linalg.inv(np.asarray(rprimd, float)).T                 # rows b_i, a_i.b_j = delta_ij
    m3, m2, m1 = np.meshgrid(np.fft.fftfreq(n3) * n3, np.fft.fftfreq(n2) * n2,
                             np.fft.fftfreq(n1) * n1, indexing="ij")
    G = 2 * np.pi * (m1[..., None] * Bm[0] + m2[..., None] * Bm[1] + m3[..., None] * Bm[2])
    nu = amp * np.exp(-np.sum(G * G, axis=-1) / 4.0) * xi
    return np.real(np.fft.ifftn(nu)) * N


# ----------------------------------------------------------------------------
# configs
# ----------------------------------------------------------------------------
def _si_supercell(N):
    cells = [(c1, c2, c3) for c1 in range(N) for c2 in range(N) for c3 in range(N)]
    x = np.array([(site + np.array(c)) / N for c in cells for site in _DIAMOND_SITES])
    return x


def _mp_grid(q):
    """SURVEY.md 8(c) reading 15: k_c = (2r - q_c - 1)/(2 q_c), r1 outer, r3 inner."""
    ax = [[(2 * r - qc - 1) / (2.0 * qc) for r in range(1, qc + 1)] for qc in q]
    return np.array([(a, b, c) for a in ax[0] for b in ax[1] for c in ax[2]])


def make_config(name, with_vloc=True, **over):
    """Return a dict describing one synthetic cell.  `over` overrides ngfft/ecut/nband/kpt."""
    a_si, a_al = 10.26, 7.65
    kinds = ["Si"]
    typat = None
    depth, w, amp = -4.0, 1.5, 0.1
    if name == "c0":
        rprimd = 0.5 * a_si * np.array([[0, 1, 1], [1, 0, 1], [1, 1, 0]], float)
        xred = np.array([[0, 0, 0], [.25, .25, .25]]); kpt = [[0, 0, 0]]
        ecut, ngfft, nband = 8.0, (20, 20, 20), 8
    elif name in ("c1", "c1m"):
        rprimd = np.diag([2 * a_si] * 3); xred = _si_supercell(2); kpt = [[.25, .25, .25]]
        ecut, ngfft, nband = (15.0, (72, 72, 72), 128) if name == "c1" else (2.0, (30, 30, 30), 6)
    elif name in ("c2", "c2m"):
        rprimd = np.diag([3 * a_si] * 3); xred = _si_supercell(3); kpt = [[0, 0, 0]]
        ecut, ngfft, nband = (20.0, (128, 128, 128), 432) if name == "c2" else (1.0, (30, 30, 30), 5)
    elif name in ("c3", "c3k2"):
        rprimd = np.diag([a_al] * 3); xred = _FCC_SITES.copy(); kinds = ["Al"]
        kpt = _mp_grid((4, 4, 2)) if name == "c3" else _mp_grid((4, 4, 2))[[0, 10]]
        ecut, ngfft, nband = 20.0, (32, 32, 32), (64 if name == "c3" else 5)
        depth, w, amp = -3.0, 2.0, 0.05
    elif name in ("c4", "c4m"):
        rprimd = np.diag([4 * a_si] * 3); xred = _si_supercell(4); kpt = [[0, 0, 0]]
        ecut, ngfft, nband = (20.0, (180, 180, 180), 1024) if name == "c4" else (0.5, (36, 36, 36), 7)
    elif name in ("aniso", "anisok3"):     # SURVEY.md 8(c) extra case (ii): triclinic, anisotropic box, two types
        rprimd = np.array([[9.0, 0.4, -0.3], [0.7, 10.5, 0.5], [-0.6, 0.8, 13.0]])
        xred = np.array([[0.0, 0.0, 0.0],                      # exactly on a grid point
                         [0.3183098861837907, 0.7071067811865476, 0.5772156649015329],  # irrational
                         [0.55, 0.25, 0.8]])
        kinds = ["Si", "Al"]; typat = np.array([0, 1, 0], np.int32)
        kpt = [[0.1, -0.2, 0.05]]
        if name == "anisok3":   # three k-points: most columns at the third, most planes at the second (scratch-size check)
            kpt = [[0.1, -0.2, 0.05], [0.0, 0.0, 0.5], [0.5, 0.5, 0.0]]
        ecut, ngfft, nband = 2.5, (20, 24, 30), 4
    elif name == "aniso8":    # aniso with two types of at most 8 projectors (8 and 4): rows of one atom are not 8-aligned
        rprimd = np.array([[9.0, 0.4, -0.3], [0.7, 10.5, 0.5], [-0.6, 0.8, 13.0]])
        xred = np.array([[0.0, 0.0, 0.0], [0.3183098861837907, 0.7071067811865476, 0.5772156649015329],
                         [0.55, 0.25, 0.8], [0.12, 0.61, 0.33]])
        kinds = ["Si", "Sip"]; typat = np.array([1, 0, 1, 0], np.int32)
        kpt = [[0.1, -0.2, 0.05]]
        ecut, ngfft, nband = 2.5, (20, 24, 30), 5
    elif name == "aniso5t":   # five atom types in mixed order (8, 9, 4, 9 and 8 projectors): more form-factor rows than the
        rprimd = np.array([[9.0, 0.4, -0.3], [0.7, 10.5, 0.5], [-0.6, 0.8, 13.0]])   # factorised kernels hold at once
        xred = np.array([[0.0, 0.0, 0.0], [0.3183098861837907, 0.7071067811865476, 0.5772156649015329],
                         [0.55, 0.25, 0.8], [0.12, 0.61, 0.33], [0.81, 0.07, 0.44], [0.37, 0.9, 0.15], [0.66, 0.52, 0.6]])
        kinds = ["Si", "Al", "Sip", "Al", "Si"]; typat = np.array([4, 1, 0, 3, 2, 1, 0], np.int32)
        kpt = [[0.1, -0.2, 0.05]]
        ecut, ngfft, nband = 2.5, (20, 24, 30), 5
    else:
        raise ValueError(name)
    ecut = float(over.get("ecut", ecut))
    ngfft = tuple(int(v) for v in over.get("ngfft", ngfft))
    nband = int(over.get("nband", nband))
    kpt = np.array(over.get("kpt", kpt), float).reshape(-1, 3)
    if "xred" in over:
        xred = np.array(over["xred"], float).reshape(-1, 3)
    natom = len(xred)
    if typat is None or len(typat) != natom:
        typat = np.zeros(natom, np.int32)
    seed = config_seed(name)
    # |k+G| <= sqrt(2 ecut) inside the sphere: table range is input data, not method arithmetic
    types = [_proj_type(kd, np.sqrt(2.0 * ecut)) for kd in kinds]
    lmax = max(t["nlmn"] for t in types)
    # D_ij: upper triangle 0.5*N(0,1), mirrored; zero outside the atom's nlmn
    dij = np.zeros((natom, lmax, lmax))
    idx = np.arange(natom * lmax * lmax, dtype=np.uint64).reshape(natom, lmax, lmax)
    raw = 0.5 * rng.normals(seed, STREAM_DIJ, idx)
    for a in range(natom):
        nl = types[typat[a]]["nlmn"]
        up = np.triu(raw[a, :nl, :nl])
        dij[a, :nl, :nl] = up + np.triu(up, 1).T
    cfg = dict(name=name, seed=seed, rprimd=np.ascontiguousarray(rprimd, float), kpt=kpt, nkpt=len(kpt),
               ecut=ecut, ngfft=ngfft, natom=natom, typat=np.ascontiguousarray(typat, np.int32),
               xred=np.ascontiguousarray(xred, float), types=types, ntypat=len(types),
               nlmn_max=lmax, nproj=int(sum(types[t]["nlmn"] for t in typat)),
               dij=dij, nband=nband, vloc_params=(depth, w, amp))
    if with_vloc:
        cfg["vloc"] = gen_vloc(cfg)
    return cfg


def gen_vloc(cfg):
    """V_loc(r_j), shape [n3][n2][n1] (i1 fastest), float64."""
    depth, w, amp = cfg["vloc_params"]
    V = _vloc_gauss(cfg["rprimd"], cfg["ngfft"], cfg["xred"], depth, w)
    V = V + _vloc_noise(cfg["rprimd"], cfg["ngfft"], amp, cfg["seed"])
    return np.ascontiguousarray(V)


def gen_psi_band(seed, kin, flat_band_index, mpw):
    """One band: c(G) = (xi1 + i xi2)/(1 + |k+G|^2), |k+G|^2 = 2*kin, RNG index = band*mpw + ipw."""
    npw = len(kin)
    idx = np.uint64(flat_band_index) * np.uint64(mpw) + np.arange(npw, dtype=np.uint64)
    out = np.zeros(mpw, np.complex128)
    env = 1.0 / (1.0 + 2.0 * np.asarray(kin))
    out[:npw] = (rng.normals(seed, STREAM_PSI, idx, 0) + 1j * rng.normals(seed, STREAM_PSI, idx, 1)) * env
    return out


def gen_psi(cfg, kin_list, nband=None, bands=None, threads=8):
    """psi[nkpt][nband][mpw] complex128 (entries ipw >= npw_k are zero).

    kin_list: one kin array per k-point, from whichever side (oracle or library)
    the caller trusts; both are required to be bit-identical.
    `bands`: optional explicit list of band numbers (for sampled-band checks).
    """
    nband = cfg["nband"] if nband is None else nband
    bands = list(range(nband)) if bands is None else list(bands)
    mpw = max(len(k) for k in kin_list)
    nk = len(kin_list)
    psi = np.zeros((nk, len(bands), mpw), np.complex128)

    def work(t):
        ik, j = t
        # flat band index uses the config's full band count so that a sampled
        # band equals the same band of the full block
        psi[ik, j] = gen_psi_band(cfg["seed"], kin_list[ik], ik * cfg["nband"] + bands[j], mpw)
    jobs = [(ik, j) for ik in range(nk) for j in range(len(bands))]
    if len(jobs) > 4 and threads > 1:
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(work, jobs))
    else:
        for t in jobs:
            work(t)
    return psi


def gen_psi_torch(cfg, kin_list, device, nband=None):
    """Same block as gen_psi, drawn on a torch device: tensor [nkpt][nband][mpw] complex128."""
    import torch
    nband = cfg["nband"] if nband is None else nband
    mpw = max(len(k) for k in kin_list)
    nk = len(kin_list)
    psi = torch.zeros((nk, nband, mpw), dtype=torch.complex128, device=device)
    for ik, kin in enumerate(kin_list):
        npw = len(kin)
        env = 1.0 / (1.0 + 2.0 * torch.as_tensor(np.asarray(kin), device=device))
        step = max(1, (1 << 24) // max(npw, 1))
        for b0 in range(0, nband, step):
            b1 = min(nband, b0 + step)
            flat = torch.arange(ik * cfg["nband"] + b0, ik * cfg["nband"] + b1, device=device, dtype=torch.int64)
            idx = flat[:, None] * mpw + torch.arange(npw, device=device, dtype=torch.int64)[None, :]
            n0, n1 = rng.torch_normals_pair(cfg["seed"], STREAM_PSI, idx)
            psi[ik, b0:b1, :npw] = torch.complex(n0 * env, n1 * env)
    return psi


# ----------------------------------------------------------------------------
# inputs of the NEXT row 4 variants: Gamma-point real-symmetry storage, two-component spinors
# ----------------------------------------------------------------------------
STREAM_BFIELD, STREAM_DSPIN = 4, 5


def projector_l(cfg):
    """Angular momentum l of every projector row of the table (atoms in order, i = 0 .. nlmn-1)."""
    return np.concatenate([np.asarray(cfg["types"][t]["l"], np.int64) for t in cfg["typat"]])


def gamma_dij(cfg):
    """D_ij of the cell with the entries that couple projectors of different l-parity set to zero: with the projector
    convention of DESIGN.md reading 6 (no (-i)^l factor) those are the entries that break time-reversal symmetry, so a
    real-in-r-space psi stays real under H only without them (reading 26)."""
    d = np.array(cfg["dij"], float)
    for a in range(cfg["natom"]):
        l = np.asarray(cfg["types"][cfg["typat"][a]]["l"], np.int64)
        nl = len(l)
        odd = ((l[:, None] + l[None, :]) % 2) == 1
        d[a, :nl, :nl][odd] = 0.0
    return d


def spinor_inputs(cfg):
    """(v4, dspin) for the two-component variant (reading 27):
    v4 [4][n3][n2][n1] = V_upup, V_dndn, Re V_updn, Im V_updn with V = V_loc + B.sigma for a smooth seeded field B(r)
    (so V_upup = V + Bz, V_dndn = V - Bz, V_updn = Bx - i By); dspin [natom][2][2][lm][lm] complex, Hermitian in the
    combined index (sigma i), (sigma' j): delta_ss' D_ij plus a seeded Hermitian perturbation of relative size 0.3."""
    V = np.asarray(cfg["vloc"], float)
    B = [_vloc_noise(cfg["rprimd"], cfg["ngfft"], 0.5 * cfg["vloc_params"][2], cfg["seed"] + 7919 * (c + 1)) for c in range(3)]
    v4 = np.ascontiguousarray(np.stack([V + B[2], V - B[2], B[0], -B[1]]))
    natom, lm = cfg["natom"], cfg["nlmn_max"]
    n = 2 * lm
    idx = np.arange(natom * n * n, dtype=np.uint64).reshape(natom, n, n)
    z = 0.15 * (rng.normals(cfg["seed"], STREAM_DSPIN, idx, 0) + 1j * rng.normals(cfg["seed"], STREAM_DSPIN, idx, 1))
    dspin = np.zeros((natom, 2, 2, lm, lm), np.complex128)
    for a in range(natom):
        nl = cfg["types"][cfg["typat"][a]]["nlmn"]
        h = z[a] + z[a].conj().T                                 # Hermitian [2 lm][2 lm], index = sigma * lm + i
        h = h.reshape(2, lm, 2, lm).transpose(0, 2, 1, 3).copy()   # [s][s'][i][j]
        h[:, :, nl:, :] = 0.0; h[:, :, :, nl:] = 0.0
        dspin[a] = h
        for s in range(2):
            dspin[a, s, s] += cfg["dij"][a]
    return v4, dspin
