"""paper_2507_08578_b200 -- thin ctypes binding of libdftb200.so (C ABI in include/dft.h).

The library applies the plane-wave Kohn-Sham Hamiltonian to a block of bands on one B200
(Sec. V, :456, Eq. 26 :470-:475).  This module only marshals arguments: every step of
the path (G-sphere builder, pruned FFT passes, projector GEMMs) runs in the CUDA kernels of
csrc/.  PyTorch is used for device memory and streams only.  There is no CPU fallback: if the
shared library cannot be loaded, importing `lib()` raises.

Function names mirror the C ABI (dft_plan_create, dft_set_vloc, dft_apply_h, ...); `Plan` is a
small convenience wrapper around them.
"""
import ctypes as C
import os

import numpy as np

from . import _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdftb200.so")

DFT_OK = 0
DFT_ERR_INVALID_ARG = -1
DFT_ERR_GRID_TOO_SMALL = -2
DFT_ERR_TABLE_RANGE = -3
DFT_NOALLOC_SCRATCH_BYTES = 64 << 20     # include/dft.h: static scratch of dft_apply_vloc_noalloc
DFT_ERR_ALLOC = -4
DFT_ERR_CUDA = -5
DFT_ERR_NOT_READY = -6
DFT_ERR_UNSUPPORTED = -7

PHASES = ("fft_A_scatter", "fft_B", "fft_C_V_Cinv", "fft_Binv", "fft_Ainv_gather", "gemm1", "dij", "gemm2_kinetic",
          "fft_small_fused", "pack_unpack")

# every symbol include/dft.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = ("dft_plan_create", "dft_plan_create_opts", "dft_apply_vloc_noalloc", "dft_plan_get_info", "dft_plan_workspace_bytes", "dft_plan_get_kg", "dft_plan_get_projectors", "dft_plan_copy_projectors_device", "dft_set_dij",
           "dft_set_sij", "dft_apply_s", "dft_apply_hs", "dft_get_cprj", "dft_chebyshev_filter",
           "dft_set_vector_potential", "dft_accumulate_density", "dft_accumulate_tau",
           "dft_set_vtau", "dft_plan_get_kg_gamma", "dft_apply_h_gamma", "dft_chebyshev_filter_gamma", "dft_set_vloc_spinor", "dft_set_dij_spinor",
           "dft_apply_h_spinor",
           "dft_set_vloc", "dft_set_workspace", "dft_plan_set_option", "dft_apply_h", "dft_apply_h_host",
           "dft_plan_last_launches", "dft_plan_set_timing", "dft_plan_phase_ms", "dft_plan_destroy", "dft_last_error")


class DftError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libdftb200 error %d: %s" % (code, msg))
        self.code = code


class dft_proj_table(C.Structure):
    _fields_ = [("nlmn", C.c_int32), ("l", C.POINTER(C.c_int32)), ("m", C.POINTER(C.c_int32)),
                ("irad", C.POINTER(C.c_int32)), ("nrad", C.c_int32), ("nq", C.c_int32), ("dq", C.c_double),
                ("f", C.POINTER(C.c_double)), ("f2", C.POINTER(C.c_double))]


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def lib():
    """Load (building first if the sources are newer and nvcc is present) the shared library."""
    global _lib
    if _lib is not None:
        return _lib
    if os.path.exists(_build.NVCC):
        _build.build()
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libdftb200.so is missing and nvcc is not available to build it; "
                           "run `python -m paper_2507_08578_b200._build` (there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.dft_last_error.restype = C.c_char_p
    L.dft_plan_last_launches.restype = C.c_int64
    L.dft_plan_last_launches.argtypes = [C.c_void_p]
    L.dft_plan_create.argtypes = [C.POINTER(C.c_void_p), _dp, C.c_int32, _dp, C.c_double, _ip, C.c_int32, _ip, _dp,
                                  C.c_int32, C.POINTER(dft_proj_table), _dp]
    L.dft_plan_create_opts.argtypes = L.dft_plan_create.argtypes + [C.c_int32, C.POINTER(C.c_char_p), C.POINTER(C.c_int64)]
    L.dft_plan_get_info.argtypes = [C.c_void_p, _ip, _ip, _ip, _ip, C.POINTER(C.c_int64)]
    L.dft_plan_workspace_bytes.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.dft_plan_get_kg.argtypes = [C.c_void_p, C.c_int32, _ip, _ip, _dp]
    L.dft_plan_get_projectors.argtypes = [C.c_void_p, C.c_int32, _dp]
    L.dft_set_dij.argtypes = [C.c_void_p, _dp]
    L.dft_plan_copy_projectors_device.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    L.dft_set_vloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.dft_set_workspace.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
    L.dft_plan_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int64]
    L.dft_apply_h.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_apply_vloc_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_apply_h_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32]
    L.dft_set_sij.argtypes = [C.c_void_p, _dp]
    L.dft_set_vector_potential.argtypes = [C.c_void_p, _dp]
    L.dft_set_vtau.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.dft_accumulate_density.argtypes = [C.c_void_p, C.c_void_p, _dp, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_accumulate_tau.argtypes = [C.c_void_p, C.c_void_p, _dp, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_chebyshev_filter.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double,
                                       C.c_void_p]
    L.dft_apply_s.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_apply_hs.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_get_cprj.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_plan_get_kg_gamma.argtypes = [C.c_void_p, _ip, _ip, _ip, _dp]
    L.dft_apply_h_gamma.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_chebyshev_filter_gamma.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double,
                                             C.c_void_p]
    L.dft_set_vloc_spinor.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.dft_set_dij_spinor.argtypes = [C.c_void_p, _dp]
    L.dft_apply_h_spinor.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.dft_plan_set_timing.argtypes = [C.c_void_p, C.c_int32]
    L.dft_plan_phase_ms.argtypes = [C.c_void_p, C.c_int32, _dp, C.POINTER(C.c_int64)]
    L.dft_plan_destroy.argtypes = [C.c_void_p]
    _lib = L
    return L


def dft_last_error():
    return lib().dft_last_error().decode()


def _check(rc):
    if rc != DFT_OK:
        raise DftError(rc, dft_last_error())


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _d(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _i(a):
    return a.ctypes.data_as(_ip) if a is not None else None


# ------------------------------------------------------------------------------------- C-ABI mirrors
def dft_plan_create(rprimd, kpt, ecut, ngfft, typat, xred, types, dij, options=None):
    """types: list of dicts with keys nlmn, l, m, irad, nrad, nq, dq, f[nrad][nq], f2[nrad][nq] (host).
    options: None, or a dict / list of (key, value) pairs handed to dft_plan_create_opts (proj_mode = 1 there means the
    materialised projector table is never built).  Returns the opaque plan handle (int)."""
    rp = _f64(rprimd).reshape(9)
    kp = _f64(kpt).reshape(-1, 3)
    ng = _i32(ngfft).reshape(3)
    ty = _i32(typat).reshape(-1)
    xr = _f64(xred).reshape(-1, 3)
    natom = len(ty)
    keep = []
    tabs = (dft_proj_table * max(1, len(types)))()
    for t, T in enumerate(types):
        l, m, ir = _i32(T["l"]), _i32(T["m"]), _i32(T["irad"])
        f, f2 = _f64(T["f"]), _f64(T["f2"])
        keep += [l, m, ir, f, f2]
        tabs[t].nlmn = int(T["nlmn"]); tabs[t].l = _i(l); tabs[t].m = _i(m); tabs[t].irad = _i(ir)
        tabs[t].nrad = int(T["nrad"]); tabs[t].nq = int(T["nq"]); tabs[t].dq = float(T["dq"])
        tabs[t].f = _d(f); tabs[t].f2 = _d(f2)
    dj = _f64(dij) if dij is not None else None
    out = C.c_void_p()
    if options is None:
        rc = lib().dft_plan_create(C.byref(out), _d(rp), len(kp), _d(kp), float(ecut), _i(ng), natom,
                                   _i(ty) if natom else None, _d(xr) if natom else None, len(types), tabs, _d(dj))
    else:
        items = list(options.items()) if isinstance(options, dict) else list(options)
        keys = (C.c_char_p * max(1, len(items)))(*[str(k).encode() for k, _ in items])
        vals = (C.c_int64 * max(1, len(items)))(*[int(v) for _, v in items])
        rc = lib().dft_plan_create_opts(C.byref(out), _d(rp), len(kp), _d(kp), float(ecut), _i(ng), natom,
                                        _i(ty) if natom else None, _d(xr) if natom else None, len(types), tabs, _d(dj),
                                        len(items), keys, vals)
    _check(rc)
    return out.value


def dft_plan_get_info(plan):
    nk = C.c_int32()
    _check(lib().dft_plan_get_info(plan, C.byref(nk), None, None, None, None))
    npw = np.zeros(nk.value, np.int32)
    mpw, nproj, ws = C.c_int32(), C.c_int32(), C.c_int64()
    _check(lib().dft_plan_get_info(plan, C.byref(nk), _i(npw), C.byref(mpw), C.byref(nproj), C.byref(ws)))
    return dict(nkpt=nk.value, npw=npw, mpw=mpw.value, nproj=nproj.value, workspace_bytes_per_band=ws.value)


def dft_plan_workspace_bytes(plan, nband):
    """(min_bytes, full_bytes) of device scratch for dft_set_workspace."""
    lo, hi = C.c_int64(), C.c_int64()
    _check(lib().dft_plan_workspace_bytes(plan, nband, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def dft_plan_get_kg(plan, ik, npw):
    kg = np.zeros((npw, 3), np.int32); ig = np.zeros(npw, np.int32); kin = np.zeros(npw)
    _check(lib().dft_plan_get_kg(plan, ik, _i(kg), _i(ig), _d(kin)))
    return kg, ig, kin


def dft_plan_get_projectors(plan, ik, nproj, npw):
    out = np.zeros((nproj, npw), np.complex128)
    _check(lib().dft_plan_get_projectors(plan, ik, _d(out.view(np.float64))))
    return out


def dft_plan_copy_projectors_device(plan, ik, ptab_dev_ptr, stream=0):
    _check(lib().dft_plan_copy_projectors_device(plan, ik, ptab_dev_ptr, stream))


def dft_set_dij(plan, dij):
    _check(lib().dft_set_dij(plan, _d(_f64(dij))))


def dft_set_vloc(plan, v_dev_ptr, stream=0):
    _check(lib().dft_set_vloc(plan, v_dev_ptr, stream))


def dft_set_workspace(plan, dev_ptr, nbytes):
    _check(lib().dft_set_workspace(plan, dev_ptr, nbytes))


def dft_plan_set_option(plan, key, value):
    _check(lib().dft_plan_set_option(plan, key.encode(), int(value)))


def dft_apply_h(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream=0):
    _check(lib().dft_apply_h(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream))


def dft_apply_vloc_noalloc(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream=0):
    _check(lib().dft_apply_vloc_noalloc(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream))


def dft_set_sij(plan, sij):
    _check(lib().dft_set_sij(plan, _d(_f64(sij))))


def dft_apply_s(plan, psi_dev_ptr, spsi_dev_ptr, nband, stream=0):
    _check(lib().dft_apply_s(plan, psi_dev_ptr, spsi_dev_ptr, nband, stream))


def dft_apply_hs(plan, psi_dev_ptr, hpsi_dev_ptr, spsi_dev_ptr, nband, stream=0):
    _check(lib().dft_apply_hs(plan, psi_dev_ptr, hpsi_dev_ptr, spsi_dev_ptr, nband, stream))


def dft_get_cprj(plan, psi_dev_ptr, cprj_dev_ptr, nband, stream=0):
    _check(lib().dft_get_cprj(plan, psi_dev_ptr, cprj_dev_ptr, nband, stream))


def dft_accumulate_density(plan, psi_dev_ptr, weights, rho_dev_ptr, nband, stream=0):
    _check(lib().dft_accumulate_density(plan, psi_dev_ptr, _d(_f64(weights)), rho_dev_ptr, nband, stream))


def dft_accumulate_tau(plan, psi_dev_ptr, weights, tau_dev_ptr, nband, stream=0):
    _check(lib().dft_accumulate_tau(plan, psi_dev_ptr, _d(_f64(weights)), tau_dev_ptr, nband, stream))


def dft_set_vtau(plan, vtau_dev_ptr, stream=0):
    _check(lib().dft_set_vtau(plan, vtau_dev_ptr, stream))


def dft_set_vector_potential(plan, a_cart):
    _check(lib().dft_set_vector_potential(plan, None if a_cart is None else _d(_f64(a_cart))))


def dft_chebyshev_filter(plan, psi_dev_ptr, work_dev_ptr, nband, degree, center, halfwidth, stream=0):
    _check(lib().dft_chebyshev_filter(plan, psi_dev_ptr, work_dev_ptr, nband, degree, center, halfwidth, stream))


def dft_plan_get_kg_gamma(plan):
    n = C.c_int32(0)
    _check(lib().dft_plan_get_kg_gamma(plan, C.byref(n), None, None, None))
    kg = np.zeros((n.value, 3), np.int32); ig = np.zeros(n.value, np.int32); kin = np.zeros(n.value)
    _check(lib().dft_plan_get_kg_gamma(plan, C.byref(n), _i(kg), _i(ig), _d(kin)))
    return kg, ig, kin


def dft_apply_h_gamma(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream=0):
    _check(lib().dft_apply_h_gamma(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream))


def dft_chebyshev_filter_gamma(plan, psi_dev_ptr, work_dev_ptr, nband, degree, center, halfwidth, stream=0):
    _check(lib().dft_chebyshev_filter_gamma(plan, psi_dev_ptr, work_dev_ptr, nband, degree, center, halfwidth, stream))


def dft_set_vloc_spinor(plan, v4_dev_ptr, stream=0):
    _check(lib().dft_set_vloc_spinor(plan, v4_dev_ptr, stream))


def dft_set_dij_spinor(plan, dspin):
    if dspin is None:
        _check(lib().dft_set_dij_spinor(plan, None))
        return
    d = np.ascontiguousarray(dspin, np.complex128)
    _check(lib().dft_set_dij_spinor(plan, _d(d.view(np.float64))))


def dft_apply_h_spinor(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream=0):
    _check(lib().dft_apply_h_spinor(plan, psi_dev_ptr, hpsi_dev_ptr, nband, stream))


def dft_apply_h_host(plan, psi_host_ptr, hpsi_host_ptr, nband):
    _check(lib().dft_apply_h_host(plan, psi_host_ptr, hpsi_host_ptr, nband))


def dft_plan_last_launches(plan):
    return int(lib().dft_plan_last_launches(plan))


def dft_plan_set_timing(plan, on):
    _check(lib().dft_plan_set_timing(plan, 1 if on else 0))


def dft_plan_phase_ms(plan, phase):
    ms = C.c_double(); n = C.c_int64()
    _check(lib().dft_plan_phase_ms(plan, phase, C.byref(ms), C.byref(n)))
    return ms.value, n.value


def dft_plan_destroy(plan):
    _check(lib().dft_plan_destroy(plan))


# ------------------------------------------------------------------------------------- convenience
class Plan:
    """Owns one dft_plan.  `cfg` is a dict with rprimd, kpt, ecut, ngfft, typat, xred, types, dij
    (the layout synth.make_config produces); tensors are torch CUDA tensors."""

    def __init__(self, cfg, options=None):
        self.h = dft_plan_create(cfg["rprimd"], cfg["kpt"], cfg["ecut"], cfg["ngfft"], cfg["typat"], cfg["xred"],
                                 cfg["types"], cfg["dij"], options)
        info = dft_plan_get_info(self.h)
        self.nkpt, self.npw, self.mpw, self.nproj = info["nkpt"], info["npw"], info["mpw"], info["nproj"]
        self.workspace_bytes_per_band = info["workspace_bytes_per_band"]
        self.ngfft = tuple(int(v) for v in cfg["ngfft"])
        self._keep = []

    def workspace_bytes(self, nband):
        return dft_plan_workspace_bytes(self.h, nband)

    def get_kg(self, ik=0):
        return dft_plan_get_kg(self.h, ik, int(self.npw[ik]))

    def get_projectors(self, ik=0):
        return dft_plan_get_projectors(self.h, ik, self.nproj, int(self.npw[ik]))

    def projectors_device(self, ik=0):
        """The materialised table of k-point ik as a torch complex128 CUDA tensor [nproj][mpw] (a copy)."""
        import torch
        out = torch.empty((self.nproj, self.mpw), dtype=torch.complex128, device="cuda")
        dft_plan_copy_projectors_device(self.h, ik, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
        return out

    def set_dij(self, dij):
        dft_set_dij(self.h, dij)

    def set_vloc(self, v):
        """v: torch float64 CUDA tensor [n3][n2][n1] (or anything with that many elements)."""
        import torch
        assert v.is_cuda and v.dtype == torch.float64 and v.is_contiguous()
        assert v.numel() == self.ngfft[0] * self.ngfft[1] * self.ngfft[2]
        dft_set_vloc(self.h, v.data_ptr(), torch.cuda.current_stream().cuda_stream)

    def set_workspace(self, t):
        if t is None:
            dft_set_workspace(self.h, None, 0)
        else:
            assert t.is_cuda and t.is_contiguous()
            self._keep = [t]
            dft_set_workspace(self.h, t.data_ptr(), t.numel() * t.element_size())

    def set_option(self, key, value):
        dft_plan_set_option(self.h, key, value)

    def apply_h(self, psi, hpsi=None):
        """psi: torch complex128 CUDA tensor [nkpt][nband][mpw] (or [nband][mpw] when nkpt = 1)."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous()
        assert psi.shape[-1] == self.mpw and (self.mpw == 0 or psi.numel() % (self.nkpt * self.mpw) == 0)
        nband = psi.numel() // (self.nkpt * self.mpw) if self.mpw else 0
        if hpsi is None:
            hpsi = torch.empty_like(psi)
        assert hpsi.is_cuda and hpsi.dtype == torch.complex128 and hpsi.is_contiguous() and hpsi.shape == psi.shape
        dft_apply_h(self.h, psi.data_ptr(), hpsi.data_ptr(), nband, torch.cuda.current_stream().cuda_stream)
        return hpsi

    def apply_vloc_noalloc(self, psi, hpsi):
        """hpsi = V_loc psi through dft_apply_vloc_noalloc (static scratch inside the library, no allocation): both tensors
        are the caller's, laid out as for apply_h."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous()
        assert hpsi.is_cuda and hpsi.dtype == torch.complex128 and hpsi.is_contiguous() and hpsi.shape == psi.shape
        assert psi.shape[-1] == self.mpw and (self.mpw == 0 or psi.numel() % (self.nkpt * self.mpw) == 0)
        nband = psi.numel() // (self.nkpt * self.mpw) if self.mpw else 0
        dft_apply_vloc_noalloc(self.h, psi.data_ptr(), hpsi.data_ptr(), nband, torch.cuda.current_stream().cuda_stream)
        return hpsi

    def get_kg_gamma(self):
        """(kg, igfft, kin) of the stored half sphere (option gamma_real = 1)."""
        return dft_plan_get_kg_gamma(self.h)

    def apply_h_gamma(self, psi, hpsi=None):
        """Gamma storage: psi torch complex128 CUDA tensor [nband][nhalf]."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.dim() == 2
        if hpsi is None:
            hpsi = torch.empty_like(psi)
        assert hpsi.is_cuda and hpsi.dtype == torch.complex128 and hpsi.is_contiguous() and hpsi.shape == psi.shape
        dft_apply_h_gamma(self.h, psi.data_ptr(), hpsi.data_ptr(), psi.shape[0], torch.cuda.current_stream().cuda_stream)
        return hpsi

    def chebyshev_filter_gamma(self, psi, degree, center, halfwidth, work=None):
        """In place, Gamma storage: psi [nband][nhalf] := T_degree((H - center)/halfwidth) psi."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.dim() == 2
        if work is None:
            work = torch.empty(2 * psi.numel(), dtype=torch.complex128, device=psi.device)
        assert work.is_cuda and work.dtype == torch.complex128 and work.numel() >= 2 * psi.numel()
        dft_chebyshev_filter_gamma(self.h, psi.data_ptr(), work.data_ptr(), psi.shape[0], degree, center, halfwidth,
                                   torch.cuda.current_stream().cuda_stream)
        return psi

    def set_vloc_spinor(self, v4):
        """v4: torch float64 CUDA tensor [4][n3][n2][n1] = V_upup, V_dndn, Re V_updn, Im V_updn."""
        import torch
        assert v4.is_cuda and v4.dtype == torch.float64 and v4.is_contiguous() and v4.numel() == 4 * int(np.prod(self.ngfft))
        dft_set_vloc_spinor(self.h, v4.data_ptr(), torch.cuda.current_stream().cuda_stream)

    def set_dij_spinor(self, dspin):
        dft_set_dij_spinor(self.h, dspin)

    def apply_h_spinor(self, psi, hpsi=None):
        """psi: torch complex128 CUDA tensor [nkpt][nband][2][mpw] (or [nband][2][mpw] when nkpt = 1)."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.shape[-1] == self.mpw and psi.shape[-2] == 2
        nband = psi.numel() // (self.nkpt * 2 * self.mpw) if self.mpw else 0
        if hpsi is None:
            hpsi = torch.empty_like(psi)
        assert hpsi.is_cuda and hpsi.dtype == torch.complex128 and hpsi.is_contiguous() and hpsi.shape == psi.shape
        dft_apply_h_spinor(self.h, psi.data_ptr(), hpsi.data_ptr(), nband, torch.cuda.current_stream().cuda_stream)
        return hpsi

    def set_sij(self, sij):
        dft_set_sij(self.h, sij)

    def apply_s(self, psi, spsi=None):
        """S psi (PAW overlap); same tensors as apply_h."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.shape[-1] == self.mpw
        nband = psi.numel() // (self.nkpt * self.mpw) if self.mpw else 0
        if spsi is None:
            spsi = torch.empty_like(psi)
        assert spsi.is_cuda and spsi.dtype == torch.complex128 and spsi.is_contiguous() and spsi.shape == psi.shape
        dft_apply_s(self.h, psi.data_ptr(), spsi.data_ptr(), nband, torch.cuda.current_stream().cuda_stream)
        return spsi

    def apply_hs(self, psi):
        """(H psi, S psi) from one set of projections; same tensors as apply_h."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.shape[-1] == self.mpw
        nband = psi.numel() // (self.nkpt * self.mpw) if self.mpw else 0
        hpsi = torch.empty_like(psi); spsi = torch.empty_like(psi)
        dft_apply_hs(self.h, psi.data_ptr(), hpsi.data_ptr(), spsi.data_ptr(), nband, torch.cuda.current_stream().cuda_stream)
        return hpsi, spsi

    def get_cprj(self, psi):
        """<p|psi> as a torch complex128 CUDA tensor [nkpt][nband][nproj]."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.shape[-1] == self.mpw
        nband = psi.numel() // (self.nkpt * self.mpw) if self.mpw else 0
        out = torch.zeros((self.nkpt, nband, self.nproj), dtype=torch.complex128, device=psi.device)
        dft_get_cprj(self.h, psi.data_ptr(), out.data_ptr(), nband, torch.cuda.current_stream().cuda_stream)
        return out

    def accumulate_density(self, psi, weights, rho=None, tau=False):
        """rho[n3][n2][n1] += sum_kn weights[k][n] |psi_kn(r)|^2; rho: torch float64 CUDA tensor (created as zeros if None).
        tau=True accumulates the kinetic-energy density 1/2 sum w |grad psi|^2 instead."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.shape[-1] == self.mpw
        nband = psi.numel() // (self.nkpt * self.mpw) if self.mpw else 0
        n1, n2, n3 = self.ngfft
        if rho is None:
            rho = torch.zeros((n3, n2, n1), dtype=torch.float64, device=psi.device)
        assert rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous() and rho.numel() == n1 * n2 * n3
        w = np.ascontiguousarray(weights, np.float64)
        assert w.size == self.nkpt * nband
        fn = dft_accumulate_tau if tau else dft_accumulate_density
        fn(self.h, psi.data_ptr(), w, rho.data_ptr(), nband, torch.cuda.current_stream().cuda_stream)
        return rho

    def set_vtau(self, v):
        """Meta-GGA v_tau(r): torch float64 CUDA tensor with n1*n2*n3 elements ([n3][n2][n1]); None switches the term off."""
        import torch
        if v is None:
            dft_set_vtau(self.h, None)
            return
        assert v.is_cuda and v.dtype == torch.float64 and v.is_contiguous() and v.numel() == int(np.prod(self.ngfft))
        dft_set_vtau(self.h, v.data_ptr(), torch.cuda.current_stream().cuda_stream)

    def set_vector_potential(self, a_cart):
        """Velocity gauge: kinetic term 1/2|k+G+A|^2 (A Cartesian, a.u.); None switches it off."""
        dft_set_vector_potential(self.h, a_cart)

    def chebyshev_filter(self, psi, degree, center, halfwidth, work=None):
        """In place: psi := T_degree((H - center)/halfwidth) psi.  work: optional complex128 CUDA tensor, 2 x psi.numel()."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.shape[-1] == self.mpw
        nband = psi.numel() // (self.nkpt * self.mpw) if self.mpw else 0
        if work is None:
            work = torch.empty(2 * psi.numel(), dtype=torch.complex128, device=psi.device)
        assert work.is_cuda and work.dtype == torch.complex128 and work.numel() >= 2 * psi.numel()
        dft_chebyshev_filter(self.h, psi.data_ptr(), work.data_ptr(), nband, degree, center, halfwidth,
                             torch.cuda.current_stream().cuda_stream)
        return psi

    def apply_h_host(self, psi, hpsi=None):
        """psi: numpy complex128 array or CPU torch tensor (pinned or not); returns the same kind."""
        is_np = isinstance(psi, np.ndarray)
        if is_np:
            psi = np.ascontiguousarray(psi, np.complex128)
            if hpsi is None:
                hpsi = np.empty_like(psi)
            pin, pout, numel = psi.ctypes.data, hpsi.ctypes.data, psi.size
        else:
            import torch
            assert not psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous()
            if hpsi is None:
                hpsi = torch.empty_like(psi, pin_memory=psi.is_pinned())
            pin, pout, numel = psi.data_ptr(), hpsi.data_ptr(), psi.numel()
        nband = numel // (self.nkpt * self.mpw) if self.mpw else 0
        dft_apply_h_host(self.h, pin, pout, nband)
        return hpsi

    def last_launches(self):
        return dft_plan_last_launches(self.h)

    def set_timing(self, on):
        dft_plan_set_timing(self.h, on)

    def phase_ms(self):
        """{phase name: (milliseconds, launches)} accumulated since the last call; synchronises."""
        return {name: dft_plan_phase_ms(self.h, i) for i, name in enumerate(PHASES)}

    def destroy(self):
        if self.h:
            dft_plan_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
