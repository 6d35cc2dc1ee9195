"""paper_1505_07851_b200 -- thin Python binding of libpcm_b200 (include/pcm.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of
``csrc/``.  PyTorch is used for device memory and streams; tensors are passed to the C ABI
as raw device pointers.  The function names are the C names.  There is no CPU fallback: if
the shared library is missing, or no CUDA device is usable, the calls raise.

This package never imports ``oracle`` (the CPU oracle is test infrastructure only).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpcm_b200.so")

PCM_OK = 0
PCM_NOT_CONVERGED = 1
PCM_NCLASS = 6
PCM_NL = 5
CLASS_NAMES = ("ss", "sp", "pp", "sd", "pd", "dd")

EXPORTS = (
    "pcm_options_default", "pcm_setup", "pcm_potential", "pcm_fock", "pcm_amatvec", "pcm_pivot_order",
    "pcm_rbj_build", "pcm_rbj_get", "pcm_cg_solve", "pcm_potential_host", "pcm_fock_host", "pcm_amatvec_host",
    "pcm_cg_solve_host", "pcm_get_info", "pcm_set_timing", "pcm_last_kernel_ms", "pcm_last_class_ms",
    "pcm_launch_count", "pcm_fp64_peak", "pcm_set_nuclei", "pcm_nuclear_potential", "pcm_rhs", "pcm_energy",
    "pcm_cg_threshold", "pcm_gradient", "pcm_last_cg_matvec_ms", "pcm_rbj_build_async", "pcm_switching", "pcm_set_cavity", "pcm_surface_gradient",
    "pcm_schwarz_bound", "pcm_last_error", "pcm_destroy",
    "pcm_build_cavity", "pcm_cavity_size", "pcm_cavity_get", "pcm_cavity_device", "pcm_cavity_destroy", "pcm_setup_cavity",
    "pcm_amatvec_static_init", "pcm_amatvec_static",
)
PCM_STATIC_MAX_POINTS = 16384


class pcm_options(C.Structure):
    _fields_ = [("screen_eps", C.c_double), ("d_pure", C.c_int), ("device", C.c_int), ("merge_products", C.c_int),
                ("gradient", C.c_int), ("store_near", C.c_int), ("cg_path", C.c_int), ("store_far", C.c_int), ("serial_classes", C.c_int), ("tma_tiles", C.c_int), ("rbj_global_scan", C.c_int), ("potential_pr", C.c_int), ("graph_calls", C.c_int)]


class pcm_info(C.Structure):
    _fields_ = [("nbf", C.c_int64), ("nshell", C.c_int64), ("npoint", C.c_int64),
                ("shell_pairs", C.c_int64 * PCM_NCLASS), ("prim_pairs", C.c_int64 * PCM_NCLASS),
                ("prim_pairs_total", C.c_int64), ("prim_pairs_unscreened", C.c_int64),
                ("products", C.c_int64 * PCM_NL), ("products_total", C.c_int64),
                ("prim_pair_points", C.c_double), ("product_points", C.c_double),
                ("zeta_min", C.c_double), ("zeta_max", C.c_double),
                ("rbj_block", C.c_int64), ("rbj_nblocks", C.c_int64), ("device_bytes", C.c_int64),
                ("amat_near_patches", C.c_int64), ("amat_stored_bytes", C.c_int64), ("amat_far_stored_bytes", C.c_int64),
                ("amat_persistent", C.c_int64), ("components", C.c_int64), ("rbj_selection", C.c_int64)]


class PcmError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"libpcm_b200 error {code}: {text}")
        self.code = code


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_lp = C.POINTER(C.c_int64)


def lib(build: bool = False):
    """The loaded shared library.  ``build=True`` compiles it first if it is stale or missing."""
    global _lib
    if _lib is None:
        if build:
            _build.build_library()
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1505_07851_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.pcm_options_default.argtypes = [C.POINTER(pcm_options)]
        L.pcm_options_default.restype = None
        L.pcm_setup.argtypes = [C.POINTER(vp), C.c_int, vp, vp, vp, vp, vp, C.c_int64, vp, vp, vp, C.POINTER(pcm_options)]
        L.pcm_potential.argtypes = [vp, vp, C.c_int64, vp, vp]
        L.pcm_fock.argtypes = [vp, vp, vp, C.c_int64, C.c_int, vp]
        L.pcm_amatvec.argtypes = [vp, vp, vp, vp]
        L.pcm_pivot_order.argtypes = [C.c_uint64, C.c_int64, vp]
        L.pcm_rbj_build.argtypes = [vp, C.c_int, C.c_uint64, vp, vp]
        L.pcm_rbj_build_async.argtypes = [vp, C.c_int, C.c_uint64, vp, vp]
        L.pcm_rbj_get.argtypes = [vp, vp, vp, vp]
        L.pcm_cg_solve.argtypes = [vp, vp, vp, C.c_double, C.c_int, C.c_int, C.c_int, _ip, _dp, vp]
        L.pcm_potential_host.argtypes = [vp, vp, C.c_int64, vp]
        L.pcm_fock_host.argtypes = [vp, vp, vp, C.c_int64, C.c_int]
        L.pcm_amatvec_host.argtypes = [vp, vp, vp]
        L.pcm_cg_solve_host.argtypes = [vp, vp, vp, C.c_double, C.c_int, C.c_int, C.c_int, _ip, _dp]
        L.pcm_get_info.argtypes = [vp, C.POINTER(pcm_info)]
        L.pcm_set_timing.argtypes = [vp, C.c_int]
        L.pcm_last_kernel_ms.argtypes = [vp, C.c_int, _dp, _ip]
        L.pcm_last_class_ms.argtypes = [vp, C.c_int, _dp]
        L.pcm_launch_count.argtypes = [vp, _lp]
        L.pcm_last_cg_matvec_ms.argtypes = [vp, _dp, _ip]
        L.pcm_fp64_peak.argtypes = [vp, C.c_int, _dp]
        L.pcm_set_nuclei.argtypes = [vp, C.c_int, vp, vp]
        L.pcm_nuclear_potential.argtypes = [vp, vp, vp]
        L.pcm_rhs.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.pcm_energy.argtypes = [vp, vp, vp, vp, C.c_double, _dp, vp]
        L.pcm_cg_threshold.argtypes = [C.c_double, C.c_double, _dp]
        L.pcm_gradient.argtypes = [vp, vp, C.c_int64, vp, vp, vp, vp]
        L.pcm_switching.argtypes = [C.c_int64, vp, vp, vp, C.c_int, vp, vp, vp, C.c_int]
        L.pcm_set_cavity.argtypes = [vp, vp, vp]
        L.pcm_surface_gradient.argtypes = [vp, vp, C.c_double, vp, vp, vp]
        L.pcm_build_cavity.argtypes = [C.POINTER(vp), C.c_int, vp, vp, C.c_int, vp, vp, C.c_double, C.c_double, C.c_int]
        L.pcm_cavity_size.argtypes = [vp, _lp]
        L.pcm_cavity_get.argtypes = [vp, vp, vp, vp, vp, vp]
        L.pcm_cavity_device.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.pcm_cavity_destroy.argtypes = [vp]
        L.pcm_setup_cavity.argtypes = [C.POINTER(vp), C.c_int, vp, vp, vp, vp, vp, vp, C.POINTER(pcm_options)]
        L.pcm_schwarz_bound.argtypes = [C.c_int, C.c_double, vp, C.c_int, C.c_double, vp, _dp]
        L.pcm_last_error.argtypes = [vp]
        L.pcm_last_error.restype = C.c_char_p
        L.pcm_destroy.argtypes = [vp]
        for name in EXPORTS:
            if name not in ("pcm_options_default", "pcm_last_error"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(rc, ctx=None):
    if rc < 0:
        raise PcmError(rc, lib().pcm_last_error(ctx).decode("utf-8", "replace"))
    return rc


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _stream(stream):
    """cudaStream_t of a torch stream (None: torch's current stream)."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dev(t, n=None, ctx=None, strided=False):
    """Device address of a CUDA float64 tensor: contiguous (unless `strided`: a row-major matrix with its own leading
    dimension), at least n elements, on the context's device."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64):
        raise TypeError("expected a CUDA float64 tensor")
    if n is not None and t.numel() < n:
        raise ValueError("tensor too small")
    if not strided and not t.is_contiguous():
        raise ValueError("expected a contiguous tensor")
    if ctx is not None and t.device.index != ctx.device:
        raise ValueError(f"tensor is on cuda:{t.device.index}, the context on cuda:{ctx.device}")
    return C.c_void_p(t.data_ptr())


def _matrix(t, n, what):
    """(device address, leading dimension) of a row-major n x n CUDA float64 matrix."""
    if n > 0 and (t.dim() != 2 or t.shape[0] < n or t.shape[1] < n or (t.shape[1] > 1 and t.stride(1) != 1)):
        raise ValueError(f"{what} must be a row-major matrix of at least {n} x {n}")
    ld = t.stride(0) if t.dim() == 2 and t.shape[0] > 1 else max(n, 1)
    if ld < n:
        raise ValueError(f"{what}: leading dimension {ld} < {n}")
    return ld


class Context:
    """Owner of a ``pcm_ctx*``; destroyed with pcm_destroy (or when garbage collected)."""

    def __init__(self, handle, nbf, M, device):
        self.handle = handle
        self.nbf = nbf
        self.M = M
        self.device = device
        self.nshell = 0
        self.natom = 0

    def __del__(self):
        try:
            pcm_destroy(self)
        except Exception:
            pass


# ----------------------------------------------------------------------------- the C calls
def pcm_options_default() -> pcm_options:
    o = pcm_options()
    lib().pcm_options_default(C.byref(o))
    return o


def pcm_setup(shell_l, shell_xyz, shell_nprim, prim_exp, prim_coef, pt_xyz, pt_zeta, pt_switch=None, *,
              screen_eps: float = 1e-12, d_pure: bool = True, device: int = -1, merge_products: bool = True,
              gradient: bool = False, store_near: bool = True, cg_path: int = 0, store_far: int = 0, tma_tiles: bool = False,
              serial_classes: bool = False, rbj_global_scan: bool = False, potential_pr: int = 0, graph_calls: int = 0) -> Context:
    """Host numpy arrays in, context out (include/pcm.h: pcm_setup)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("pcm_setup needs a CUDA device (there is no CPU fallback)")
    sl = _np(shell_l, np.int32)
    sx = _np(shell_xyz, np.float64).reshape(-1)
    sn = _np(shell_nprim, np.int32)
    pe = _np(prim_exp, np.float64)
    pc = _np(prim_coef, np.float64)
    px = _np(pt_xyz, np.float64).reshape(-1)
    pz = _np(pt_zeta, np.float64)
    ps = None if pt_switch is None else _np(pt_switch, np.float64)
    if len(sx) != 3 * len(sl) or len(sn) != len(sl) or len(pe) != int(sn.sum()) or len(pc) != len(pe):
        raise ValueError("pcm_setup: shell_xyz must hold 3 doubles per shell, prim_exp / prim_coef sum(shell_nprim) entries")
    if len(px) != 3 * len(pz) or (ps is not None and len(ps) != len(pz)):
        raise ValueError("pcm_setup: pt_xyz must hold 3 doubles per point, pt_switch one")
    if device < 0:
        device = torch.cuda.current_device()
    torch.cuda.init()
    opt = pcm_options_default()
    opt.screen_eps = float(screen_eps)
    opt.d_pure = 1 if d_pure else 0
    opt.device = int(device)
    opt.merge_products = 1 if merge_products else 0
    opt.gradient = 1 if gradient else 0
    opt.store_near = 1 if store_near else 0
    opt.cg_path = int(cg_path)
    opt.store_far = int(store_far)
    opt.tma_tiles = 1 if tma_tiles else 0
    opt.serial_classes = 1 if serial_classes else 0
    opt.rbj_global_scan = 1 if rbj_global_scan else 0
    opt.potential_pr = int(potential_pr)
    opt.graph_calls = int(graph_calls)
    h = C.c_void_p()
    rc = lib().pcm_setup(C.byref(h), len(sl), _hp(sl), _hp(sx), _hp(sn), _hp(pe), _hp(pc), len(pz), _hp(px), _hp(pz),
                         _hp(ps), C.byref(opt))
    _check(rc, None)
    ctx = Context(h, 0, len(pz), device)
    ctx.nbf = int(pcm_get_info(ctx).nbf)
    ctx.nshell = len(sl)
    return ctx


def pcm_get_info(ctx: Context) -> pcm_info:
    info = pcm_info()
    _check(lib().pcm_get_info(ctx.handle, C.byref(info)), ctx.handle)
    return info


def pcm_potential(ctx: Context, P, v=None, stream=None):
    """v = pcm_potential(P): P CUDA float64 [nbf, nbf] (row stride = ldp), v CUDA float64 [M]."""
    import torch
    if v is None:
        v = torch.empty(ctx.M, dtype=torch.float64, device=P.device)
    ldp = _matrix(P, ctx.nbf, "P")
    _check(lib().pcm_potential(ctx.handle, _dev(P, None, ctx, strided=True), ldp, _dev(v, ctx.M, ctx), _stream(stream)), ctx.handle)
    return v


def pcm_fock(ctx: Context, q, F=None, accumulate: bool = False, stream=None):
    import torch
    if F is None:
        F = torch.empty((ctx.nbf, ctx.nbf), dtype=torch.float64, device=q.device)
        accumulate = False
    ldf = _matrix(F, ctx.nbf, "F")
    _check(lib().pcm_fock(ctx.handle, _dev(q, ctx.M, ctx), _dev(F, None, ctx, strided=True), ldf, 1 if accumulate else 0, _stream(stream)), ctx.handle)
    return F


def pcm_amatvec(ctx: Context, q, y=None, stream=None):
    import torch
    if y is None:
        y = torch.empty(ctx.M, dtype=torch.float64, device=q.device)
    _check(lib().pcm_amatvec(ctx.handle, _dev(q, ctx.M, ctx), _dev(y, ctx.M, ctx), _stream(stream)), ctx.handle)
    return y


def pcm_amatvec_static_init() -> None:
    """Resolves the static scratch array on the current device (set-up; once per device, outside any graph capture)."""
    _check(lib().pcm_amatvec_static_init())


def pcm_amatvec_static(pt_xyz, pt_zeta, pt_switch, q, y=None, stream=None):
    """y = A q without a context and without any allocation inside the library (include/pcm.h).  All arguments are CUDA
    float64 tensors in the caller's point order: pt_xyz [M, 3], pt_zeta, pt_switch, q [M], M <= PCM_STATIC_MAX_POINTS.
    Pass y to keep the call free of allocations on the Python side too."""
    import torch
    M = int(q.numel())
    if y is None:
        y = torch.empty(M, dtype=torch.float64, device=q.device)
    _check(lib().pcm_amatvec_static(C.c_int64(M), _dev(pt_xyz, 3 * M), _dev(pt_zeta, M), _dev(pt_switch, M), _dev(q, M), _dev(y, M),
                                    _stream(stream)))
    return y


def pcm_set_nuclei(ctx: Context, atom_xyz, z) -> None:
    xyz = _np(atom_xyz, np.float64).reshape(-1)
    zz = _np(z, np.float64)
    if len(xyz) != 3 * len(zz):
        raise ValueError("atom_xyz must hold 3 doubles per nuclear charge")
    _check(lib().pcm_set_nuclei(ctx.handle, len(zz), _hp(xyz), _hp(zz)), ctx.handle)
    ctx.natom = len(zz)


def pcm_nuclear_potential(ctx: Context, u=None, stream=None):
    import torch
    if u is None:
        u = torch.empty(ctx.M, dtype=torch.float64, device=torch.device("cuda", torch.cuda.current_device()))
    _check(lib().pcm_nuclear_potential(ctx.handle, _dev(u, ctx.M), _stream(stream)), ctx.handle)
    return u


def pcm_rhs(ctx: Context, u, v, f: float, b=None, stream=None):
    import torch
    if b is None:
        b = torch.empty(ctx.M, dtype=torch.float64, device=u.device)
    _check(lib().pcm_rhs(ctx.handle, _dev(u, ctx.M), _dev(v, ctx.M), float(f), _dev(b, ctx.M), _stream(stream)), ctx.handle)
    return b


def pcm_energy(ctx: Context, u, v, q, f: float, stream=None) -> np.ndarray:
    """[(B z).q, c.q, q.A q/(2 f), total] (Eq. 13, c = -v)."""
    terms = np.zeros(4)
    _check(lib().pcm_energy(ctx.handle, _dev(u, ctx.M), _dev(v, ctx.M), _dev(q, ctx.M), float(f),
                            terms.ctypes.data_as(_dp), _stream(stream)), ctx.handle)
    return terms


def pcm_gradient(ctx: Context, P, q, stream=None):
    """(g_shell [nshell, 3], g_point [M, 3]) of E = v.q at fixed P and q (Eq. 14/22; needs pcm_setup(gradient=True))."""
    import torch
    if P.dim() != 2 or P.shape[0] != ctx.nbf or P.shape[1] != ctx.nbf or P.stride(1) != 1:
        raise ValueError("P must be nbf x nbf, row-major")
    gs = torch.empty((ctx.nshell, 3), dtype=torch.float64, device=P.device)
    gp = torch.empty((ctx.M, 3), dtype=torch.float64, device=P.device)
    _dev(P)
    _check(lib().pcm_gradient(ctx.handle, C.c_void_p(P.data_ptr()), P.stride(0), _dev(q, ctx.M), C.c_void_p(gs.data_ptr()),
                              C.c_void_p(gp.data_ptr()), _stream(stream)), ctx.handle)
    return gs, gp


def pcm_switching(pt_xyz, pt_zeta, pt_atom, atom_xyz, atom_radius, device: int = -1) -> np.ndarray:
    """S_k of Eq. 9 (device arithmetic, host arrays)."""
    px, pz = _np(pt_xyz, np.float64).reshape(-1), _np(pt_zeta, np.float64)
    pa = _np(pt_atom, np.int32)
    ax, ar = _np(atom_xyz, np.float64).reshape(-1), _np(atom_radius, np.float64)
    S = np.zeros(len(pz))
    _check(lib().pcm_switching(len(pz), _hp(px), _hp(pz), _hp(pa), len(ar), _hp(ax), _hp(ar), _hp(S), int(device)))
    return S


class Cavity:
    """Owner of a ``pcm_cavity*`` (device arrays of the kept surface points)."""

    def __init__(self, handle, natom):
        self.handle = handle
        self.natom = natom

    @property
    def npoint(self) -> int:
        n = C.c_int64(0)
        _check(lib().pcm_cavity_size(self.handle, C.byref(n)))
        return int(n.value)

    def __del__(self):
        try:
            pcm_cavity_destroy(self)
        except Exception:
            pass


def pcm_build_cavity(atom_xyz, atom_radius, grid_xyz, grid_weight, zeta_tab: float, s_min: float = 1e-8, device: int = -1) -> Cavity:
    """ISWIG cavity of Eq. 7 / Eq. 9 with the S_k >= s_min screening, built on the device (include/pcm.h)."""
    ax, ar = _np(atom_xyz, np.float64).reshape(-1), _np(atom_radius, np.float64)
    gx, gw = _np(grid_xyz, np.float64).reshape(-1), _np(grid_weight, np.float64)
    if len(ax) != 3 * len(ar) or len(gx) != 3 * len(gw):
        raise ValueError("atom_xyz / grid_xyz must hold 3 doubles per radius / weight")
    h = C.c_void_p()
    _check(lib().pcm_build_cavity(C.byref(h), len(ar), _hp(ax), _hp(ar), len(gw), _hp(gx), _hp(gw), float(zeta_tab), float(s_min), int(device)))
    return Cavity(h, len(ar))


def pcm_cavity_get(cav: Cavity):
    """(xyz [n, 3], zeta [n], S [n], atom [n], node [n]) as host arrays."""
    n = cav.npoint
    xyz, zeta, S = np.zeros((n, 3)), np.zeros(n), np.zeros(n)
    atom, node = np.zeros(n, np.int32), np.zeros(n, np.int32)
    _check(lib().pcm_cavity_get(cav.handle, _hp(xyz), _hp(zeta), _hp(S), _hp(atom), _hp(node)))
    return xyz, zeta, S, atom, node


def pcm_cavity_device(cav: Cavity):
    """Raw device addresses (xyz, zeta, S, atom, node) of the cavity's arrays."""
    p = [C.c_void_p() for _ in range(5)]
    _check(lib().pcm_cavity_device(cav.handle, *[C.byref(x) for x in p]))
    return tuple(x.value for x in p)


def pcm_cavity_destroy(cav: Cavity) -> None:
    if cav is not None and getattr(cav, "handle", None):
        h, cav.handle = cav.handle, None
        lib().pcm_cavity_destroy(h)


def pcm_setup_cavity(shell_l, shell_xyz, shell_nprim, prim_exp, prim_coef, cav: Cavity, *, screen_eps: float = 1e-12,
                     d_pure: bool = True, merge_products: bool = True, gradient: bool = False, store_near: bool = True) -> Context:
    """pcm_setup with the surface points of a built cavity."""
    import torch
    sl = _np(shell_l, np.int32)
    sx = _np(shell_xyz, np.float64).reshape(-1)
    sn = _np(shell_nprim, np.int32)
    pe = _np(prim_exp, np.float64)
    pc = _np(prim_coef, np.float64)
    if len(sx) != 3 * len(sl) or len(sn) != len(sl) or len(pe) != int(sn.sum()) or len(pc) != len(pe):
        raise ValueError("pcm_setup_cavity: inconsistent shell array lengths")
    opt = pcm_options_default()
    opt.screen_eps = float(screen_eps)
    opt.d_pure = 1 if d_pure else 0
    opt.merge_products = 1 if merge_products else 0
    opt.gradient = 1 if gradient else 0
    opt.store_near = 1 if store_near else 0
    h = C.c_void_p()
    _check(lib().pcm_setup_cavity(C.byref(h), len(sl), _hp(sl), _hp(sx), _hp(sn), _hp(pe), _hp(pc), cav.handle, C.byref(opt)), None)
    ctx = Context(h, 0, cav.npoint, torch.cuda.current_device())
    ctx.nbf = int(pcm_get_info(ctx).nbf)
    ctx.nshell = len(sl)
    return ctx


def pcm_set_cavity(ctx: Context, atom_radius, pt_atom) -> None:
    ar, pa = _np(atom_radius, np.float64), _np(pt_atom, np.int32)
    if len(pa) != ctx.M:
        raise ValueError("pt_atom must have one entry per surface point")
    if len(ar) != ctx.natom:
        raise ValueError("atom_radius must have one entry per atom given to pcm_set_nuclei")
    _check(lib().pcm_set_cavity(ctx.handle, _hp(ar), _hp(pa)), ctx.handle)


def pcm_surface_gradient(ctx: Context, q, f: float, stream=None):
    """(g_point [M, 3], g_atom [natom, 3]) of (B z).q + q.A q/(2 f) at fixed q (Eq. 14 surface terms)."""
    import torch
    gp = torch.empty((ctx.M, 3), dtype=torch.float64, device=q.device)
    ga = torch.empty((ctx.natom, 3), dtype=torch.float64, device=q.device)
    _check(lib().pcm_surface_gradient(ctx.handle, _dev(q, ctx.M), float(f), C.c_void_p(gp.data_ptr()), C.c_void_p(ga.data_ptr()),
                                      _stream(stream)), ctx.handle)
    return gp, ga


def pcm_cg_threshold(diis_prev: float, delta_min: float = 1e-6) -> float:
    out = C.c_double(0.0)
    _check(lib().pcm_cg_threshold(float(diis_prev), float(delta_min), C.byref(out)))
    return out.value


def pcm_pivot_order(seed: int, M: int) -> np.ndarray:
    perm = np.zeros(M, np.int64)
    _check(lib().pcm_pivot_order(C.c_uint64(seed & 0xFFFFFFFFFFFFFFFF), M, _hp(perm)))
    return perm


def pcm_rbj_build(ctx: Context, block: int, seed: int = 0, pivot_order=None, stream=None):
    po = None if pivot_order is None else _np(pivot_order, np.int64)
    _check(lib().pcm_rbj_build(ctx.handle, int(block), C.c_uint64(seed & 0xFFFFFFFFFFFFFFFF), _hp(po), _stream(stream)),
           ctx.handle)


def pcm_rbj_build_async(ctx: Context, block: int, seed: int = 0, pivot_order=None, stream=None):
    """pcm_rbj_build queued on `stream` without synchronising; the next pcm_cg_solve(precond=2) completes it."""
    po = None if pivot_order is None else _np(pivot_order, np.int64)
    _check(lib().pcm_rbj_build_async(ctx.handle, int(block), C.c_uint64(seed & 0xFFFFFFFFFFFFFFFF), _hp(po), _stream(stream)), ctx.handle)


def pcm_rbj_get(ctx: Context):
    """(order[M], bstart[nblocks+1], list of inverse blocks)."""
    info = pcm_get_info(ctx)
    M, l, nb = ctx.M, int(info.rbj_block), int(info.rbj_nblocks)
    order = np.zeros(M, np.int64)
    bstart = np.zeros(nb + 1, np.int64)
    sizes = [min(l, M - b * l) for b in range(nb)]
    inv = np.zeros(int(sum(n * n for n in sizes)))
    _check(lib().pcm_rbj_get(ctx.handle, _hp(order), _hp(bstart), _hp(inv)), ctx.handle)
    blocks, off = [], 0
    for n in sizes:
        blocks.append(inv[off:off + n * n].reshape(n, n))
        off += n * n
    return order, bstart, blocks


def pcm_cg_solve(ctx: Context, b, x=None, tol: float = 1e-8, max_iter: int = 1000, precond: int = 1, use_x0: bool = False,
                 stream=None):
    """Returns (x, iterations, recurrence residual, true residual, converged)."""
    import torch
    if x is None:
        x = torch.zeros(ctx.M, dtype=torch.float64, device=b.device)
        use_x0 = False
    it = C.c_int(0)
    resid = (C.c_double * 2)()
    rc = _check(lib().pcm_cg_solve(ctx.handle, _dev(b, ctx.M, ctx), _dev(x, ctx.M, ctx), float(tol), int(max_iter), int(precond),
                                   1 if use_x0 else 0, C.byref(it), resid, _stream(stream)), ctx.handle)
    return x, int(it.value), float(resid[0]), float(resid[1]), rc == PCM_OK


def pcm_potential_host(ctx: Context, P: np.ndarray, v: np.ndarray | None = None) -> np.ndarray:
    P = _np(P, np.float64)
    if v is None:
        v = np.empty(ctx.M)
    _check(lib().pcm_potential_host(ctx.handle, _hp(P), P.shape[1] if P.ndim == 2 else ctx.nbf, _hp(v)), ctx.handle)
    return v


def pcm_fock_host(ctx: Context, q: np.ndarray, F: np.ndarray | None = None, accumulate: bool = False) -> np.ndarray:
    q = _np(q, np.float64)
    if F is None:
        F = np.empty((ctx.nbf, ctx.nbf))
        accumulate = False
    assert F.flags.c_contiguous and F.dtype == np.float64
    _check(lib().pcm_fock_host(ctx.handle, _hp(q), _hp(F), F.shape[1], 1 if accumulate else 0), ctx.handle)
    return F


def pcm_amatvec_host(ctx: Context, q: np.ndarray, y: np.ndarray | None = None) -> np.ndarray:
    q = _np(q, np.float64)
    if y is None:
        y = np.empty(ctx.M)
    _check(lib().pcm_amatvec_host(ctx.handle, _hp(q), _hp(y)), ctx.handle)
    return y


def pcm_cg_solve_host(ctx: Context, b: np.ndarray, x0: np.ndarray | None = None, tol: float = 1e-8, max_iter: int = 1000,
                      precond: int = 1):
    b = _np(b, np.float64)
    x = np.zeros(ctx.M) if x0 is None else _np(x0, np.float64).copy()
    it = C.c_int(0)
    resid = (C.c_double * 2)()
    rc = _check(lib().pcm_cg_solve_host(ctx.handle, _hp(b), _hp(x), float(tol), int(max_iter), int(precond),
                                        0 if x0 is None else 1, C.byref(it), resid), ctx.handle)
    return x, int(it.value), float(resid[0]), float(resid[1]), rc == PCM_OK


def pcm_set_timing(ctx: Context, enable: bool) -> None:
    _check(lib().pcm_set_timing(ctx.handle, 1 if enable else 0), ctx.handle)


OP_POTENTIAL, OP_FOCK, OP_AMATVEC = 0, 1, 2


def pcm_last_kernel_ms(ctx: Context, op: int):
    """(main kernels ms, transforms/reductions ms, kernels launched) of the last timed call of `op`."""
    ms = (C.c_double * 2)()
    n = C.c_int(0)
    _check(lib().pcm_last_kernel_ms(ctx.handle, int(op), ms, C.byref(n)), ctx.handle)
    return float(ms[0]), float(ms[1]), int(n.value)


def pcm_last_class_ms(ctx: Context, op: int):
    """device ms of the main kernel of each total angular momentum L = 0..4 in the last timed call of `op`"""
    ms = (C.c_double * PCM_NL)()
    _check(lib().pcm_last_class_ms(ctx.handle, int(op), ms), ctx.handle)
    return [float(x) for x in ms]


def pcm_last_cg_matvec_ms(ctx: Context):
    """(mean ms of the first <= 16 A q launches of the last timed pcm_cg_solve, how many)"""
    ms, n = C.c_double(0.0), C.c_int(0)
    _check(lib().pcm_last_cg_matvec_ms(ctx.handle, C.byref(ms), C.byref(n)), ctx.handle)
    return ms.value, n.value


def pcm_launch_count(ctx: Context) -> int:
    n = C.c_int64(0)
    _check(lib().pcm_launch_count(ctx.handle, C.byref(n)), ctx.handle)
    return int(n.value)


def pcm_fp64_peak(ctx: Context, reps: int = 10) -> float:
    t = C.c_double(0.0)
    _check(lib().pcm_fp64_peak(ctx.handle, int(reps), C.byref(t)), ctx.handle)
    return float(t.value)


def pcm_schwarz_bound(la: int, alpha: float, A, lb: int, beta: float, B) -> float:
    out = C.c_double(0.0)
    A = _np(A, np.float64)
    B = _np(B, np.float64)
    _check(lib().pcm_schwarz_bound(int(la), float(alpha), _hp(A), int(lb), float(beta), _hp(B), C.byref(out)))
    return float(out.value)


def pcm_last_error(ctx: Context | None = None) -> str:
    return lib().pcm_last_error(None if ctx is None else ctx.handle).decode("utf-8", "replace")


def pcm_destroy(ctx: Context) -> None:
    if ctx is not None and getattr(ctx, "handle", None):
        h, ctx.handle = ctx.handle, None
        lib().pcm_destroy(h)


def setup_from_workload(basis, surface, **kw) -> Context:
    """Convenience: pcm_setup from synth.Basis / synth.Surface-shaped objects (attribute access only)."""
    return pcm_setup(basis.shell_l, basis.shell_xyz, basis.shell_nprim, basis.prim_exp, basis.prim_coef, surface.xyz,
                     surface.zeta, surface.switch, d_pure=bool(basis.d_pure), **kw)
