"""ctypes front end of the CPU oracle (oracle/pcm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this package.  It never imports ``paper_1505_07851_b200`` and shares no code
with it.  Argument marshalling only: all arithmetic is in pcm_oracle.c, whose header lists the
passages of PAPER.md each function follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pcm_oracle.c")
_LIB = os.path.join(_HERE, "libpcm_oracle.so")
_lib = None

_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_lp = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared -fPIC -o libpcm_oracle.so pcm_oracle.c -lm"""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_boys.argtypes = [C.c_int, C.c_double, _dp]
        L.orc_prim_integral.restype = C.c_double
        L.orc_prim_integral.argtypes = [_ip, C.c_double, _dp, _ip, C.c_double, _dp, C.c_double, _dp, C.c_int]
        L.orc_prim_block.argtypes = [C.c_int, C.c_double, _dp, C.c_int, C.c_double, _dp, C.c_double, _dp, C.c_int, _dp]
        basis = [C.c_int, _ip, _dp, _ip, _dp, _dp, C.c_int]
        L.orc_shell_block.argtypes = basis + [C.c_int, C.c_int, C.c_double, _dp, _dp]
        L.orc_potential.argtypes = basis + [_dp, _dp, _dp, C.c_long, C.c_double, C.c_long, C.c_void_p, _dp]
        L.orc_fock_blocks.argtypes = basis + [C.c_long, _dp, _dp, _dp, C.c_double, C.c_long, _ip, _ip, _dp]
        L.orc_a_entry.restype = C.c_double
        L.orc_a_entry.argtypes = [_dp, _dp, C.c_void_p, C.c_long, C.c_long]
        L.orc_amatrix.argtypes = [C.c_long, _dp, _dp, C.c_void_p, _dp]
        L.orc_amatvec.argtypes = [C.c_long, _dp, _dp, C.c_void_p, _dp, C.c_long, C.c_void_p, _dp]
        L.orc_pivot_order.argtypes = [C.c_uint64, C.c_long, _lp]
        L.orc_rbj_build.restype = C.c_long
        L.orc_rbj_build.argtypes = [C.c_long, _dp, _dp, C.c_void_p, C.c_int, _lp, _lp, _lp, _dp]
        L.orc_pcg.restype = C.c_long
        L.orc_pcg.argtypes = [C.c_long, C.c_void_p, _dp, _dp, C.c_void_p, _dp, _dp, C.c_int, C.c_double, C.c_long,
                              C.c_int, C.c_long, C.c_void_p, C.c_void_p, C.c_void_p, _dp, C.c_void_p]
        L.orc_prim_deriv.argtypes = [C.c_int, C.c_double, _dp, C.c_int, C.c_double, _dp, C.c_double, _dp, _dp, _dp]
        L.orc_gradient.argtypes = basis + [C.c_long, _dp, _dp, _dp, _dp, C.c_long, C.c_double, C.c_long, C.c_void_p,
                                           C.c_long, C.c_void_p, _dp, _dp]
        L.orc_switching.argtypes = [C.c_long, _dp, _dp, _lp, C.c_long, _dp, _dp, _dp]
        L.orc_surface_gradient.argtypes = [C.c_long, _dp, _dp, _lp, C.c_long, _dp, _dp, _dp, _dp, C.c_double, _dp, _dp]
        L.orc_build_cavity.restype = C.c_long
        L.orc_build_cavity.argtypes = [C.c_long, _dp, _dp, C.c_long, _dp, _dp, C.c_double, C.c_double, _dp, _dp, _dp, _lp, _lp]
        L.orc_bz.argtypes = [C.c_long, _dp, _dp, C.c_long, _dp, _dp, _dp]
        L.orc_rhs.argtypes = [C.c_long, _dp, _dp, C.c_double, _dp]
        L.orc_energy.argtypes = [C.c_long, _dp, _dp, _dp, _dp, C.c_double, _dp]
        L.orc_cg_threshold.restype = C.c_double
        L.orc_cg_threshold.argtypes = [C.c_double, C.c_double]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


def _f(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


# ------------------------------------------------------------------ Boys / primitives
def boys(nmax: int, T: float) -> np.ndarray:
    F = np.zeros(nmax + 1)
    lib().orc_boys(int(nmax), float(T), F)
    return F


def prim_integral(a, alpha, A, b, beta, B, zeta, Cpt, path: int = 0) -> float:
    return float(lib().orc_prim_integral(np.asarray(a, np.int32), float(alpha), _f(A), np.asarray(b, np.int32),
                                         float(beta), _f(B), float(zeta), _f(Cpt), int(path)))


_NCART = (1, 3, 6)


def prim_block(la, alpha, A, lb, beta, B, zeta, Cpt, path: int = 0) -> np.ndarray:
    out = np.zeros(_NCART[la] * _NCART[lb])
    lib().orc_prim_block(int(la), float(alpha), _f(A), int(lb), float(beta), _f(B), float(zeta), _f(Cpt), int(path), out)
    return out.reshape(_NCART[la], _NCART[lb])


# ------------------------------------------------------------------ contracted quantities
def _basis_args(basis):
    return (int(basis.nshell), np.ascontiguousarray(basis.shell_l, np.int32), _f(basis.shell_xyz).reshape(-1),
            np.ascontiguousarray(basis.shell_nprim, np.int32), _f(basis.prim_exp), _f(basis.prim_coef),
            1 if basis.d_pure else 0)


def shell_block(basis, I, J, zeta, Cpt) -> np.ndarray:
    nc = basis.ncomp
    out = np.zeros(int(nc[I]) * int(nc[J]))
    lib().orc_shell_block(*_basis_args(basis), int(I), int(J), float(zeta), _f(Cpt), out)
    return out.reshape(int(nc[I]), int(nc[J]))


def potential(basis, surface, P, points=None, cutoff: float = 1e-20) -> np.ndarray:
    """v_k = sum_{mu nu} P_mu,nu (mu|J_k|nu) for the selected points (all if None)."""
    P = _f(P)
    if points is None:
        nsel, sel, selp = surface.M, None, None
    else:
        sel = np.ascontiguousarray(points, np.int64)
        nsel, selp = len(sel), _ptr(sel)
    v = np.zeros(nsel)
    lib().orc_potential(*_basis_args(basis), _f(surface.xyz).reshape(-1), _f(surface.zeta), P, P.shape[1], float(cutoff),
                        nsel, selp, v)
    return v


def fock_blocks(basis, surface, q, pairs, cutoff: float = 1e-20):
    """Blocks F[I,J] = sum_k q_k (mu in I|J_k|nu in J) for the ORDERED shell pairs listed."""
    pairs = np.asarray(pairs, np.int32).reshape(-1, 2)
    pI = np.ascontiguousarray(pairs[:, 0])
    pJ = np.ascontiguousarray(pairs[:, 1])
    nc = basis.ncomp
    sizes = nc[pI].astype(np.int64) * nc[pJ].astype(np.int64)
    out = np.zeros(int(sizes.sum()))
    lib().orc_fock_blocks(*_basis_args(basis), surface.M, _f(surface.xyz).reshape(-1), _f(surface.zeta), _f(q),
                          float(cutoff), len(pI), pI, pJ, out)
    off = np.concatenate([[0], np.cumsum(sizes)])
    return [out[off[n]:off[n + 1]].reshape(int(nc[pI[n]]), int(nc[pJ[n]])) for n in range(len(pI))]


def fock(basis, surface, q, cutoff: float = 1e-20) -> np.ndarray:
    """Dense F over the full square of ordered shell pairs (small cases only)."""
    ns = basis.nshell
    pairs = np.array([(i, j) for i in range(ns) for j in range(ns)], np.int32)
    blocks = fock_blocks(basis, surface, q, pairs, cutoff)
    off = basis.bf_offset
    F = np.zeros((basis.nbf, basis.nbf))
    for (i, j), b in zip(pairs, blocks):
        F[off[i]:off[i + 1], off[j]:off[j + 1]] = b
    return F


# ------------------------------------------------------------------ A matrix, RBJ, PCG
def a_entry(surface, i, j) -> float:
    return float(lib().orc_a_entry(_f(surface.xyz).reshape(-1), _f(surface.zeta), _ptr(_f(surface.switch)), int(i), int(j)))


def amatrix(surface) -> np.ndarray:
    A = np.zeros((surface.M, surface.M))
    sw = _f(surface.switch)
    lib().orc_amatrix(surface.M, _f(surface.xyz).reshape(-1), _f(surface.zeta), _ptr(sw), A.reshape(-1))
    return A


def amatvec(surface, q, rows=None) -> np.ndarray:
    sw = _f(surface.switch)
    if rows is None:
        nsel, sel = surface.M, None
    else:
        sel = np.ascontiguousarray(rows, np.int64)
        nsel = len(sel)
    y = np.zeros(nsel)
    lib().orc_amatvec(surface.M, _f(surface.xyz).reshape(-1), _f(surface.zeta), _ptr(sw), _f(q), nsel, _ptr(sel), y)
    return y


def pivot_order(seed: int, M: int) -> np.ndarray:
    perm = np.zeros(M, np.int64)
    lib().orc_pivot_order(C.c_uint64(seed & 0xFFFFFFFFFFFFFFFF), M, perm)
    return perm


def rbj_build(surface, l: int, pivots: np.ndarray):
    """Returns (order[M], bstart[nb+1], inv blocks list)."""
    M = surface.M
    nbmax = (M + l - 1) // l + 1
    order = np.zeros(M, np.int64)
    bstart = np.zeros(nbmax + 1, np.int64)
    inv = np.zeros(M * l + l * l)
    sw = _f(surface.switch)
    nb = lib().orc_rbj_build(M, _f(surface.xyz).reshape(-1), _f(surface.zeta), _ptr(sw), int(l),
                             np.ascontiguousarray(pivots, np.int64), order, bstart, inv)
    if nb < 0:
        raise RuntimeError("oracle RBJ: a diagonal block is not positive definite")
    return order, bstart[:nb + 1].copy(), inv


def pcg(surface, b, tol, max_iter=1000, precond=0, rbj=None, x0=None, A=None, history=False):
    """Returns (x, iterations, recurrence residual, true residual[, history])."""
    M = surface.M
    x = np.zeros(M) if x0 is None else _f(x0).copy()
    resid = np.zeros(2)
    hist = np.zeros(max_iter + 1) if history else None
    sw = _f(surface.switch)
    if rbj is not None:
        order, bstart, inv = rbj
        nb = len(bstart) - 1
    else:
        order = bstart = inv = None
        nb = 0
    if A is not None:
        A = _f(A)
    it = lib().orc_pcg(M, _ptr(A), _f(surface.xyz).reshape(-1), _f(surface.zeta), _ptr(sw), _f(b), x,
                       0 if x0 is None else 1, float(tol), int(max_iter), int(precond), nb, _ptr(order), _ptr(bstart),
                       _ptr(inv), resid, _ptr(hist))
    out = (x, int(it), float(resid[0]), float(resid[1]))
    if history:
        out = out + (hist[:it + 1].copy(),)
    return out


# ------------------------------------------------------------------ the rest of a C-PCM step (Eq. 1, 4, 13, 21)
def nuclear_potential(surface, atom_xyz, z) -> np.ndarray:
    """u = B z (Eq. 4)."""
    u = np.zeros(surface.M)
    a = _f(atom_xyz).reshape(-1)
    lib().orc_bz(surface.M, _f(surface.xyz).reshape(-1), _f(surface.zeta), len(a) // 3, a, _f(z), u)
    return u


def rhs(u, v, f: float) -> np.ndarray:
    """b = -f (B z - v): the right-hand side of Eq. 1 with c = -v."""
    b = np.zeros(len(u))
    lib().orc_rhs(len(u), _f(u), _f(v), float(f), b)
    return b


def energy(u, v, q, Aq, f: float) -> np.ndarray:
    """Eq. 13: [(B z).q, c.q, q.A q/(2 f), total] with c = -v."""
    out = np.zeros(4)
    lib().orc_energy(len(u), _f(u), _f(v), _f(q), _f(Aq), float(f), out)
    return out


def cg_threshold(diis_prev: float, delta_min: float = 1e-6) -> float:
    """Eq. 21: the dynamic CG threshold for the next SCF iteration (diis_prev <= 0: first iteration, delta = 1)."""
    return float(lib().orc_cg_threshold(float(diis_prev), float(delta_min)))


# ------------------------------------------------------------------ gradient of E = v.q (Eq. 14 / 22, one-electron term)

def prim_deriv(la, alpha, A, lb, beta, B, zeta, Cpt):
    """Cartesian blocks d/dA_x and d/dB_x of [chi_a|J|chi_b]: two arrays [3, NCART[la], NCART[lb]]."""
    n = _NCART[la] * _NCART[lb]
    dA, dB = np.zeros(3 * n), np.zeros(3 * n)
    lib().orc_prim_deriv(int(la), float(alpha), _f(A), int(lb), float(beta), _f(B), float(zeta), _f(Cpt), dA, dB)
    return dA.reshape(3, _NCART[la], _NCART[lb]), dB.reshape(3, _NCART[la], _NCART[lb])


def gradient(basis, surface, P, q, shells=None, points=None, cutoff: float = 1e-20):
    """dE/d(shell centre) [nsel, 3] and dE/d(point position) [nsel, 3] for E = v.q at fixed P and q (the paper's
    (grad* c^T) q is the negative).  shells / points: index lists (None: all)."""
    def sel(x, n):
        if x is None:
            return n, None
        a = np.ascontiguousarray(x, np.int64)
        return len(a), a
    nS, sS = sel(shells, basis.nshell)
    nK, sK = sel(points, surface.M)
    gs, gp = np.zeros((nS, 3)), np.zeros((nK, 3))
    Pm = _f(P)
    lib().orc_gradient(*_basis_args(basis), surface.M, _f(surface.xyz).reshape(-1), _f(surface.zeta), _f(q), Pm.reshape(-1),
                       Pm.shape[1], float(cutoff), nS, _ptr(sS), nK, _ptr(sK), gs.reshape(-1), gp.reshape(-1))
    return gs, gp


# ------------------------------------------------------------------ ISWIG switching function and surface gradient terms
def switching(surface, atom_xyz, atom_radius) -> np.ndarray:
    """S_k of Eq. 9 (product over the atoms that do not own point k; surface.atom is the owner)."""
    S = np.zeros(surface.M)
    a = _f(atom_xyz).reshape(-1)
    own = np.ascontiguousarray(surface.atom, np.int64)
    lib().orc_switching(surface.M, _f(surface.xyz).reshape(-1), _f(surface.zeta), own, len(a) // 3, a, _f(atom_radius), S)
    return S


def surface_gradient(surface, atom_xyz, atom_radius, z, q, f: float):
    """Gradient of (B z).q + q.A q/(2 f) at fixed q (A_kk through the S_k of Eq. 9): (g_point [M, 3], g_atom [N, 3])."""
    a = _f(atom_xyz).reshape(-1)
    n = len(a) // 3
    gp, ga = np.zeros((surface.M, 3)), np.zeros((n, 3))
    own = np.ascontiguousarray(surface.atom, np.int64)
    lib().orc_surface_gradient(surface.M, _f(surface.xyz).reshape(-1), _f(surface.zeta), own, n, a, _f(atom_radius), _f(z), _f(q),
                               float(f), gp.reshape(-1), ga.reshape(-1))
    return gp, ga


# ------------------------------------------------------------------ ISWIG cavity construction (Eq. 7, Eq. 9, the 1e-8 screening)
def build_cavity(atom_xyz, atom_radius, unit_grid, weights, zeta_tab: float, s_min: float = 1e-8):
    """Points r = R_I + rad_I u_g of every atom with zeta = zeta_tab/(rad_I sqrt(w_g)) (Eq. 7) and S of Eq. 9, those with
    S >= s_min kept, atom after atom.  Returns (synth-shaped surface fields) xyz [n,3], zeta [n], S [n],
    atom [n], node [n]."""
    a = _f(atom_xyz).reshape(-1)
    N = len(a) // 3
    u = _f(unit_grid).reshape(-1)
    G = len(u) // 3
    cap = max(N * G, 1)
    xyz, zeta, S = np.zeros(3 * cap), np.zeros(cap), np.zeros(cap)
    own, node = np.zeros(cap, np.int64), np.zeros(cap, np.int64)
    n = lib().orc_build_cavity(N, a, _f(atom_radius), G, u, _f(weights), float(zeta_tab), float(s_min), xyz, zeta, S, own, node)
    return xyz[:3 * n].reshape(n, 3).copy(), zeta[:n].copy(), S[:n].copy(), own[:n].copy(), node[:n].copy()
