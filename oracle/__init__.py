"""ORACLE — TEST INFRASTRUCTURE ONLY.

ctypes binding of the plain single-threaded C++ oracle in this directory (see orc.hpp for
what it is and what pins it). Only tests/, __graft_entry__.smoke() and the cpu_baseline /
--impl reference legs of bench.py may import this package. It imports nothing from the
CUDA product (paper_2510_13965_b200) and the product imports nothing from here.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SOURCES = ["orc_stencil.cpp", "orc_eos.cpp", "orc_c2p.cpp", "orc_ccz4.cpp", "orc_grmhd.cpp",
            "orc_rk.cpp", "orc_m1.cpp", "orc_m1_patch.cpp", "orc_amr.cpp", "orc_les.cpp", "orc_capi.cpp"]
_LIB = os.path.join(_HERE, "liboracle.so")

NSTATE, NPRIM = 32, 10
# field indices (mirror orc.hpp)
GXX, AXX, CHI, KHAT, THETA, GAMX, ALPHA, BETAX = 0, 6, 12, 13, 14, 15, 18, 19
DBAR, DYEBAR, TAUBAR, SXBAR, BXBAR, PHIBAR = 22, 23, 24, 25, 28, 31
RHO, YE, EPS, PRESS, VX, WLOR, TEMP, CS2 = 0, 1, 2, 3, 4, 7, 8, 9


def build(force=False):
    """Compile liboracle.so with g++ -O2 -ffp-contract=off (no FMA contraction)."""
    srcs = [os.path.join(_HERE, s) for s in _SOURCES]
    deps = srcs + [os.path.join(_HERE, "orc.hpp")]
    if not force and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in deps):
        return _LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wno-unknown-pragmas", "-o", _LIB] + srcs
    subprocess.run(cmd, check=True)
    return _LIB


_LIB_OMP = os.path.join(_HERE, "liboracle_omp.so")


def build_omp(force=False):
    """The same sources with -fopenmp: the outermost grid loops run on several host cores, the arithmetic of every point is
    unchanged (results are bit-identical to the plain build)."""
    srcs = [os.path.join(_HERE, s) for s in _SOURCES]
    deps = srcs + [os.path.join(_HERE, "orc.hpp")]
    if not force and os.path.exists(_LIB_OMP) and all(os.path.getmtime(_LIB_OMP) >= os.path.getmtime(d) for d in deps):
        return _LIB_OMP
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _LIB_OMP] + srcs
    subprocess.run(cmd, check=True)
    return _LIB_OMP


_LIB_COUNT = os.path.join(_HERE, "liboracle_count.so")


def build_counting(force=False):
    """Operation-counting build (orc_count.cpp: the same sources with `double` replaced by a counting wrapper)."""
    deps = [os.path.join(_HERE, s) for s in _SOURCES + ["orc.hpp", "orc_count.cpp"]]
    if not force and os.path.exists(_LIB_COUNT) and all(os.path.getmtime(_LIB_COUNT) >= os.path.getmtime(d) for d in deps):
        return _LIB_COUNT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB_COUNT, os.path.join(_HERE, "orc_count.cpp")]
    subprocess.run(cmd, check=True)
    return _LIB_COUNT


_libs = {}
_counting = False
_threads = 1


def use_threads(n):
    """n = 1: the plain single-threaded build (the default, and what `cpu_baseline` quotes first); n > 1: the -fopenmp build on
    n host cores. Returns the thread count in effect."""
    global _threads
    _threads = max(1, int(n))
    if _threads > 1:
        return int(_load("omp").orc_set_threads(_threads))
    return 1


def use_counting(flag):
    """Route every call of this module through the operation-counting library (for the F_alg measurement)."""
    global _counting
    _counting = bool(flag)


def count_reset():
    _load(True).orc_count_reset()


def count_get():
    """dict of operation counts since the last reset: add (incl. sub), mul, div, sqrt, cmp (incl. min/max), trans"""
    out = (ctypes.c_ulonglong * 6)()
    _load(True).orc_count_get(out)
    return dict(zip(("add", "mul", "div", "sqrt", "cmp", "trans"), [int(v) for v in out]))


def lib():
    return _load(True if _counting else ("omp" if _threads > 1 else False))


def _load(counting):
    if counting not in _libs:
        _libs[counting] = ctypes.CDLL(build_omp() if counting == "omp" else (build_counting() if counting else build()))
        L = _libs[counting]
        dp, vp, i32, f64 = ctypes.POINTER(ctypes.c_double), ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.orc_new.restype = vp
        L.orc_set_threads.argtypes = [i32]
        L.orc_set_threads.restype = i32
        L.orc_free.argtypes = [vp]
        L.orc_set.argtypes = [vp, ctypes.c_char_p, f64]
        L.orc_set_array.argtypes = [vp, ctypes.c_char_p, vp, i32]
        L.orc_set_table.argtypes = [vp, vp, vp, vp]
        L.orc_finalize.argtypes = [vp]
        L.orc_set_grid.argtypes = [vp, i32, i32, i32, i32, f64, f64, f64]
        L.orc_fill_ghosts.argtypes = [vp, vp, i32, vp]
        L.orc_con2prim.argtypes = [vp, vp, vp, vp]
        L.orc_prim2con.argtypes = [vp, vp, vp]
        for name in ("orc_rhs", "orc_rhs_ccz4", "orc_rhs_grmhd", "orc_rhs_grmhd_flux", "orc_rhs_grmhd_src"):
            getattr(L, name).argtypes = [vp, vp, vp, vp]
        L.orc_rk_combine.argtypes = [vp, i32, vp, vp, i32, vp, vp, f64]
        L.orc_evolve.argtypes = [vp, vp, vp, vp, vp, i32, vp, vp, f64, i32]
        for name, n in (("orc_d1", 1), ("orc_d2", 1)):
            getattr(L, name).argtypes = [vp, ctypes.c_long, f64]
            getattr(L, name).restype = f64
        L.orc_d11.argtypes = [vp, ctypes.c_long, f64, ctypes.c_long, f64]
        L.orc_d11.restype = f64
        L.orc_dadv.argtypes = [vp, ctypes.c_long, f64, f64]
        L.orc_dadv.restype = f64
        L.orc_dko.argtypes = [vp, ctypes.c_long, f64, f64]
        L.orc_dko.restype = f64
        L.orc_mp5.argtypes = [f64] * 6
        L.orc_mp5.restype = f64
        L.orc_weno5.argtypes = [f64] * 6
        L.orc_weno5.restype = f64
        L.orc_eos.argtypes = [vp, f64, f64, f64, vp]
        L.orc_eos_eps_from_T.argtypes = [vp, f64, f64, f64]
        L.orc_eos_eps_from_T.restype = f64
        L.orc_con2prim_point.argtypes = [vp, vp, f64, f64, vp, vp]
        L.orc_con2prim_point.restype = i32
        L.orc_prim2con_point.argtypes = [vp, vp, vp, vp]
        L.orc_m1_closure_point.argtypes = [f64, vp, vp, f64, vp, vp, vp]
        L.orc_m1_JH.argtypes = [f64, vp, vp, f64, vp, vp, f64, f64, vp]
        L.orc_m1_jacobian.argtypes = [f64, vp, vp, f64, vp, vp, f64, f64, f64, f64, f64, vp]
        L.orc_m1_implicit_point.argtypes = [vp, i32, vp, f64, f64, vp, f64, f64, f64, vp, vp, vp, vp]
        L.orc_m1_implicit_point.restype = i32
        L.orc_m1_rhs.argtypes = [vp, vp, vp, vp, vp]
        L.orc_m1_implicit.argtypes = [vp, vp, vp, vp, vp, f64, vp]
        L.orc_m1_backreaction.argtypes = [vp, vp, vp, vp, vp]
        L.orc_m1_gravity.argtypes = [vp, vp, vp, vp, vp]
        L.orc_evolve_imex.argtypes = [vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, f64, i32]
        L.orc_eos_dp.argtypes = [vp, f64, f64, f64, vp]
        L.orc_les_flux.argtypes = [vp, vp, vp, vp, vp]
        L.orc_les_HM_point.argtypes = [vp, vp, vp, f64, vp]
        L.orc_les_H_point.argtypes = [vp, vp, vp, vp, f64, f64, vp, vp, vp, vp]
        L.orc_les_aux_point.argtypes = [vp, vp, f64, vp, vp, vp]
        L.orc_prolong.argtypes = [vp, i32, vp, vp, i32, vp, i32, vp, vp, vp]
        L.orc_restrict.argtypes = [vp, i32, vp, vp, i32, vp, i32, vp]
        L.orc_dense_weights.argtypes = [i32, f64, i32, vp]
        L.orc_dense_weights.restype = i32
        L.orc_dense_output.argtypes = [vp, i32, vp, vp, i32, vp, f64, f64, i32]
        L.orc_prolong_mid.argtypes = [vp, ctypes.c_long]
        L.orc_prolong_mid.restype = f64
    return _libs[counting]


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


class Oracle:
    """One oracle instance = parameters + grid. Arrays are numpy float64, SoA (field, k, j, i)."""

    def __init__(self, params, nx, ny, nz, ng, dx, dy=None, dz=None, table=None):
        L = lib()
        self.h = L.orc_new()
        self._keep = []
        for k, v in params.items():
            if isinstance(v, (list, tuple, np.ndarray)):
                arr = _f64(v)
                if L.orc_set_array(self.h, k.encode(), _ptr(arr), arr.size) != 0:
                    raise KeyError(k)
            elif L.orc_set(self.h, k.encode(), float(v)) != 0:
                raise KeyError(k)
        if table is not None:
            for k in ("n_rho", "n_T", "n_ye", "lr0", "dlr", "lT0", "dlT", "ye0", "dye", "tab_eps_shift", "tab_h0"):
                L.orc_set(self.h, k.encode(), float(table[k]))
            self._keep = [_f64(table["logp"]), _f64(table["loge"]), _f64(table["cs2"])]
            L.orc_set_table(self.h, *[_ptr(a) for a in self._keep])
        L.orc_finalize(self.h)
        dy = dx if dy is None else dy
        dz = dx if dz is None else dz
        L.orc_set_grid(self.h, nx, ny, nz, ng, dx, dy, dz)
        self.shape = (nz + 2 * ng, ny + 2 * ng, nx + 2 * ng)
        self.npts = int(np.prod(self.shape))
        self.ng = ng

    def __del__(self):
        try:
            lib().orc_free(self.h)
        except Exception:
            pass

    def fill_ghosts(self, U, bc):
        assert U.dtype == np.float64 and U.flags.c_contiguous
        b = np.asarray(bc, dtype=np.int32)
        lib().orc_fill_ghosts(self.h, _ptr(U), U.shape[0], _ptr(b))
        return U

    def con2prim(self, U):
        P = np.zeros((NPRIM,) + self.shape)
        flags = np.zeros(self.shape, dtype=np.uint8)
        lib().orc_con2prim(self.h, _ptr(U), _ptr(P), _ptr(flags))
        return P, flags

    def prim2con(self, U, P):
        """P: rho, Ye, eps, v^i given; fills p, W, T, cs2 in P and the fluid conserved fields in U (in place)."""
        assert P.dtype == np.float64 and P.flags.c_contiguous and U.flags.c_contiguous
        lib().orc_prim2con(self.h, _ptr(U), _ptr(P))
        return U, P

    def rhs(self, U, P, part="all"):
        K = np.zeros_like(U)
        fn = {"all": "orc_rhs", "ccz4": "orc_rhs_ccz4", "grmhd": "orc_rhs_grmhd", "grmhd_flux": "orc_rhs_grmhd_flux",
              "grmhd_src": "orc_rhs_grmhd_src"}[part]
        getattr(lib(), fn)(self.h, _ptr(U), _ptr(P), _ptr(K))
        return K

    def rk_combine(self, U0, Ks, coef, dt):
        out = U0.copy()
        ptrs = (ctypes.c_void_p * len(Ks))(*[k.ctypes.data for k in Ks])
        c = _f64(coef)
        lib().orc_rk_combine(self.h, U0.shape[0], _ptr(out), _ptr(U0), len(Ks), ptrs, _ptr(c), float(dt))
        return out

    def evolve(self, U, bc, a_expl, w_expl, dt, n_steps):
        """Advance U in place by n_steps full RK steps; returns (P, flags) of the final state."""
        P = np.zeros((NPRIM,) + self.shape)
        flags = np.zeros(self.shape, dtype=np.uint8)
        a = _f64(a_expl)
        w = _f64(w_expl)
        b = np.asarray(bc, dtype=np.int32)
        lib().orc_evolve(self.h, _ptr(U), _ptr(P), _ptr(flags), _ptr(b), len(w), _ptr(a), _ptr(w), float(dt), int(n_steps))
        return P, flags

    def eos(self, rho, eps, ye=0.3):
        out = np.zeros(3)
        lib().orc_eos(self.h, rho, eps, ye, _ptr(out))
        return out  # p, T, cs2

    def eps_from_T(self, rho, T, ye):
        return lib().orc_eos_eps_from_T(self.h, rho, T, ye)

    def con2prim_point(self, gt, chi, alpha, ucons):
        gt = _f64(gt)
        uc = _f64(ucons).copy()
        prim = np.zeros(NPRIM)
        flag = lib().orc_con2prim_point(self.h, _ptr(gt), chi, alpha, _ptr(uc), _ptr(prim))
        return prim, flag, uc


def prim2con_point(gl, prim, B):
    out = np.zeros(5)
    lib().orc_prim2con_point(_ptr(_f64(gl)), _ptr(_f64(prim)), _ptr(_f64(B)), _ptr(out))
    return out  # D, tau, S_x, S_y, S_z


def stencil(name, u, s, h, *extra):
    """Apply one oracle stencil at the centre element of the 1-D/2-D numpy array u (for the pins)."""
    u = _f64(u)
    L = lib()
    flat = u.reshape(-1)
    c = flat.size // 2
    p = ctypes.c_void_p(flat.ctypes.data + 8 * c)
    return getattr(L, "orc_" + name)(p, s, h, *extra)


# ---- M1 (config 5) ------------------------------------------------------------------------------------------
NM1 = 15


def m1_closure_point(E, F, vu, W, gl, gu):
    """Eqs. (42)-(50) at one point; gl, gu 3x3 physical metric and inverse. Returns dict xi, chi, J, Hn, H (3), P (3x3)."""
    out = np.zeros(16)
    lib().orc_m1_closure_point(float(E), _ptr(_f64(F)), _ptr(_f64(vu)), float(W), _ptr(_f64(gl)), _ptr(_f64(gu)), _ptr(out))
    return dict(xi=out[0], chi=out[1], J=out[2], Hn=out[3], H=out[4:7].copy(), P=out[7:16].reshape(3, 3).copy())


def m1_JH(E, F, vu, W, gl, gu, dthin, dthick):
    out = np.zeros(4)
    lib().orc_m1_JH(float(E), _ptr(_f64(F)), _ptr(_f64(vu)), float(W), _ptr(_f64(gl)), _ptr(_f64(gu)), float(dthin), float(dthick), _ptr(out))
    return out[0], out[1:4].copy()


def m1_jacobian(E, F, vu, W, gl, gu, dthin, dthick, alpha, ka, ks):
    out = np.zeros(16)
    lib().orc_m1_jacobian(float(E), _ptr(_f64(F)), _ptr(_f64(vu)), float(W), _ptr(_f64(gl)), _ptr(_f64(gu)), float(dthin), float(dthick),
                          float(alpha), float(ka), float(ks), _ptr(out))
    return out.reshape(4, 4)


def _m1_implicit_point(self, species, Vstar, adt, alpha, vu, W, rho, T, gl, gu):
    V, R = np.zeros(5), np.zeros(5)
    flag = lib().orc_m1_implicit_point(self.h, int(species), _ptr(_f64(Vstar)), float(adt), float(alpha), _ptr(_f64(vu)), float(W), float(rho),
                                       float(T), _ptr(_f64(gl)), _ptr(_f64(gu)), _ptr(V), _ptr(R))
    return V, R, flag


def _m1_rhs(self, U, P, V):
    KV = np.zeros_like(V)
    lib().orc_m1_rhs(self.h, _ptr(U), _ptr(P), _ptr(V), _ptr(KV))
    return KV


def _m1_implicit(self, U, P, V, adt, flags=None):
    """V: V* in, V^(i) out (in place). Returns (R, flags)."""
    R = np.zeros_like(V)
    fl = np.zeros(self.shape, dtype=np.uint8) if flags is None else flags
    lib().orc_m1_implicit(self.h, _ptr(U), _ptr(P), _ptr(V), _ptr(R), float(adt), _ptr(fl))
    return R, fl


def _m1_backreaction(self, U, P, R, K):
    lib().orc_m1_backreaction(self.h, _ptr(U), _ptr(P), _ptr(R), _ptr(K))
    return K


def _m1_gravity(self, U, P, V, K):
    """adds the radiation terms of the CCZ4 matter sources (R6) to K in place"""
    lib().orc_m1_gravity(self.h, _ptr(U), _ptr(P), _ptr(V), _ptr(K))
    return K


def _evolve_imex(self, U, V, bc, a_expl, w_expl, a_impl, w_impl, dt, n_steps):
    P = np.zeros((NPRIM,) + self.shape)
    flags = np.zeros(self.shape, dtype=np.uint8)
    ae, we, ai, wi = _f64(a_expl), _f64(w_expl), _f64(a_impl), _f64(w_impl)
    b = np.asarray(bc, dtype=np.int32)
    lib().orc_evolve_imex(self.h, _ptr(U), _ptr(V), _ptr(P), _ptr(flags), _ptr(b), len(we), _ptr(ae), _ptr(we), _ptr(ai), _ptr(wi), float(dt), int(n_steps))
    return P, flags


Oracle.m1_implicit_point = _m1_implicit_point
Oracle.m1_rhs = _m1_rhs
Oracle.m1_implicit = _m1_implicit
Oracle.m1_backreaction = _m1_backreaction
Oracle.m1_gravity = _m1_gravity
Oracle.evolve_imex = _evolve_imex


# ---- AMR transfer operators on a patch pair -----------------------------------------------------
def _i3(v):
    return np.asarray(v, dtype=np.int32)


def prolong(Uc, ngc, Uf, ngf, origin, lo, hi):
    """Fill the index box [lo, hi) (x, y, z; ghosted fine array indices) of the fine array Uf (fields, MZ, MY, MX) from the coarse array
    Uc by Eq. (80) / copy; origin = coarse interior index (x, y, z) of the coarse point under fine interior point (0, 0, 0)."""
    nc = _i3([Uc.shape[3] - 2 * ngc, Uc.shape[2] - 2 * ngc, Uc.shape[1] - 2 * ngc])
    nf = _i3([Uf.shape[3] - 2 * ngf, Uf.shape[2] - 2 * ngf, Uf.shape[1] - 2 * ngf])
    o, l, h = _i3(origin), _i3(lo), _i3(hi)
    lib().orc_prolong(_ptr(nc), ngc, _ptr(Uc), _ptr(nf), ngf, _ptr(Uf), Uc.shape[0], _ptr(o), _ptr(l), _ptr(h))
    return Uf


def restrict(Uf, ngf, Uc, ngc, origin):
    """Copy the even fine interior points onto the coarse points they coincide with (l.626)."""
    nc = _i3([Uc.shape[3] - 2 * ngc, Uc.shape[2] - 2 * ngc, Uc.shape[1] - 2 * ngc])
    nf = _i3([Uf.shape[3] - 2 * ngf, Uf.shape[2] - 2 * ngf, Uf.shape[1] - 2 * ngf])
    o = _i3(origin)
    lib().orc_restrict(_ptr(nf), ngf, _ptr(Uf), _ptr(nc), ngc, _ptr(Uc), Uc.shape[0], _ptr(o))
    return Uc


def dense_weights(scheme, theta, deriv=0):
    """b_j(theta) of Eq. (58) (scheme 0, RK4) / Eq. (59) (scheme 1, SSP-RK3) or their deriv-th theta-derivative (Eq. 57)"""
    b = np.zeros(4)
    s = lib().orc_dense_weights(int(scheme), float(theta), int(deriv), _ptr(b))
    return b[:s].copy()


def _dense_output(self, U0, Ks, scheme, theta, dt, deriv=0):
    out = U0.copy()
    ptrs = (ctypes.c_void_p * len(Ks))(*[k.ctypes.data for k in Ks])
    lib().orc_dense_output(self.h, U0.shape[0], _ptr(out), _ptr(U0), int(scheme), ptrs, float(theta), float(dt), int(deriv))
    return out


Oracle.dense_output = _dense_output


# ---- LES gradient SGS term of the induction equation (App. A) ------------------------------------------
LES_NAUX = 31
LES_NFLUX = 24
LES_NAMES = ["Bu0", "Bu1", "Bu2", "vu0", "vu1", "vu2", "vl0", "vl1", "vl2", "Bl0", "Bl1", "Bl2", "El0", "El1", "El2", "Eu0", "Eu1", "Eu2",
             "vB", "Theta", "Wm2", "rho", "eps", "h", "dpdrho", "dpdeps", "Ye", "dpdYe", "D", "calE", "DYe"]


def les_HM_point(a, da, gu, p):
    """H_M^{ki} (first index = flux direction) from the 26 auxiliary fields a, their partial derivatives da[m][f], gamma^{ij}, pressure"""
    out = np.zeros(9)
    lib().orc_les_HM_point(_ptr(_f64(a)), _ptr(_f64(da)), _ptr(_f64(gu)), float(p), _ptr(out))
    return out.reshape(3, 3)


def les_H_point(a, da, gu, gl, sqrtg, p):
    """(H_M^{ki}, H_N^k, H_{N_Y}^k, H_T^{ki}) of (A15)-(A17) at one point (first index of H_M = flux direction)"""
    HM, HN, HNY, HT = np.zeros(9), np.zeros(3), np.zeros(3), np.zeros(9)
    lib().orc_les_H_point(_ptr(_f64(a)), _ptr(_f64(da)), _ptr(_f64(gu)), _ptr(_f64(gl)), float(sqrtg), float(p), _ptr(HM), _ptr(HN), _ptr(HNY), _ptr(HT))
    return HM.reshape(3, 3), HN, HNY, HT.reshape(3, 3)


def _les_aux_point(self, gl, sqrtg, Bu, prim):
    out = np.zeros(LES_NAUX)
    lib().orc_les_aux_point(self.h, _ptr(_f64(gl)), float(sqrtg), _ptr(_f64(Bu)), _ptr(_f64(prim)), _ptr(out))
    return out


def _les_flux(self, U, P):
    """(L, A): L[3 k + i] = -alpha G_B^{ki}, the SGS part of the k-flux of Bbar^i (zero within 2 points of the array edge); A = auxiliary fields"""
    L = np.zeros((LES_NFLUX,) + self.shape)
    A = np.zeros((LES_NAUX,) + self.shape)
    lib().orc_les_flux(self.h, _ptr(U), _ptr(P), _ptr(L), _ptr(A))
    return L, A


def _eos_dp(self, rho, eps, ye=0.3):
    """(dp/drho at fixed eps, Ye; dp/deps at fixed rho, Ye; dp/dYe at fixed rho, eps)"""
    out = np.zeros(3)
    lib().orc_eos_dp(self.h, float(rho), float(eps), float(ye), _ptr(out))
    return out


Oracle.eos_dp = _eos_dp
Oracle.les_aux_point = _les_aux_point
Oracle.les_flux = _les_flux
