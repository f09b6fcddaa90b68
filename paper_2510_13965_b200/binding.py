"""Thin ctypes binding of libmhd_b200.so (include/mhd.h). Argument marshalling only: every step of the hot
path runs in the library's CUDA kernels. PyTorch is used for device memory and streams, nothing else.

The module-level functions carry the C names (mhd_patch_create, mhd_fill_ghosts, mhd_con2prim, mhd_rhs,
mhd_rk_stage, ...). `Patch` is a convenience owner of the torch tensors bound to the slots.
There is no fallback: if the shared library is missing or fails to load, importing `lib()` raises.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmhd_b200.so")

NSTATE, NPRIM, NWORK, MAX_STAGES, MAX_PIECES = 32, 10, 33, 8, 8
SLOT_U, SLOT_U0, SLOT_P, SLOT_FLAGS, SLOT_WORK, SLOT_K1 = 0, 1, 2, 3, 4, 5
NM1, NM1WORK = 15, 75
SLOT_V, SLOT_V0, SLOT_M1WORK, SLOT_KV1, SLOT_R1, SLOT_U1, SLOT_LESWORK = 13, 14, 15, 16, 24, 32, 33
NLESWORK = 31
OK = 0

_d, _i, _p = ctypes.c_double, ctypes.c_int, ctypes.c_void_p


class mhd_patch_desc(ctypes.Structure):
    _fields_ = [
        ("nx", _i), ("ny", _i), ("nz", _i), ("ng", _i),
        ("dx", _d), ("dy", _d), ("dz", _d),
        ("n_species", _i), ("eos_kind", _i),
        ("eos_gamma", _d), ("eos_gamma_th", _d),
        ("n_pieces", _i),
        ("pp_K", _d * MAX_PIECES), ("pp_Gamma", _d * MAX_PIECES), ("pp_rho", _d * MAX_PIECES),
        ("tab_logp", _p), ("tab_loge", _p), ("tab_cs2", _p),
        ("n_rho", _i), ("n_T", _i), ("n_ye", _i),
        ("lr0", _d), ("dlr", _d), ("lT0", _d), ("dlT", _d), ("ye0", _d), ("dye", _d), ("tab_eps_shift", _d), ("tab_h0", _d),
        ("kappa_z", _d), ("kappa_c", _d), ("kappa_2", _d), ("eta_shift", _d), ("f_alpha", _d), ("f_beta", _d), ("beta0", _d * 3),
        ("grav_G", _d), ("sigma_ko_spacetime", _d), ("sigma_ko_matter", _d),
        ("c_b", _d), ("kappa_b", _d), ("mp5_alpha", _d),
        ("rho_atmo", _d), ("rho_cut", _d), ("rho_low", _d), ("alpha_bh", _d), ("w_max", _d), ("rho_max", _d),
        ("eps_min", _d), ("eps_max", _d), ("ye_min", _d), ("ye_max", _d), ("ye_atmo", _d), ("eps_atmo", _d), ("T_atmo", _d),
        ("c2p_maxit", _i),
        ("m1_kappa0", _d), ("m1_rho0", _d), ("m1_species_scale", _d * 3), ("m1_efloor", _d), ("m1_tol", _d), ("m1_mb", _d),
        ("m1_maxit", _i), ("m1_odd_even", _i),
        ("m1_arad", _d), ("m1_oe_guard", _d),
        ("recon_kind", _i), ("weno_eps", _d), ("les_C_M", _d), ("les_C_N", _d), ("les_C_Y", _d), ("les_C_T", _d),
    ]


class mhd_tableau(ctypes.Structure):
    _fields_ = [("stages", _i), ("a_expl", _p), ("w_expl", _p), ("a_impl", _p), ("w_impl", _p)]


class mhd_status(ctypes.Structure):
    _fields_ = [(n, ctypes.c_ulonglong) for n in
                ("n_points", "n_atmo", "n_eps_lo", "n_eps_hi", "n_vmax", "n_ye", "n_fatal", "n_noconv", "n_m1fix", "halo_timeout")]


EXPORTS = ["mhd_desc_sizeof", "mhd_patch_create", "mhd_patch_destroy", "mhd_patch_bind", "mhd_fill_ghosts", "mhd_con2prim",
           "mhd_prim2con", "mhd_rhs", "mhd_rk_stage", "mhd_advance", "mhd_advance_host", "mhd_patch_status",
           "mhd_patch_profile", "mhd_patch_profile_read", "mhd_probe_fp64_flops", "mhd_strerror",
           "mhd_m1_implicit", "mhd_m1_rhs", "mhd_m1_backreaction", "mhd_m1_gravity", "mhd_advance_imex",
           "mhd_prolong", "mhd_restrict", "mhd_dense_weights", "mhd_dense_output",
           "mhd_advance_imex_host", "mhd_les_flux", "mhd_patch_set_neighbor", "mhd_patch_halo_words", "mhd_patch_set_neighbor_word", "mhd_ipc_export", "mhd_ipc_import", "mhd_ipc_close", "mhd_flag_census_static"]
NKERNELS = 13
KERNEL_CLASSES = ["fill_ghosts", "con2prim", "ccz4_algebra", "recon_x", "recon_y", "recon_z", "rk_combine", "point_flux", "adv_ko",
                  "m1_point", "m1_div", "m1_implicit", "les"]

_lib = None


def lib():
    """Load libmhd_b200.so (fails loudly if it has not been built: python -m paper_2510_13965_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libmhd_b200.so not built; run `python -m paper_2510_13965_b200.build` (no CPU fallback exists)")
        L = ctypes.CDLL(LIB_PATH)
        L.mhd_desc_sizeof.restype = ctypes.c_size_t
        L.mhd_patch_create.argtypes = [ctypes.POINTER(mhd_patch_desc), ctypes.POINTER(_p)]
        L.mhd_patch_destroy.argtypes = [_p]
        L.mhd_patch_destroy.restype = None
        L.mhd_patch_bind.argtypes = [_p, _i, _p, ctypes.c_size_t]
        L.mhd_fill_ghosts.argtypes = [_p, _i, ctypes.POINTER(_i), _p]
        L.mhd_con2prim.argtypes = [_p, _i, _i, _i, _p]
        L.mhd_prim2con.argtypes = [_p, _i, _i, _p]
        L.mhd_rhs.argtypes = [_p, _i, _i, _i, _p]
        L.mhd_rk_stage.argtypes = [_p, ctypes.POINTER(mhd_tableau), _i, _d, _p]
        L.mhd_advance.argtypes = [_p, ctypes.POINTER(mhd_tableau), ctypes.POINTER(_i), _d, _i, _p]
        L.mhd_advance_host.argtypes = [_p, ctypes.POINTER(mhd_tableau), ctypes.POINTER(_i), _d, _i, _p, _p, _p]
        L.mhd_patch_status.argtypes = [_p, _i, ctypes.POINTER(mhd_status), _p]
        L.mhd_patch_profile.argtypes = [_p, _i]
        L.mhd_patch_profile_read.argtypes = [_p, ctypes.POINTER(_d), ctypes.POINTER(ctypes.c_ulonglong), _p]
        L.mhd_probe_fp64_flops.argtypes = [_p]
        L.mhd_probe_fp64_flops.restype = _d
        L.mhd_strerror.argtypes = [_i]
        L.mhd_flag_census_static.argtypes = [_p, ctypes.c_longlong, _p, _p]
        L.mhd_m1_implicit.argtypes = [_p, _i, _i, _d, _p]
        L.mhd_m1_rhs.argtypes = [_p, _i, _i, _p]
        L.mhd_m1_backreaction.argtypes = [_p, _i, _i, _p]
        L.mhd_m1_gravity.argtypes = [_p, _i, _i, _p]
        L.mhd_advance_imex.argtypes = [_p, ctypes.POINTER(mhd_tableau), ctypes.POINTER(_i), _d, _i, _p]
        L.mhd_strerror.restype = ctypes.c_char_p
        L.mhd_les_flux.argtypes = [_p, _i, _i, _p]
        L.mhd_advance_imex_host.argtypes = [_p, ctypes.POINTER(mhd_tableau), ctypes.POINTER(_i), _d, _i, _p, _p, _p, _p]
        L.mhd_patch_set_neighbor.argtypes = [_p, _i, ctypes.POINTER(_i), _p, ctypes.c_size_t]
        L.mhd_patch_halo_words.argtypes = [_p]
        L.mhd_patch_halo_words.restype = _p
        L.mhd_patch_set_neighbor_word.argtypes = [_p, ctypes.POINTER(_i), _p]
        L.mhd_ipc_export.argtypes = [_p, ctypes.c_char_p, ctypes.POINTER(ctypes.c_size_t)]
        L.mhd_ipc_import.argtypes = [ctypes.c_char_p, ctypes.c_size_t, ctypes.POINTER(_p)]
        L.mhd_ipc_close.argtypes = [_p, ctypes.c_size_t]
        L.mhd_prolong.argtypes = [_p, _i, _p, _i, ctypes.POINTER(_i), ctypes.POINTER(_i), ctypes.POINTER(_i), _p]
        L.mhd_restrict.argtypes = [_p, _i, _p, _i, ctypes.POINTER(_i), _p]
        L.mhd_dense_weights.argtypes = [_i, _d, _i, ctypes.POINTER(_d)]
        L.mhd_dense_output.argtypes = [_p, _i, _d, _d, _i, _i, _p]
        if L.mhd_desc_sizeof() != ctypes.sizeof(mhd_patch_desc):
            raise RuntimeError("mhd_patch_desc layout mismatch between include/mhd.h and binding.py")
        _lib = L
    return _lib


class MhdError(RuntimeError):
    pass


def _check(rc):
    if rc != OK:
        raise MhdError("libmhd_b200: %s (%d)" % (lib().mhd_strerror(rc).decode(), rc))


def make_desc(params, nx, ny, nz, ng, dx, dy=None, dz=None, table_ptrs=None, table=None, n_species=0):
    """Marshal a parameter dictionary (paper_2510_13965_b200.synth.default_params) into mhd_patch_desc."""
    d = mhd_patch_desc()
    d.nx, d.ny, d.nz, d.ng = nx, ny, nz, ng
    d.dx, d.dy, d.dz = dx, dx if dy is None else dy, dx if dz is None else dz
    d.n_species = n_species
    names = {f[0] for f in mhd_patch_desc._fields_}
    for k, v in params.items():
        if k not in names:
            raise KeyError(k)
        if isinstance(v, (list, tuple, np.ndarray)):
            arr = getattr(d, k)
            for i, x in enumerate(v):
                arr[i] = float(x)
        elif k in ("eos_kind", "n_pieces", "c2p_maxit", "m1_maxit", "m1_odd_even", "recon_kind"):
            setattr(d, k, int(v))
        else:
            setattr(d, k, float(v))
    if table is not None:
        for k in ("n_rho", "n_T", "n_ye"):
            setattr(d, k, int(table[k]))
        for k in ("lr0", "dlr", "lT0", "dlT", "ye0", "dye", "tab_eps_shift", "tab_h0"):
            setattr(d, k, float(table[k]))
        d.tab_logp, d.tab_loge, d.tab_cs2 = table_ptrs
    return d


def make_tableau(a_expl, w_expl, a_impl=None, w_impl=None):
    a = np.ascontiguousarray(a_expl, dtype=np.float64)
    w = np.ascontiguousarray(w_expl, dtype=np.float64)
    t = mhd_tableau()
    t.stages = len(w)
    t.a_expl, t.w_expl, t.a_impl, t.w_impl = a.ctypes.data, w.ctypes.data, None, None
    t._keep = (a, w)
    if a_impl is not None:
        ai = np.ascontiguousarray(a_impl, dtype=np.float64)
        wi = np.ascontiguousarray(w_impl, dtype=np.float64)
        t.a_impl, t.w_impl = ai.ctypes.data, wi.ctypes.data
        t._keep = (a, w, ai, wi)
    return t


# ---- C-named entry points (argument marshalling only) ---------------------------------------------------
def mhd_patch_create(desc):
    h = _p()
    _check(lib().mhd_patch_create(ctypes.byref(desc), ctypes.byref(h)))
    return h


def mhd_patch_destroy(h):
    lib().mhd_patch_destroy(h)


def mhd_patch_bind(h, slot, dev_ptr, field_stride):
    _check(lib().mhd_patch_bind(h, slot, dev_ptr, field_stride))


def _bc(bc):
    return (_i * 6)(*[int(b) for b in bc])


def mhd_fill_ghosts(h, slot_state, bc, stream=None):
    _check(lib().mhd_fill_ghosts(h, slot_state, _bc(bc), stream))


def mhd_con2prim(h, slot_state=SLOT_U, slot_prim=SLOT_P, slot_flags=SLOT_FLAGS, stream=None):
    _check(lib().mhd_con2prim(h, slot_state, slot_prim, slot_flags, stream))


def mhd_prim2con(h, slot_state=SLOT_U, slot_prim=SLOT_P, stream=None):
    _check(lib().mhd_prim2con(h, slot_state, slot_prim, stream))


def mhd_rhs(h, slot_state, slot_prim, slot_rhs, stream=None):
    _check(lib().mhd_rhs(h, slot_state, slot_prim, slot_rhs, stream))


def mhd_les_flux(h, slot_state=SLOT_U, slot_prim=SLOT_P, stream=None):
    _check(lib().mhd_les_flux(h, slot_state, slot_prim, stream))


def mhd_rk_stage(h, tableau, stage, dt, stream=None):
    _check(lib().mhd_rk_stage(h, ctypes.byref(tableau), stage, dt, stream))


def mhd_advance(h, tableau, bc, dt, n_steps, stream=None):
    _check(lib().mhd_advance(h, ctypes.byref(tableau), _bc(bc), dt, n_steps, stream))


def mhd_advance_host(h, tableau, bc, dt, n_steps, host_U_ptr, host_flags_ptr=None, stream=None):
    _check(lib().mhd_advance_host(h, ctypes.byref(tableau), _bc(bc), dt, n_steps, host_U_ptr, host_flags_ptr, stream))


def mhd_m1_implicit(h, slot_V, slot_R, adt, stream=None):
    _check(lib().mhd_m1_implicit(h, slot_V, slot_R, adt, stream))


def mhd_m1_rhs(h, slot_V, slot_KV, stream=None):
    _check(lib().mhd_m1_rhs(h, slot_V, slot_KV, stream))


def mhd_m1_backreaction(h, slot_R, slot_K, stream=None):
    _check(lib().mhd_m1_backreaction(h, slot_R, slot_K, stream))


def mhd_m1_gravity(h, slot_V, slot_K, stream=None):
    _check(lib().mhd_m1_gravity(h, slot_V, slot_K, stream))


def mhd_advance_imex(h, tableau, bc, dt, n_steps, stream=None):
    _check(lib().mhd_advance_imex(h, ctypes.byref(tableau), _bc(bc), dt, n_steps, stream))


def _i3(v):
    return (_i * 3)(*[int(x) for x in v])


def mhd_patch_set_neighbor(h, slot, direction, peer_dev_ptr, peer_field_stride):
    _check(lib().mhd_patch_set_neighbor(h, slot, _i3(direction), peer_dev_ptr, peer_field_stride))


def mhd_patch_halo_words(h):
    return lib().mhd_patch_halo_words(h)


def mhd_patch_set_neighbor_word(h, direction, peer_halo_words):
    _check(lib().mhd_patch_set_neighbor_word(h, _i3(direction), peer_halo_words))


def mhd_ipc_export(dev_ptr):
    """(64-byte handle, offset) of a device pointer, to be sent to the process that owns the neighbouring GPU"""
    buf = ctypes.create_string_buffer(64)
    off = ctypes.c_size_t(0)
    _check(lib().mhd_ipc_export(dev_ptr, buf, ctypes.byref(off)))
    return buf.raw, int(off.value)


def mhd_ipc_import(handle, offset):
    out = _p()
    _check(lib().mhd_ipc_import(handle, offset, ctypes.byref(out)))
    return out.value


def mhd_ipc_close(dev_ptr, offset):
    _check(lib().mhd_ipc_close(dev_ptr, offset))


def mhd_prolong(h_coarse, slot_c, h_fine, slot_f, origin, lo, hi, stream=None):
    _check(lib().mhd_prolong(h_coarse, slot_c, h_fine, slot_f, _i3(origin), _i3(lo), _i3(hi), stream))


def mhd_restrict(h_fine, slot_f, h_coarse, slot_c, origin, stream=None):
    _check(lib().mhd_restrict(h_fine, slot_f, h_coarse, slot_c, _i3(origin), stream))


def mhd_dense_weights(scheme, theta, deriv=0):
    b = (_d * 4)()
    s = lib().mhd_dense_weights(scheme, theta, deriv, b)
    if s < 0:
        _check(s)
    return [b[j] for j in range(s)]


def mhd_dense_output(h, scheme, theta, dt, deriv, slot_out, stream=None):
    _check(lib().mhd_dense_output(h, scheme, theta, dt, deriv, slot_out, stream))


def mhd_advance_imex_host(h, tableau, bc, dt, n_steps, host_U_ptr, host_V_ptr, host_flags_ptr=None, stream=None):
    _check(lib().mhd_advance_imex_host(h, ctypes.byref(tableau), _bc(bc), dt, n_steps, host_U_ptr, host_V_ptr, host_flags_ptr, stream))


def mhd_patch_status(h, slot_flags=SLOT_FLAGS, stream=None):
    st = mhd_status()
    _check(lib().mhd_patch_status(h, slot_flags, ctypes.byref(st), stream))
    return {n: getattr(st, n) for n, _ in mhd_status._fields_}


def mhd_patch_profile(h, enable):
    _check(lib().mhd_patch_profile(h, int(enable)))


def mhd_patch_profile_read(h, stream=None):
    ms = (_d * NKERNELS)()
    n = (ctypes.c_ulonglong * NKERNELS)()
    _check(lib().mhd_patch_profile_read(h, ms, n, stream))
    return {k: (ms[i], int(n[i])) for i, k in enumerate(KERNEL_CLASSES)}


CENSUS_MAX_POINTS = 1 << 28


def mhd_flag_census_static(d_flags_ptr, n_points, d_counts_ptr, stream=None):
    """Allocation-free flag census (include/mhd.h): device pointers in, 9 device words out; see the header for the sharing rule."""
    _check(lib().mhd_flag_census_static(d_flags_ptr, n_points, d_counts_ptr, stream))


def mhd_probe_fp64_flops(stream=None):
    return lib().mhd_probe_fp64_flops(stream)


class Patch:
    """Owns the torch device tensors of one patch and binds them to the library's slots."""

    def __init__(self, params, n, ng, dx, stages=4, table=None, device="cuda:0", m1=False, fused=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libmhd_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        nx, ny, nz = n
        self.n, self.ng, self.dx = (nx, ny, nz), ng, dx
        self.shape = (nz + 2 * ng, ny + 2 * ng, nx + 2 * ng)
        self.npts = int(np.prod(self.shape))
        self.stages = stages
        self._table_t = None
        ptrs = None
        if table is not None:
            self._table_t = [torch.as_tensor(np.ascontiguousarray(table[k], dtype=np.float64), device=self.device)
                             for k in ("logp", "loge", "cs2")]
            ptrs = [t.data_ptr() for t in self._table_t]
        self.desc = make_desc(params, nx, ny, nz, ng, dx, table_ptrs=ptrs, table=table, n_species=3 if m1 else 0)
        self.h = mhd_patch_create(self.desc)
        z = lambda nf, dt=torch.float64: torch.zeros((nf,) + self.shape, dtype=dt, device=self.device)
        self.U, self.U0, self.P = z(NSTATE), z(NSTATE), z(NPRIM)
        self.flags = z(1, torch.uint8)
        self.K = [z(NSTATE) for _ in range(stages)]
        self.work = z(NWORK)
        for slot, t in [(SLOT_U, self.U), (SLOT_U0, self.U0), (SLOT_P, self.P), (SLOT_FLAGS, self.flags), (SLOT_WORK, self.work)] + \
                       [(SLOT_K1 + j, k) for j, k in enumerate(self.K)]:
            mhd_patch_bind(self.h, slot, t.data_ptr(), self.npts)
        self.leswork = None
        if any(float(params.get(c, 0.0)) != 0.0 for c in ("les_C_M", "les_C_N", "les_C_Y", "les_C_T")):             # LES sub-grid-scale term: scratch for the auxiliary fields of App. A
            self.leswork = z(NLESWORK)
            mhd_patch_bind(self.h, SLOT_LESWORK, self.leswork.data_ptr(), self.npts)
        self.U1 = None
        if fused and not m1:                                # third state buffer: mhd_advance then fuses the RK combine into the RHS kernels (measured slower on B200
                                                            # with the present latency-bound k_adv_ko / k_recon_march: 111.9 vs 107.5 ms per step at c4_256; off by default)
            self.U1 = z(NSTATE)
            mhd_patch_bind(self.h, SLOT_U1, self.U1.data_ptr(), self.npts)
        if m1:                                              # grey M1, 3 species: V, V^n, per-stage explicit parts and stiff sources
            self.V, self.V0, self.m1work = z(NM1), z(NM1), z(NM1WORK)
            self.KV = [z(NM1) for _ in range(stages)]
            self.R = [z(NM1) for _ in range(stages)]
            for slot, t in [(SLOT_V, self.V), (SLOT_V0, self.V0), (SLOT_M1WORK, self.m1work)] + \
                           [(SLOT_KV1 + j, k) for j, k in enumerate(self.KV)] + [(SLOT_R1 + j, k) for j, k in enumerate(self.R)]:
                mhd_patch_bind(self.h, slot, t.data_ptr(), self.npts)

    def m1_implicit(self, adt, j=1):
        """V* -> V^(i) in place; stiff source to R_j"""
        mhd_m1_implicit(self.h, SLOT_V, SLOT_R1 + j - 1, adt, self.stream())
        return self.R[j - 1]

    def m1_rhs(self, j=1):
        mhd_m1_rhs(self.h, SLOT_V, SLOT_KV1 + j - 1, self.stream())
        return self.KV[j - 1]

    def m1_backreaction(self, j=1):
        mhd_m1_backreaction(self.h, SLOT_R1 + j - 1, SLOT_K1 + j - 1, self.stream())

    def m1_gravity(self, j=1):
        """radiation terms of the CCZ4 matter sources added to K_j (after m1_rhs on the same V)"""
        mhd_m1_gravity(self.h, SLOT_V, SLOT_K1 + j - 1, self.stream())

    def advance_imex(self, tableau, bc, dt, n_steps):
        mhd_advance_imex(self.h, tableau, bc, dt, n_steps, self.stream())

    def close(self):
        if getattr(self, "h", None) is not None:
            mhd_patch_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def stream(self):
        return self.torch.cuda.current_stream(self.device).cuda_stream

    def upload(self, U=None, P=None):
        if U is not None:
            self.U.copy_(self.torch.as_tensor(U))
        if P is not None:
            self.P.copy_(self.torch.as_tensor(P))

    def fill_ghosts(self, bc, slot=SLOT_U):
        mhd_fill_ghosts(self.h, slot, bc, self.stream())

    def con2prim(self):
        mhd_con2prim(self.h, SLOT_U, SLOT_P, SLOT_FLAGS, self.stream())

    def prim2con(self):
        mhd_prim2con(self.h, SLOT_U, SLOT_P, self.stream())

    def rhs(self, j=1):
        """K_j <- F(U)"""
        mhd_rhs(self.h, SLOT_U, SLOT_P, SLOT_K1 + j - 1, self.stream())
        return self.K[j - 1]

    def rk_stage(self, tableau, stage, dt):
        mhd_rk_stage(self.h, tableau, stage, dt, self.stream())

    def advance(self, tableau, bc, dt, n_steps):
        mhd_advance(self.h, tableau, bc, dt, n_steps, self.stream())

    def advance_host(self, tableau, bc, dt, n_steps, host_U, host_flags=None):
        """host_U: pinned CPU float64 tensor (NSTATE, MZ, MY, MX), updated in place; host_flags: uint8 tensor or None."""
        mhd_advance_host(self.h, tableau, bc, dt, n_steps, host_U.data_ptr(),
                         None if host_flags is None else host_flags.data_ptr(), self.stream())

    def advance_imex_host(self, tableau, bc, dt, n_steps, host_U, host_V, host_flags=None):
        mhd_advance_imex_host(self.h, tableau, bc, dt, n_steps, host_U.data_ptr(), host_V.data_ptr(),
                              None if host_flags is None else host_flags.data_ptr(), self.stream())

    def profile(self, enable):
        mhd_patch_profile(self.h, enable)

    def profile_read(self):
        """{kernel class: (milliseconds, launches)} since the last read (CUDA events on the launching stream)"""
        return mhd_patch_profile_read(self.h, self.stream())

    def status(self):
        return mhd_patch_status(self.h, SLOT_FLAGS, self.stream())
