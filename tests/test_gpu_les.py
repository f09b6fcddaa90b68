"""GPU parity of the LES sub-grid-scale term of the induction equation (App. A, C_M = 8) against the oracle, through
the C ABI. Ghost width 5 (the gradients of the auxiliary fields are needed at every node the reconstruction reads).
Tolerances: auxiliary fields 1e-13, the SGS flux 1e-11 of its own magnitude, RHS 1e-11 per component (north_star), 10 steps 1e-9."""
import numpy as np
import pytest

from paper_2510_13965_b200 import synth

pytestmark = pytest.mark.gpu
NG = 5


def _boost_B(cfg, factor=30.0):
    """config 1 has B^2/rho ~ 1e-3: scale the magnetic field up so that the SGS tensor is not negligible beside the resolved flux"""
    cfg["U"][28:31] *= factor
    return cfg


def _setup(oracle_mod, cfg):
    from paper_2510_13965_b200 import binding
    n = cfg["n"]
    o = oracle_mod.Oracle(cfg["params"], n[0], n[1], n[2], NG, cfg["dx"])
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    patch = binding.Patch(cfg["params"], n, NG, cfg["dx"], stages=4)
    return binding, o, patch, U, P


def _rel(a, b):
    s = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
    num = np.abs(a[s] - b[s]).reshape(a.shape[0], -1).max(axis=1)
    den = np.abs(b[s]).reshape(b.shape[0], -1).max(axis=1)
    return num / np.where(den > 0, den, 1.0), den


@pytest.mark.parametrize("kind", [0, 1])
def test_les_flux_and_one_stage_parity(oracle_mod, kind):
    cfg = _boost_B(synth.config1(n=20, gauge_perturbation=True, ng=NG))
    cfg["params"].update(les_C_M=8.0)
    if kind == 1:
        cfg["params"].update(eos_kind=1, eos_gamma_th=1.8, n_pieces=3, pp_K=[30.0, 0.0, 0.0], pp_Gamma=[1.9, 2.4, 2.9], pp_rho=[1.0e-3, 5.0e-3, 1e300])
        cfg["P"][synth.EPS] = 0.25
    binding, o, patch, U, P = _setup(oracle_mod, cfg)
    Uo = U.copy()
    o.fill_ghosts(Uo, cfg["bc"])
    Po, Fo = o.con2prim(Uo)
    Lo, Ao = o.les_flux(Uo, Po)
    Ko = o.rhs(Uo, Po)
    K0 = oracle_mod.Oracle(dict(cfg["params"], les_C_M=0.0), *cfg["n"], NG, cfg["dx"]).rhs(Uo, Po)
    patch.upload(U=U)
    patch.fill_ghosts(cfg["bc"])
    patch.con2prim()
    assert np.array_equal(patch.flags.cpu().numpy()[0], Fo)
    patch.work.zero_()
    binding.mhd_les_flux(patch.h, binding.SLOT_U, binding.SLOT_P, patch.stream())
    Ag, Wg = patch.leswork.cpu().numpy(), patch.work.cpu().numpy()
    Ag, Ao = Ag[:26], Ao[:26]                                  # Ye, dp/dYe, D are staged only for the tabulated EoS, calE and D Ye only with C_N / C_Y / C_T
    den = np.abs(Ao).reshape(Ao.shape[0], -1).max(axis=1)
    ra = np.abs(Ag - Ao).reshape(Ao.shape[0], -1).max(axis=1) / np.where(den > 0, den, 1.0)
    assert np.all(ra < 1e-13), ra
    scale = np.abs(Lo).max()
    assert scale > 0
    for k in range(3):
        for i in range(3):
            assert np.abs(Wg[11 * k + 6 + i] - Lo[3 * k + i]).max() <= 1e-11 * scale, (k, i)
    used = {11 * k + 6 + i for k in range(3) for i in range(3) if i != k}
    assert all(np.all(Wg[f] == 0) for f in range(33) if f not in used)              # nothing else is touched
    Kg = patch.rhs(1).cpu().numpy()
    rk, den = _rel(Kg, Ko)
    assert np.all(rk[den > 0] < 1e-11), rk
    # the term is live: it changes the induction equation by more than the parity tolerance
    d, _ = _rel(Ko[28:31], K0[28:31])
    assert np.all(d > 1e-6), d
    patch.close()


def test_les_ten_steps(oracle_mod):
    cfg = _boost_B(synth.config1(n=12, gauge_perturbation=True, ng=NG))
    cfg["params"].update(les_C_M=8.0)
    binding, o, patch, U, P = _setup(oracle_mod, cfg)
    a, w = synth.tableau("rk4")
    dt = 0.25 * cfg["dx"]
    patch.upload(U=U)
    patch.advance(binding.make_tableau(a, w), cfg["bc"], dt, 10)
    Uo = U.copy()
    _, Fo = o.evolve(Uo, cfg["bc"], a, w, dt, 10)
    Ug = patch.U.cpu().numpy()
    num = np.abs(Ug - Uo).reshape(32, -1).max(axis=1)
    den = np.abs(Uo).reshape(32, -1).max(axis=1)
    assert np.all(num <= 1e-9 * np.where(den > 0, den, 1.0)), num / np.where(den > 0, den, 1.0)
    assert np.array_equal(patch.flags.cpu().numpy()[0], Fo)
    patch.close()


def test_les_ragged_outflow_and_refusals(oracle_mod):
    from paper_2510_13965_b200 import binding
    cfg = _boost_B(synth.config1(n=20, gauge_perturbation=True, ng=NG))
    cfg["params"].update(les_C_M=8.0)
    nx, ny, nz = 23, 13, 9
    cfg["U"] = np.ascontiguousarray(np.tile(cfg["U"], (1, 1, 1, 2))[:, :nz + 2 * NG, :ny + 2 * NG, :nx + 2 * NG])
    cfg["P"] = np.ascontiguousarray(np.tile(cfg["P"], (1, 1, 1, 2))[:, :nz + 2 * NG, :ny + 2 * NG, :nx + 2 * NG])
    cfg["n"] = (nx, ny, nz)
    cfg["bc"] = [1, 1, 0, 1, 1, 0]
    binding, o, patch, U, P = _setup(oracle_mod, cfg)
    Uo = U.copy()
    o.fill_ghosts(Uo, cfg["bc"])
    Po, Fo = o.con2prim(Uo)
    Ko = o.rhs(Uo, Po)
    patch.upload(U=U)
    patch.fill_ghosts(cfg["bc"])
    patch.con2prim()
    Kg = patch.rhs(1).cpu().numpy()
    rk, den = _rel(Kg, Ko)
    assert np.all(rk[den > 0] < 1e-11), rk
    patch.close()
    # ghost width 3, and the tabulated EoS, are refused at create time
    with pytest.raises(binding.MhdError):
        binding.mhd_patch_create(binding.make_desc(synth.default_params(les_C_M=8.0), 8, 8, 8, 3, 0.1))


def test_les_with_the_tabulated_eos(oracle_mod):
    """config 4 (hot star, table EoS) with C_M = 8: the EoS derivatives are those of the interpolant inside the table cell (R42) and the
    Y_e terms of (A12) are live (auxiliary fields Ye, dp/dYe, D). Auxiliary fields, SGS flux and one-stage RHS against the oracle."""
    cfg = synth.config4(n=24, ng=NG)
    cfg["params"].update(les_C_M=8.0)
    cfg["U"][28:31] *= 300.0                                   # B^2 / p ~ 1e-3 in the core: the SGS tensor is not negligible
    from paper_2510_13965_b200 import binding
    n = cfg["n"]
    o = oracle_mod.Oracle(cfg["params"], n[0], n[1], n[2], NG, cfg["dx"], table=cfg["table"])
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    patch = binding.Patch(cfg["params"], n, NG, cfg["dx"], stages=4, table=cfg["table"])
    Uo = U.copy()
    o.fill_ghosts(Uo, cfg["bc"])
    Po, Fo = o.con2prim(Uo)
    Lo, Ao = o.les_flux(Uo, Po)
    Ko = o.rhs(Uo, Po)
    patch.upload(U=U)
    patch.fill_ghosts(cfg["bc"])
    patch.con2prim()
    assert np.array_equal(patch.flags.cpu().numpy()[0], Fo)
    patch.work.zero_()
    binding.mhd_les_flux(patch.h, binding.SLOT_U, binding.SLOT_P, patch.stream())
    Ag, Wg = patch.leswork.cpu().numpy(), patch.work.cpu().numpy()
    Ag, Ao = Ag[:29], Ao[:29]                                  # calE and D Ye are staged only with C_N / C_Y / C_T
    den = np.abs(Ao).reshape(Ao.shape[0], -1).max(axis=1)
    for g0 in range(0, 18, 3):                                 # components of a vector share the vector's norm (v^z = 0 for rotation about z)
        den[g0:g0 + 3] = den[g0:g0 + 3].max()
    den[18] = den[3] * den[9]                                  # v.B vanishes analytically (azimuthal v, poloidal B): its scale is |v| |B|
    ra = np.abs(Ag - Ao).reshape(Ao.shape[0], -1).max(axis=1) / np.where(den > 0, den, 1.0)
    assert np.all(ra < 1e-11), [(int(f), float(ra[f])) for f in np.nonzero(ra >= 1e-11)[0]]     # primitives through the table's T inversion: 1e-11 (N3)
    assert den[26] > 0 and den[27] > 0 and den[28] > 0         # Ye, dp/dYe, D are live
    scale = np.abs(Lo).max()
    for k in range(3):
        for i in range(3):
            assert np.abs(Wg[11 * k + 6 + i] - Lo[3 * k + i]).max() <= 1e-9 * scale, (k, i, np.abs(Wg[11 * k + 6 + i] - Lo[3 * k + i]).max() / scale)
    Kg = patch.rhs(1).cpu().numpy()
    rk, dn = _rel(Kg, Ko)
    assert np.all(rk[dn > 0] < 1e-11), rk
    patch.close()


FULL = dict(les_C_M=8.0, les_C_N=2.0, les_C_Y=1.5, les_C_T=0.75)


def _check_all_fluxes(Wg, Lo, tol):
    """work slot (field 11 k + f of direction k: 0 Dbar, 1 DYebar, 3 + i Sbar_i, 6 + i Bbar^i) against the oracle's 24 SGS flux fields, each tensor on
    its own scale"""
    for k in range(3):
        for name, wf, lf in (("N", [0], [9 + k]), ("NY", [1], [12 + k]), ("T", [3, 4, 5], [15 + 3 * k + i for i in range(3)]),
                             ("M", [6, 7, 8], [3 * k + i for i in range(3)])):
            scale = {"N": np.abs(Lo[9:12]).max(), "NY": np.abs(Lo[12:15]).max(), "T": np.abs(Lo[15:24]).max(), "M": np.abs(Lo[0:9]).max()}[name]
            assert scale > 0, name
            for a, b in zip(wf, lf):
                err = np.abs(Wg[11 * k + a] - Lo[b]).max()
                assert err <= tol * scale, (name, k, a, err / scale)
        assert np.all(Wg[11 * k + 2] == 0) and np.all(Wg[11 * k + 9] == 0) and np.all(Wg[11 * k + 10] == 0)    # taubar (R47), phibar, speed: untouched


@pytest.mark.parametrize("kind", [0, 1])
def test_les_all_four_tensors(oracle_mod, kind):
    """C_M, C_N, C_Y, C_T all set ((A15)-(A17) beside (A16)): SGS fluxes of Dbar, DYebar, Sbar_i, Bbar^i and the one-stage RHS against the oracle;
    once on a block-aligned patch (TMA kernel) and once on a ragged one with an odd row length (no tensor map: the L1 kernel)."""
    for shape in (None, (23, 13, 9)):
        cfg = _boost_B(synth.config1(n=20, gauge_perturbation=True, ng=NG))
        cfg["params"].update(FULL)
        if kind == 1:
            cfg["params"].update(eos_kind=1, eos_gamma_th=1.8, n_pieces=3, pp_K=[30.0, 0.0, 0.0], pp_Gamma=[1.9, 2.4, 2.9], pp_rho=[1.0e-3, 5.0e-3, 1e300])
            cfg["P"][synth.EPS] = 0.25
        if shape is not None:
            nx, ny, nz = shape
            cfg["U"] = np.ascontiguousarray(np.tile(cfg["U"], (1, 1, 1, 2))[:, :nz + 2 * NG, :ny + 2 * NG, :nx + 2 * NG])
            cfg["P"] = np.ascontiguousarray(np.tile(cfg["P"], (1, 1, 1, 2))[:, :nz + 2 * NG, :ny + 2 * NG, :nx + 2 * NG])
            cfg["n"] = shape
            cfg["bc"] = [1, 1, 0, 1, 1, 0]
        binding, o, patch, U, P = _setup(oracle_mod, cfg)
        Uo = U.copy()
        o.fill_ghosts(Uo, cfg["bc"])
        Po, Fo = o.con2prim(Uo)
        Lo, Ao = o.les_flux(Uo, Po)
        Ko = o.rhs(Uo, Po)
        K0 = oracle_mod.Oracle(dict(cfg["params"], les_C_N=0.0, les_C_Y=0.0, les_C_T=0.0), *cfg["n"], NG, cfg["dx"]).rhs(Uo, Po)
        patch.upload(U=U)
        patch.fill_ghosts(cfg["bc"])
        patch.con2prim()
        assert np.array_equal(patch.flags.cpu().numpy()[0], Fo)
        patch.work.zero_()
        binding.mhd_les_flux(patch.h, binding.SLOT_U, binding.SLOT_P, patch.stream())
        Ag, Wg = patch.leswork.cpu().numpy(), patch.work.cpu().numpy()
        for f in (28, 29, 30):                                 # D, calE, D Ye are staged now
            assert np.abs(Ag[f] - Ao[f]).max() <= 1e-13 * np.abs(Ao[f]).max(), f
        _check_all_fluxes(Wg, Lo, 1e-11)
        Kg = patch.rhs(1).cpu().numpy()
        rk, den = _rel(Kg, Ko)
        assert np.all(rk[den > 0] < 1e-11), (shape, rk)
        d, _ = _rel(Ko[22:28], K0[22:28])                      # the three new tensors are live in Dbar, DYebar, Sbar_i (taubar has none)
        assert np.all(d[[0, 1, 3, 4, 5]] > 1e-6) and d[2] == 0, d
        patch.close()


def test_les_all_four_tensors_tabulated_eos(oracle_mod):
    cfg = synth.config4(n=24, ng=NG)
    cfg["params"].update(FULL)
    cfg["U"][28:31] *= 300.0
    from paper_2510_13965_b200 import binding
    n = cfg["n"]
    o = oracle_mod.Oracle(cfg["params"], n[0], n[1], n[2], NG, cfg["dx"], table=cfg["table"])
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    patch = binding.Patch(cfg["params"], n, NG, cfg["dx"], stages=4, table=cfg["table"])
    Uo = U.copy()
    o.fill_ghosts(Uo, cfg["bc"])
    Po, Fo = o.con2prim(Uo)
    Lo, Ao = o.les_flux(Uo, Po)
    Ko = o.rhs(Uo, Po)
    patch.upload(U=U)
    patch.fill_ghosts(cfg["bc"])
    patch.con2prim()
    assert np.array_equal(patch.flags.cpu().numpy()[0], Fo)
    patch.work.zero_()
    binding.mhd_les_flux(patch.h, binding.SLOT_U, binding.SLOT_P, patch.stream())
    Wg = patch.work.cpu().numpy()
    _check_all_fluxes(Wg, Lo, 1e-9)                            # EoS derivatives through the table's T inversion (N3), as in the C_M-only test
    Kg = patch.rhs(1).cpu().numpy()
    rk, dn = _rel(Kg, Ko)
    assert np.all(rk[dn > 0] < 1e-11), rk
    patch.close()
