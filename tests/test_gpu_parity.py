"""GPU parity tests proper: the CUDA library (through the C ABI / ctypes binding) against the oracle,
element by element on the same seeded inputs. Tolerances:
  RHS after one stage: per component  max|gpu - oracle| / max|oracle|  <= 1e-11   (north_star, reading R28)
  state after 10 RK steps: <= 1e-9;  flags: bit-exact;  ghost fill / copies: bit-exact.
"""
import numpy as np
import pytest

from paper_2510_13965_b200 import synth

pytestmark = pytest.mark.gpu
NG = 3


def _rel(a, b, interior=True):
    """per-field inf-norm relative difference (R28)"""
    s = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG)) if interior else (slice(None),) * 4
    a, b = a[s], b[s]
    num = np.abs(a - b).reshape(a.shape[0], -1).max(axis=1)
    den = np.abs(b).reshape(b.shape[0], -1).max(axis=1)
    return num / np.where(den > 0, den, 1.0), den


def _setup(oracle_mod, cfg):
    from paper_2510_13965_b200 import binding
    n = cfg["n"]
    o = oracle_mod.Oracle(cfg["params"], n[0], n[1], n[2], cfg["ng"], cfg["dx"], table=cfg.get("table"))
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    patch = binding.Patch(cfg["params"], n, cfg["ng"], cfg["dx"], stages=4, table=cfg.get("table"))
    return o, patch, U, P


def _one_stage(oracle_mod, cfg, rhs_tol=1e-11, prim_tol=1e-12):
    o, patch, U, P = _setup(oracle_mod, cfg)
    # oracle
    Uo = U.copy()
    o.fill_ghosts(Uo, cfg["bc"])
    Po, Fo = o.con2prim(Uo)
    Ko = o.rhs(Uo, Po)
    # gpu
    patch.upload(U=U)
    patch.fill_ghosts(cfg["bc"])
    assert np.array_equal(patch.U.cpu().numpy(), _filled(o, U, cfg["bc"]))        # ghost fill is bit-exact
    patch.con2prim()
    Pg, Fg, Ug = patch.P.cpu().numpy(), patch.flags.cpu().numpy()[0], patch.U.cpu().numpy()
    assert np.array_equal(Fg, Fo), "flag masks must agree bit for bit"
    rp, _ = _rel(Pg, Po, interior=False)
    assert np.all(rp < prim_tol), rp
    ru, _ = _rel(Ug, Uo, interior=False)
    assert np.all(ru < prim_tol), ru
    Kg = patch.rhs(1).cpu().numpy()
    rk, den = _rel(Kg, Ko)
    live = den > 0
    assert np.all(rk[live] < rhs_tol), (rk, den)
    assert np.all(np.abs(Kg[~live][:, NG:-NG, NG:-NG, NG:-NG]) == 0) if (~live).any() else True
    patch.close()
    return rk


def _filled(o, U, bc):
    V = U.copy()
    o.fill_ghosts(V, bc)
    return V


def test_config1_one_stage_parity(oracle_mod):
    """BASELINE.json configs[0]: coupled CCZ4+GRMHD RHS, one stage, 32^3 + 3 ghosts, periodic."""
    _one_stage(oracle_mod, synth.config1(n=32))


def test_config1_all_terms_exercised(oracle_mod):
    """Same with perturbed lapse, shift (both upwind branches), Theta, Z^i and phi, so every term is live."""
    _one_stage(oracle_mod, synth.config1(n=32, gauge_perturbation=True))


def test_ragged_sizes_and_outflow(oracle_mod):
    """Sizes that are not multiples of any tile (several tiles + ragged tail in x, y and z), outflow boundaries."""
    cfg = synth.config1(n=32, gauge_perturbation=True)
    nx, ny, nz = 61, 19, 13
    cfg["U"] = np.ascontiguousarray(np.tile(cfg["U"], (1, 1, 1, 2))[:, :nz + 6, :ny + 6, :nx + 6])
    cfg["P"] = np.ascontiguousarray(np.tile(cfg["P"], (1, 1, 1, 2))[:, :nz + 6, :ny + 6, :nx + 6])
    cfg["n"] = (nx, ny, nz)
    cfg["bc"] = [1, 1, 0, 1, 1, 0]
    _one_stage(oracle_mod, cfg, rhs_tol=1e-11)


def test_prim2con_parity(oracle_mod):
    cfg = synth.config1(n=16)
    o, patch, U, P = _setup(oracle_mod, cfg)
    patch.upload(U=cfg["U"], P=cfg["P"])
    patch.prim2con()
    ru, _ = _rel(patch.U.cpu().numpy(), U, interior=False)
    rp, _ = _rel(patch.P.cpu().numpy(), P, interior=False)
    assert np.all(ru < 1e-14) and np.all(rp < 1e-14), (ru, rp)
    patch.close()


def test_atmosphere_and_error_policy_flags(oracle_mod):
    """Cells below the density cut, with eps < 0, with Ye out of range: identical flags and identical resets."""
    cfg = synth.config1(n=16)
    cfg["params"].update(ye_min=0.27, ye_max=0.33, rho_low=1e-8)
    o, patch, U, P = _setup(oracle_mod, cfg)
    rng = np.random.default_rng(7)
    m = rng.random(U.shape[1:])
    U[22][m < 0.2] *= 1e-8                        # -> atmosphere
    U[24][(m > 0.2) & (m < 0.3)] *= -1.0          # tau < 0 -> eps floor
    U[22:28, m > 0.9] *= 1e-6                     # low density: Ye excursions are repaired, not fatal
    Uo = U.copy()
    Po, Fo = o.con2prim(Uo)
    patch.upload(U=U)
    patch.con2prim()
    Fg = patch.flags.cpu().numpy()[0]
    assert np.array_equal(Fg, Fo)
    assert set(np.unique(Fo)) >= {0, 1, 2}
    assert np.all(_rel(patch.P.cpu().numpy(), Po, interior=False)[0] < 1e-12)
    assert np.all(_rel(patch.U.cpu().numpy(), Uo, interior=False)[0] < 1e-12)
    st = patch.status()
    assert st["n_points"] == Fo.size and st["n_atmo"] == int((Fo & 1).sum()) and st["n_eps_lo"] == int(((Fo >> 1) & 1).sum())
    assert st["n_ye"] == int(((Fo >> 4) & 1).sum()) and st["n_fatal"] == int(((Fo >> 5) & 1).sum())
    patch.close()


def test_rk_stage_matches_oracle_combine(oracle_mod):
    from paper_2510_13965_b200 import binding
    cfg = synth.config1(n=16)
    o, patch, U, P = _setup(oracle_mod, cfg)
    rng = np.random.default_rng(11)
    a, w = synth.tableau("rk4")
    tab = binding.make_tableau(a, w)
    Ks = [rng.standard_normal(U.shape) for _ in range(4)]
    patch.upload(U=U)
    patch.rk_stage(tab, 0, 0.0)
    assert np.array_equal(patch.U0.cpu().numpy(), U)
    for j in range(4):
        patch.K[j].copy_(patch.torch.as_tensor(Ks[j]))
    dt = 0.013
    for stage in (1, 2, 3, 4):
        patch.rk_stage(tab, stage, dt)
        coef = a[stage, :stage] if stage < 4 else w
        ref = o.rk_combine(U, Ks[:len(coef)], coef, dt)
        got = patch.U.cpu().numpy()
        s = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
        assert np.abs(got[s] - ref[s]).max() < 1e-15 * (1 + np.abs(ref[s]).max() + dt * 4)
    patch.close()


def test_ten_rk_steps_parity(oracle_mod):
    """north_star: <= 1e-9 after 10 full RK4 steps (16^3 keeps the oracle to seconds; Courant 0.25)."""
    from paper_2510_13965_b200 import binding
    cfg = synth.config1(n=16, gauge_perturbation=True)
    o, patch, U, P = _setup(oracle_mod, cfg)
    a, w = synth.tableau("rk4")
    dt = 0.25 * cfg["dx"]
    Uo = U.copy()
    Po, Fo = o.evolve(Uo, cfg["bc"], a, w, dt, 10)
    patch.upload(U=U)
    patch.advance(binding.make_tableau(a, w), cfg["bc"], dt, 10)
    Ug, Pg, Fg = patch.U.cpu().numpy(), patch.P.cpu().numpy(), patch.flags.cpu().numpy()[0]
    assert np.array_equal(Fg, Fo)
    ru, _ = _rel(Ug, Uo, interior=False)
    rp, _ = _rel(Pg, Po, interior=False)
    assert np.all(ru < 1e-9) and np.all(rp < 1e-9), (ru, rp)
    # and the end-to-end host-buffer entry point gives the same state
    import torch
    hostU = torch.as_tensor(U).clone().pin_memory()
    hostF = torch.zeros(Fo.shape, dtype=torch.uint8).pin_memory()
    patch.advance_host(binding.make_tableau(a, w), cfg["bc"], dt, 10, hostU, hostF)
    assert np.array_equal(hostU.numpy(), Ug) and np.array_equal(hostF.numpy(), Fg)
    patch.close()
