"""GPU parity of the AMR transfer operators against the oracle, through the C ABI: mhd_prolong (Eq. 80),
mhd_restrict (copy), mhd_dense_output (Eqs. 56-59). Tolerances: copies bit-exact; Eq. (80) sums 6^3 terms in a different order on the
two sides -> 1e-14 of the field's magnitude; dense output 1e-14."""
import numpy as np
import pytest

from paper_2510_13965_b200 import synth

pytestmark = pytest.mark.gpu
NG = 3


def _pair(nc, nf, seed=1):
    from paper_2510_13965_b200 import binding
    par = synth.default_params()
    pc = binding.Patch(par, (nc,) * 3 if isinstance(nc, int) else nc, NG, 0.2, stages=4)
    pf = binding.Patch(par, (nf,) * 3 if isinstance(nf, int) else nf, NG, 0.1, stages=4)
    rng = np.random.default_rng(seed)
    Uc = rng.standard_normal(tuple(pc.U.shape))
    Uf = rng.standard_normal(tuple(pf.U.shape))
    pc.upload(U=Uc)
    pf.upload(U=Uf)
    return binding, pc, pf, Uc, Uf


def test_prolong_whole_patch_and_ghost_faces(oracle_mod):
    binding, pc, pf, Uc, Uf = _pair(16, (13, 10, 9))
    org = (4, 5, 6)
    M = pf.U.shape[1:][::-1]                                   # (MX, MY, MZ)
    binding.mhd_prolong(pc.h, binding.SLOT_U, pf.h, binding.SLOT_U, org, (0, 0, 0), M, pf.stream())
    want = oracle_mod.prolong(Uc, NG, Uf.copy(), NG, org, (0, 0, 0), M)
    got = pf.U.cpu().numpy()
    assert np.abs(got - want).max() <= 1e-14 * np.abs(want).max()
    ev = (slice(None), slice(1, None, 2), slice(1, None, 2), slice(1, None, 2))     # ng odd: odd array index = even interior index
    assert np.array_equal(got[ev], want[ev])                   # coincident points are copies
    # ghost faces only, one box per face; the interior keeps its content
    pf.upload(U=Uf)
    want = Uf.copy()
    nx, ny, nz = pf.n
    boxes = [((0, 0, 0), (NG, M[1], M[2])), ((nx + NG, 0, 0), M), ((NG, 0, 0), (nx + NG, NG, M[2])), ((NG, ny + NG, 0), (nx + NG, M[1], M[2])),
             ((NG, NG, 0), (nx + NG, ny + NG, NG)), ((NG, NG, nz + NG), (nx + NG, ny + NG, M[2]))]
    for lo, hi in boxes:
        binding.mhd_prolong(pc.h, binding.SLOT_U, pf.h, binding.SLOT_U, org, lo, hi, pf.stream())
        oracle_mod.prolong(Uc, NG, want, NG, org, lo, hi)
    got = pf.U.cpu().numpy()
    assert np.abs(got - want).max() <= 1e-14 * np.abs(want).max()
    inner = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
    assert np.array_equal(got[inner], Uf[inner])
    # other slots with matching field counts (primitives), and a stencil that leaves the coarse array is refused
    pc.P.copy_(pc.torch.as_tensor(Uc[:10]))
    binding.mhd_prolong(pc.h, binding.SLOT_P, pf.h, binding.SLOT_P, org, (0, 0, 0), M, pf.stream())
    wantP = oracle_mod.prolong(np.ascontiguousarray(Uc[:10]), NG, np.zeros((10,) + Uf.shape[1:]), NG, org, (0, 0, 0), M)
    assert np.abs(pf.P.cpu().numpy() - wantP).max() <= 1e-14 * np.abs(wantP).max()
    with pytest.raises(binding.MhdError):
        binding.mhd_prolong(pc.h, binding.SLOT_U, pf.h, binding.SLOT_U, (12, 5, 6), (0, 0, 0), M, pf.stream())
    with pytest.raises(binding.MhdError):
        binding.mhd_prolong(pc.h, binding.SLOT_U, pf.h, binding.SLOT_P, org, (0, 0, 0), M, pf.stream())
    pc.close(); pf.close()


def test_restrict_is_bit_exact(oracle_mod):
    binding, pc, pf, Uc, Uf = _pair(16, (13, 10, 9), seed=2)
    org = (3, 2, 7)
    binding.mhd_restrict(pf.h, binding.SLOT_U, pc.h, binding.SLOT_U, org, pf.stream())
    want = oracle_mod.restrict(Uf, NG, Uc.copy(), NG, org)
    assert np.array_equal(pc.U.cpu().numpy(), want)
    with pytest.raises(binding.MhdError):
        binding.mhd_restrict(pf.h, binding.SLOT_U, pc.h, binding.SLOT_U, (3, 2, 15), pf.stream())
    pc.close(); pf.close()


def test_prolong_full_size_polynomial(oracle_mod):
    """256^3 fine patch (the bench launch configuration of the state slot) from a 140^3 coarse patch: exact for a polynomial of degree
    5 in each variable at every fine point (a property that holds at any size), sampled boxes against the oracle."""
    from paper_2510_13965_b200 import binding
    import torch
    par = synth.default_params()
    nc, nf, org = 140, 256, (6, 5, 4)
    pc = binding.Patch(par, (nc,) * 3, NG, 2.0 / nc, stages=1)
    pf = binding.Patch(par, (nf,) * 3, NG, 1.0 / nc, stages=1)
    xc = (torch.arange(nc + 2 * NG, dtype=torch.float64, device="cuda") - NG) / nc
    fx = 1 + xc - 0.5 * xc ** 5
    fy = 2 - xc ** 2 + 0.25 * xc ** 5
    fz = 1 + 0.3 * xc ** 3 + xc ** 4
    pc.U[0] = fz[:, None, None] * fy[None, :, None] * fx[None, None, :]
    pc.U[1:] = 0.0
    M = (nf + 2 * NG,) * 3
    binding.mhd_prolong(pc.h, binding.SLOT_U, pf.h, binding.SLOT_U, org, (0, 0, 0), M, pf.stream())
    xf = [org[d] / nc + (torch.arange(nf + 2 * NG, dtype=torch.float64, device="cuda") - NG) / (2 * nc) for d in range(3)]
    gx = 1 + xf[0] - 0.5 * xf[0] ** 5
    gy = 2 - xf[1] ** 2 + 0.25 * xf[1] ** 5
    gz = 1 + 0.3 * xf[2] ** 3 + xf[2] ** 4
    exact = gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    err = (pf.U[0] - exact).abs().max().item()
    assert err < 1e-12 * exact.abs().max().item(), err
    assert pf.U[1:].abs().max().item() == 0.0
    Uc = pc.U[:1].cpu().numpy()
    got = pf.U[:1].cpu().numpy()
    for lo in ((0, 0, 0), (250, 120, 7), (131, 255, 250)):
        hi = tuple(l + 12 for l in lo)
        want = oracle_mod.prolong(Uc, NG, np.zeros_like(got), NG, org, lo, hi)
        sl = (slice(None), slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
        assert np.abs(got[sl] - want[sl]).max() <= 1e-14 * np.abs(want[sl]).max()
    pc.close(); pf.close()


@pytest.mark.parametrize("scheme,name", [(0, "rk4"), (1, "ssprk3")])
def test_dense_output_parity(oracle_mod, scheme, name):
    """One RK step of config 1 driven stage by stage (U0 and K_j stay in their slots), then the interpolant at several theta and its
    time derivatives, against the oracle's dense_output applied to the GPU's own U0 and K_j; theta = 1 reproduces the step."""
    from paper_2510_13965_b200 import binding
    cfg = synth.config1(n=12, gauge_perturbation=True)
    n = cfg["n"]
    o = oracle_mod.Oracle(cfg["params"], n[0], n[1], n[2], NG, cfg["dx"])
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    a, w = synth.tableau(name)
    s = len(w)
    tab = binding.make_tableau(a, w)
    patch = binding.Patch(cfg["params"], n, NG, cfg["dx"], stages=s, fused=True)     # fused=True only to own a third state buffer (U1)
    patch.upload(U=U)
    dt = 0.25 * cfg["dx"]
    patch.fill_ghosts(cfg["bc"])
    patch.con2prim()
    patch.rk_stage(tab, 0, dt)
    for st in range(1, s + 1):
        patch.rhs(st)
        patch.rk_stage(tab, st, dt)
        patch.fill_ghosts(cfg["bc"])
        patch.con2prim()
    U0 = patch.U0.cpu().numpy()
    Ks = [k.cpu().numpy() for k in patch.K]
    for theta, deriv in ((0.0, 0), (0.3, 0), (0.5, 0), (1.0, 0), (0.5, 1), (0.25, 2), (0.7, 3)):
        if scheme == 1 and deriv == 3:
            continue
        patch.U1.zero_()
        binding.mhd_dense_output(patch.h, scheme, theta, dt, deriv, binding.SLOT_U1, patch.stream())
        want = o.dense_output(U0, Ks, scheme, theta, dt, deriv)
        got = patch.U1.cpu().numpy()
        inner = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
        num = np.abs(got[inner] - want[inner]).reshape(32, -1).max(axis=1)
        den = np.abs(want[inner]).reshape(32, -1).max(axis=1)
        assert np.all(num <= 1e-13 * np.where(den > 0, den, 1.0)), (theta, deriv, num / np.where(den > 0, den, 1.0))
        if theta == 1.0 and deriv == 0:                        # the interpolant ends on the step's result
            Un = patch.U.cpu().numpy()
            num = np.abs(got[inner] - Un[inner]).reshape(32, -1).max(axis=1)
            dn = np.abs(Un[inner]).reshape(32, -1).max(axis=1)
            assert np.all(num <= 1e-13 * np.where(dn > 0, dn, 1.0))
    assert np.allclose(binding.mhd_dense_weights(scheme, 0.4), oracle_mod.dense_weights(scheme, 0.4), atol=1e-16)
    with pytest.raises(binding.MhdError):
        binding.mhd_dense_output(patch.h, 2, 0.5, dt, 0, binding.SLOT_U1, patch.stream())
    with pytest.raises(binding.MhdError):
        binding.mhd_dense_output(patch.h, scheme, 0.5, dt, 0, binding.SLOT_U0, patch.stream())
    patch.close()


def test_prolong_tiled_path_ragged_boxes(oracle_mod):
    """Boxes of at least 32 x 8 x 8 fine points take the separable shared-memory kernel: whole array and boxes that start on odd indices and end
    inside a block, against the oracle; points outside the box keep their content."""
    binding, pc, pf, Uc, Uf = _pair(30, (40, 12, 10), seed=5)
    org = (5, 9, 10)
    M = pf.U.shape[1:][::-1]
    for lo, hi in (((0, 0, 0), M), ((1, 3, 2), (45, 17, 15)), ((7, 0, 5), (40, 9, 14))):
        pf.upload(U=Uf)
        binding.mhd_prolong(pc.h, binding.SLOT_U, pf.h, binding.SLOT_U, org, lo, hi, pf.stream())
        want = oracle_mod.prolong(Uc, NG, Uf.copy(), NG, org, lo, hi)
        got = pf.U.cpu().numpy()
        assert np.abs(got - want).max() <= 1e-14 * np.abs(want).max(), (lo, hi)
        mask = np.ones(got.shape[1:], bool)
        mask[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] = False
        assert np.array_equal(got[:, mask], Uf[:, mask])
    pc.close(); pf.close()
