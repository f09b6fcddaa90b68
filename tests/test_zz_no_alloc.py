"""mhd_flag_census_static (include/mhd.h): the flag census with its scratch in a file-scope device array, no allocation, no mhd_patch.
Against the existing path (the census inside mhd_patch_status), bit for bit (integer work), on two calls in a row with different flag
contents (the second call finds the first call's partial counts in the shared array and must not be affected by them), on a size that ends
inside a chunk and on one that spans several; sizes beyond the fixed capacity are refused. Collected last on purpose (the suite runs with
pytest -x); passes alone in a fresh process as well as after the other tests."""
import numpy as np
import pytest

from paper_2510_13965_b200 import synth

pytestmark = pytest.mark.gpu
ORDER = ["n_points", "n_atmo", "n_eps_lo", "n_eps_hi", "n_vmax", "n_ye", "n_fatal", "n_noconv", "n_m1fix"]


def _census(binding, torch, flags, out):
    binding.mhd_flag_census_static(flags.data_ptr(), flags.numel(), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return [int(v) for v in out.cpu().numpy().astype(np.uint64)]


def test_static_census_matches_patch_status_twice():
    from paper_2510_13965_b200 import binding
    import torch
    # a real flag field: the TOV star of config 3 after con2prim (atmosphere cells outside the star), 46^3 points: ends inside the second chunk
    cfg = synth.config3(n=40)
    patch = binding.Patch(cfg["params"], cfg["n"], 3, cfg["dx"], stages=1)
    patch.upload(U=cfg["U"], P=cfg["P"])
    patch.prim2con()
    patch.fill_ghosts(cfg["bc"])
    patch.con2prim()
    out = torch.full((9,), -1, dtype=torch.int64, device="cuda")          # caller-owned output, allocated before the calls under test
    rng = np.random.default_rng(11)
    for call in range(2):
        if call == 1:                                                      # second call in a row: every bit pattern, so all eight counters differ from call one
            patch.flags.copy_(torch.as_tensor(rng.integers(0, 256, size=tuple(patch.flags.shape), dtype=np.uint8)))
        want = patch.status()
        mem0 = torch.cuda.memory_allocated()
        got = _census(binding, torch, patch.flags, out)
        assert torch.cuda.memory_allocated() == mem0
        assert got == [want[k] for k in ORDER], (call, got, want)
        host = patch.flags.cpu().numpy().ravel()                           # and against a plain count on the host
        assert got == [host.size] + [int(((host >> b) & 1).sum()) for b in range(8)]
    assert want["n_fatal"] > 0 and want["n_m1fix"] > 0
    patch.close()
    # several chunks and a ragged tail, then a shorter array right after it (stale partial counts of the longer call stay in the array)
    for n in (5 * 65536 + 12345, 70000, 1):
        f = torch.as_tensor(rng.integers(0, 256, size=n, dtype=np.uint8)).cuda()
        got = _census(binding, torch, f, out)
        h = f.cpu().numpy()
        assert got == [n] + [int(((h >> b) & 1).sum()) for b in range(8)], n


def test_static_census_refuses_what_it_cannot_hold():
    from paper_2510_13965_b200 import binding
    import torch
    f = torch.zeros(16, dtype=torch.uint8, device="cuda")
    out = torch.zeros(9, dtype=torch.int64, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    with pytest.raises(binding.MhdError, match="capacity"):
        binding.mhd_flag_census_static(f.data_ptr(), binding.CENSUS_MAX_POINTS + 1, out.data_ptr(), s)    # refused before anything is launched or read
    for args in ((None, 16, out.data_ptr()), (f.data_ptr(), 16, None), (f.data_ptr(), 0, out.data_ptr())):
        with pytest.raises(binding.MhdError, match="invalid argument"):
            binding.mhd_flag_census_static(args[0], args[1], args[2], s)
    torch.cuda.synchronize()
    assert int(out.abs().sum()) == 0
