"""mhd_advance launches kernels on the caller's stream and nothing else (no synchronisation, no allocation, no host read after the first call on a
device), so a caller can capture it into a CUDA graph and replay it: small patches are launch-bound (about 50 launches per RK4 step). The replay
must reproduce the direct call bit for bit."""
import pytest
import torch

from paper_2510_13965_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [16, 24])
def test_advance_replays_from_a_cuda_graph(n):
    from paper_2510_13965_b200 import binding
    cfg = synth.config1(n=n, gauge_perturbation=True)
    a, w = synth.tableau("rk4")
    tab = binding.make_tableau(a, w)
    dt = 0.25 * cfg["dx"]
    patch = binding.Patch(cfg["params"], cfg["n"], 3, cfg["dx"], stages=4)
    patch.upload(U=cfg["U"], P=cfg["P"])
    patch.prim2con()
    U0, P0 = patch.U.clone(), patch.P.clone()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        patch.advance(tab, cfg["bc"], dt, 2)                   # first call on this device: opt-ins to large shared memory, lazy module load
        s.synchronize()
        ref = patch.U.clone()
        patch.U.copy_(U0); patch.P.copy_(P0)                   # P is the warm start of con2prim: same input, same iteration
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            patch.advance(tab, cfg["bc"], dt, 2)
        for _ in range(2):
            patch.U.copy_(U0); patch.P.copy_(P0)
            g.replay()
            s.synchronize()
            assert torch.equal(patch.U, ref)
        st = patch.status()
    assert st["n_fatal"] == 0 and st["n_noconv"] == 0
    patch.close()
