"""bloch_simulate is asynchronous on the caller's stream, never allocates and never synchronises, so a caller can
capture it into a CUDA graph and replay it (launch overhead of many-block sequences).
The replayed graph must give bitwise the signal of the direct call, on both execution paths (pytest -m gpu)."""
import numpy as np
import pytest

from paper_2301_02702_b200 import workloads as W
from test_gpu_parity import B  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,path,options", [("1", "per_block", None), ("2", "per_block", None), ("5", "per_block", None),
                                               ("5", "fused", None), ("4", "per_block", {"rf_const": 2})])
def test_simulate_is_graph_capturable_and_replays_bitwise(B, name, path, options):
    """(rf_const = 2: the excitation kernel whose step records are a 32 KB kernel parameter, captured by value)"""
    import torch
    w = W.small(name)
    plan = B.Plan(w.seq, path=path, phase_mode="fp32", options=options)
    dev = B.phantom_to_device(w.phantom)
    n = w.phantom.n
    sig = torch.zeros(plan.info["n_adc"], dtype=torch.complex64, device="cuda")
    Mxy = torch.zeros(n, 2, dtype=torch.float32, device="cuda")
    Mz = torch.zeros(n, dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):                       # warm-up outside capture: workspace, tables, attributes
        plan.simulate(*dev, Mxy=Mxy, Mz=Mz, signal=sig)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    direct = (sig.cpu().numpy().copy(), Mxy.cpu().numpy().copy(), Mz.cpu().numpy().copy())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        plan.simulate(*dev, Mxy=Mxy, Mz=Mz, signal=sig)
    for _ in range(3):
        sig.zero_(); Mxy.zero_(); Mz.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(sig.cpu().numpy().view(np.float32), direct[0].view(np.float32))
        assert np.array_equal(Mxy.cpu().numpy(), direct[1]) and np.array_equal(Mz.cpu().numpy(), direct[2])
    del g
    plan.close()
