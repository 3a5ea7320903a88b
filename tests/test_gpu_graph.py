"""a time-stepping caller (1e4 steps) can capture sg_set_density + sg_force in a
CUDA graph: after one warm-up call the library enqueues only kernel launches on the caller's stream (no
allocation, no synchronisation), so the pair is capturable and replays with new sigma contents."""
import numpy as np
import pytest

from workloads import make_config, nested_layout, kuzmin_sigma
from workloads.configs import cell_centres

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("mode", ["direct", "lattice"])
def test_step_is_cuda_graph_capturable(mode):
    """direct: cfg 2.  lattice: a four-level P = 16 nest, where sg_force forks its pair-class kernels onto side
    streams of the context and joins them back into the caller's stream (all of it inside the capture)."""
    import torch
    from paper_2001_02765_b200 import SgDisk
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    if mode == "direct":
        lay, sigma = make_config(2)
    else:
        lay = nested_layout(4, 64, 8.0, 16)
        x, y, _ = cell_centres(lay)
        sigma = kuzmin_sigma(x, y, a=0.3)
    rng = np.random.default_rng(0)
    sig_a = torch.as_tensor(sigma).cuda()
    sig_b = torch.as_tensor(sigma * (1.0 + 0.1 * rng.uniform(-1, 1, sigma.size))).cuda()
    with SgDisk.from_layout(lay, device=0) as d:
        d.set_interaction_mode(mode)
        buf = sig_a.clone()
        Fx = torch.empty(lay.n_cells, dtype=torch.float64, device="cuda")
        Fy = torch.empty_like(Fx)
        d.set_density(buf); d.force(Fx, Fy)                 # warm-up: sizes the partial-sum buffer
        torch.cuda.synchronize()
        ref_a = (Fx.clone(), Fy.clone())
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            d.set_density(buf)
            d.force(Fx, Fy)
        buf.copy_(sig_b)
        g.replay()
        torch.cuda.synchronize()
        got_b = (Fx.clone(), Fy.clone())
        d.set_density(sig_b); eager = d.force()
        torch.cuda.synchronize()
        assert torch.equal(got_b[0], eager[0]) and torch.equal(got_b[1], eager[1])      # deterministic: bit-equal
        buf.copy_(sig_a)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(Fx, ref_a[0]) and torch.equal(Fy, ref_a[1])
        assert not torch.equal(ref_a[0], got_b[0])
