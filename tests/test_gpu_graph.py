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


def test_lattice_slope_step_and_regrouped_step_are_capturable():
    """The round-2 paths inside a CUDA graph: (a) slope terms in lattice mode on a three-level P = 16 nest (three
    function-lattice planes, forked pair-class streams, finalise_lin), (b) a regrouped zone-wise quadtree (P = 1: scatter
    into block order, inner context, gather).  Replay with new field contents equals the eager result bit for bit."""
    import torch
    from paper_2001_02765_b200 import SgDisk
    from workloads import paper_ilr_layout
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    rng = np.random.default_rng(1)
    for case in ("slopes", "regrouped"):
        lay = nested_layout(3, 64, 4.0, 16) if case == "slopes" else paper_ilr_layout(64, 3)
        x, y, _ = cell_centres(lay)
        sigma = kuzmin_sigma(x, y, a=0.3)
        g = -3.0 * sigma / (x * x + y * y + 0.09)
        fields_a = [sigma, g * x, g * y]
        fields_b = [f * (1.0 + 0.1 * rng.uniform(-1, 1, sigma.size)) for f in fields_a]
        n_f = 3 if case == "slopes" else 1
        with SgDisk.from_layout(lay, device=0) as d:
            d.set_interaction_mode("lattice")
            bufs = [torch.as_tensor(f).cuda() for f in fields_a[:n_f]]
            Fx = torch.empty(lay.n_cells, dtype=torch.float64, device="cuda")
            Fy = torch.empty_like(Fx)

            def step():
                if n_f == 3:
                    d.set_density_linear(*bufs)
                else:
                    d.set_density(bufs[0])
                d.force(Fx, Fy)
            step()                                              # warm-up (first slope call allocates)
            torch.cuda.synchronize()
            ref_a = (Fx.clone(), Fy.clone())
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr):
                step()
            for b, f in zip(bufs, fields_b):
                b.copy_(torch.as_tensor(f))
            gr.replay()
            torch.cuda.synchronize()
            got_b = (Fx.clone(), Fy.clone())
            step()
            torch.cuda.synchronize()
            assert torch.equal(got_b[0], Fx) and torch.equal(got_b[1], Fy), case
            assert not torch.equal(got_b[0], ref_a[0]), case
            assert bool(torch.isfinite(Fx).all()) and bool(torch.isfinite(Fy).all())
