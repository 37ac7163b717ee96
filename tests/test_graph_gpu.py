"""tslb_step under CUDA graph capture: the step enqueues kernels only (no allocation, no
synchronisation, no host-side work that a replay would miss once the per-device launch attributes
and the tensor maps exist), so a caller can capture an EVEN number of steps (the two state buffers
are back in their roles) and replay the graph; small lattices are launch-bound and gain from it."""
import time

import numpy as np
import pytest

from paper_2501_00846_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_graph_replay_equals_direct_stepping(precision):
    import torch
    from paper_2501_00846_b200 import binding as B
    cfg = I.static_droplet(32, 8.0, seed=1)
    side = torch.cuda.Stream()
    a = B.Solver(32, 32, 32, cfg["params"], precision=precision, stream=side)
    b = B.Solver(32, 32, 32, cfg["params"], precision=precision)
    for s in (a, b):
        s.init(cfg["phi"], cfg["u"])
        s.step(2)                                   # warm-up: launch attributes, tensor maps
        s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        a.step(10)                                  # captured, not executed
    b.step(10)                                      # (capture advances the host-side buffer index
    reps = 7                                        #  by an even count: roles unchanged)
    for _ in range(reps):
        g.replay()
    b.step(10 * (reps - 1))
    torch.cuda.synchronize()
    # NOTE: the capture itself enqueued nothing, so a has run 2 + 10 * reps steps, b 2 + 10 * reps
    ga, gb = a.get(), b.get()
    a.synchronize(); b.synchronize()
    for k in ga:
        assert bool((ga[k] == gb[k]).all()), k
    # launch-bound regime: replaying 200 steps as graphs against 200 direct steps
    t0 = time.perf_counter()
    for _ in range(20):
        g.replay()
    torch.cuda.synchronize()
    t_graph = time.perf_counter() - t0
    t0 = time.perf_counter()
    b.step(200)
    torch.cuda.synchronize()
    t_direct = time.perf_counter() - t0
    print(f"[graph 32^3 {precision}] 200 steps: graph replay {t_graph * 1e3:.2f} ms, direct "
          f"launches {t_direct * 1e3:.2f} ms")
    a.close(); b.close()
