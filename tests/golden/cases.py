"""The golden cases: which seeded input (paper_2501_00846_b200.inputs) runs for which checkpoints.

Shared by make_golden.py (which runs the ORACLE on them) and tests/test_golden_gpu.py (which
replays them through the C ABI).  Holds recipes only: no arithmetic of the method.

One file per BASELINE.json config at the config's own grid, plus the reduced
long-horizon cases of round 1.  Horizons are what the 8-core build host affords (oracle
~2.5 MLUPS there); DESIGN.md 9 states them next to the config's nominal step count.
"""
from paper_2501_00846_b200 import inputs as I

CASES = {
    # ---- reduced-size long horizons (round 1)
    "droplet32": (lambda: I.static_droplet(32, 8.0, seed=1), [1, 10, 100, 200]),
    "collision64": (lambda: I.head_on_collision(n=64, radius=6.0, half_sep=10.0),
                    [1, 10, 100, 1000, 1500]),
    "bubble32x32x64": (lambda: I.rising_bubble(nx=32, ny=32, nz=64, radius=6.0, height=16.0),
                       [1, 10, 100, 1000, 2000, 5000, 10000, 20000]),
    # ---- configs[1]: Laplace sweep, 128^3, R in {12, 16, 24, 32}
    "laplace128_R12": (lambda: I.static_droplet(128, 12.0, seed=12), [1, 10, 100, 1000, 2000]),
    "laplace128_R16": (lambda: I.static_droplet(128, 16.0, seed=16), [1, 10, 100, 500, 1000]),
    "laplace128_R24": (lambda: I.static_droplet(128, 24.0, seed=24), [1, 10, 100, 500, 1000]),
    "laplace128_R32": (lambda: I.static_droplet(128, 32.0, seed=32), [1, 10, 100, 500, 1000]),
    # ---- configs[2]: rising bubble at 128 x 128 x 256, walls in z
    # (oracle and CUDA paths alike leave the scheme's stable range between steps 500 and 550 with
    # these parameters: the file ends at 500, with a conditioning twin)
    "bubble128x128x256": (lambda: I.rising_bubble(), [1, 10, 100, 200, 300, 400, 500]),
    # ---- configs[3]: head-on collision at the graded 256^3
    "collision256": (lambda: I.head_on_collision(n=256), [1, 10, 50, 100, 200, 500, 1000]),
    # ---- configs[3] and [4] at HALF size for their full nominal step counts (5000 / 1000);
    # the emulsion keeps its volume fraction (200 droplets / 8)
    "collision128": (lambda: I.head_on_collision(n=128, radius=12.0, half_sep=20.0),
                     [1, 10, 100, 1000, 2000, 3000, 4000, 5000]),
    "emulsion192": (lambda: I.emulsion_sweep(n=192, n_drops=25), [1, 10, 100, 500, 1000]),
    # ---- configs[4]: emulsion at 384^3 (the oracle needs ~40 GB there; 512^3 does not fit)
    "emulsion384": (lambda: I.emulsion_sweep(n=384), [1, 5, 10, 20, 50, 100, 150, 200, 250]),
    # ---- NEXT-2: off-axis collision, impact parameter 0.4, at 128^3
    "offaxis128": (lambda: I.off_axis_collision(n=128, impact=0.4), [1, 10, 100, 300]),
    # ---- NEXT-2, second workload: a train of 5 droplets falling onto the bottom
    # wall (walls in z, gravity on the liquid, R20b); first contact near step 256, then every 512
    "train64x64x192": (lambda: I.droplet_train(nx=64, ny=64, nz=192),
                       [1, 10, 100, 300, 600, 1000, 1500]),
    # ... and at the grid bench.py --workload train times (first contact near step 512)
    "train128x128x768": (lambda: I.droplet_train(nx=128, ny=128, nz=768),
                         [1, 10, 100, 300, 500, 600, 700]),
}
