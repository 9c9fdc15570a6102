"""The seeded synthetic workloads (BASELINE.json configs C1-C5) as plain parameter records.

No arithmetic of the method lives here: both the CUDA path and the oracle are driven from these
numbers and implement the pixel generators themselves (include/gray.h, oracle/gray_oracle.hpp).
"""

R_OBS = 1000.0          # image plane at r = 1000 M (paper P:130)
H = 1.0 / 32            # step parameter (paper's Delta ~ 1/32)
MAX_STEPS = 20000
R_CAPTURE_FACTOR = 1.01
R_ESCAPE_FACTOR = 1.01
SEED = 20130322         # random-pixel workloads (date of the paper's draft)

C1 = dict(name="C1", a=0.0, inc_deg=60.0, half_width=10.0, nx=64, ny=64)
C2 = dict(name="C2", a=0.9, inc_deg=60.0, half_width=10.0, nx=512, ny=512)
C3 = dict(name="C3", a=0.99, inc_deg=90.0, half_width=12.0, nx=2048, ny=2048)
C4 = dict(name="C4", a=0.7, inc_deg=45.0, half_width=15.0, seed=SEED, sizes=[2 ** 20, 2 ** 24, 2 ** 28, 2 ** 30],
          peak_steps=1000)
C5 = dict(name="C5", spins=[0.0, 0.1, 0.2, 0.3, 0.4, 0.5, 0.6, 0.7, 0.8, 0.9, 0.99],
          incs_deg=[5.0, 15.0, 25.0, 35.0, 45.0, 55.0, 65.0, 75.0, 85.0], half_width=10.0, nx=1024, ny=1024)


def shard_range(n, rank, world_size):
    """Contiguous slice [lo, hi) of n photons for `rank` of `world_size` (photons are independent,
    paper P:39: no exchange is needed during integration)."""
    lo = n * rank // world_size
    hi = n * (rank + 1) // world_size
    return lo, hi
