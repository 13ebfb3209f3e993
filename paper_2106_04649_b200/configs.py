"""The five seeded synthetic workloads of BASELINE.json `configs`.

These are stand-ins for the paper's flat-layer "oneD" data sets (901 / 1901 / 3901
co-located sources and receivers, 3.3 / 30 / 249 GB, 1 / 29 / 145 focal points), which are not
available; shapes, sizes and structure follow BASELINE.json.

This module holds parameters only — no arithmetic of the method.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Tuple

SEED0 = 210604649  # seed_k = SEED0 + k  (SURVEY.md §8(d) "Generator contract")


@dataclass(frozen=True)
class Config:
    name: str
    k: int                      # index in BASELINE.json `configs`
    n: int                      # nshot == nrec (co-located fixed spread)
    dx: float                   # m
    nt: int                     # samples per trace (power of two)
    dt: float                   # s
    nlayers: int                # L interfaces of the seeded layer model
    refl: str                   # "uniform03" | "randsign025"
    nfoc: int
    focal: str                  # rule that places the focal points
    seed: int
    A_R: float                  # frozen amplitude constant of R, units 1/(m s)
    fmin: float = 5.0
    fmax: float = 60.0
    niter: int = 16
    eps: int = 8                # window margin in samples (BASELINE.json config 0)
    fpeak: float = 25.0         # Ricker peak frequency
    half_support: float = 0.06  # s; the wavelet is set to exactly 0 for |u| > half_support
    noise_snr_db: float | None = None
    model_seed: int | None = None   # layer model seed if it differs from `seed` (config 2 reuses config 1's R)

    @property
    def rseed(self) -> int:
        return self.seed if self.model_seed is None else self.model_seed


# A_R: one frozen constant per config, chosen once so that ||N_1|| / ||N_0|| ~= 0.5 for the centre
# focal point (keeps the Neumann series convergent and every iterate far above fp32 noise).  Any
# positive constant is a valid input; DESIGN.md "Input recipe" says how these were found.
CONFIGS: Tuple[Config, ...] = (
    Config(name="tiny2d", k=0, n=101, dx=10.0, nt=512, dt=0.004, nlayers=3, refl="uniform03",
           nfoc=1, focal="single:400", seed=SEED0 + 0, A_R=0.6),
    Config(name="3GB_1foc", k=1, n=601, dx=10.0, nt=2048, dt=0.004, nlayers=8, refl="randsign025",
           nfoc=1, focal="single:800", seed=SEED0 + 1, A_R=0.125),
    Config(name="3GB_601foc", k=2, n=601, dx=10.0, nt=2048, dt=0.004, nlayers=8, refl="randsign025",
           nfoc=601, focal="line:800", seed=SEED0 + 2, A_R=0.125, model_seed=SEED0 + 1),
    Config(name="33GB_64foc", k=3, n=2001, dx=10.0, nt=2048, dt=0.004, nlayers=12, refl="randsign025",
           nfoc=64, focal="grid8x8", seed=SEED0 + 3, A_R=0.048, noise_snr_db=40.0),
    Config(name="250GB_256foc", k=4, n=3901, dx=5.0, nt=4096, dt=0.002, nlayers=16, refl="randsign025",
           nfoc=256, focal="line256:800", seed=SEED0 + 4, A_R=0.058),
)


def get(k: int) -> Config:
    return CONFIGS[k]


def scaled(k: int, **kw) -> Config:
    """A reduced copy of config k (same recipe, smaller shape) for fast parity tests."""
    return replace(CONFIGS[k], **kw)
