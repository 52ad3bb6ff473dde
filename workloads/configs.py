"""The five BASELINE.json configs as concrete synthetic inputs.

They stand in for the paper's workloads: the muMAG-SP4-shaped permalloy strip
(PAPER.md:84-161), the synthetic cubic meshes of 64K..64M cells and the
512x512x90 multilayer.  Nothing here is read from a dataset.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import generators as g

MU0 = 4.0e-7 * np.pi
SEED0 = 20260601
TERM_DEMAG, TERM_EXCHANGE, TERM_ANISOTROPY, TERM_ZEEMAN = 1, 2, 4, 8


@dataclass(frozen=True)
class Config:
    name: str
    n: tuple
    d: tuple
    Ms: float
    Aex: float
    Ku: float = 0.0
    axis: tuple = (0.0, 0.0, 1.0)
    alpha: float = 0.02
    gamma: float = 2.211e5
    Hext: tuple = (0.0, 0.0, 0.0)
    terms: int = TERM_DEMAG | TERM_EXCHANGE
    dtypes: tuple = ("f64",)
    init: str = "random"
    seed: int = SEED0
    dt: float = 1e-13

    @property
    def ncell(self):
        return self.n[0] * self.n[1] * self.n[2]

    def with_mesh(self, n, name=None):
        return Config(**{**self.__dict__, "n": tuple(n), "name": name or self.name})

    def initial_m(self) -> np.ndarray:
        if self.init == "random":
            return g.random_unit_vectors(self.seed, self.n)
        if self.init == "in_plane":
            return g.in_plane_state(self.seed, self.n)
        if self.init == "smoothed":
            return g.box_filter_renormalise(g.random_unit_vectors(self.seed, self.n))
        raise ValueError(self.init)


CONFIGS = {
    1: Config("cfg1_tiny_film_16x16x2", (16, 16, 2), (5e-9, 5e-9, 3e-9), 8.0e5, 1.3e-11,
              alpha=0.5, seed=SEED0 + 1),
    2: Config("cfg2_strip_128x32x1", (128, 32, 1), (3.90625e-9, 3.90625e-9, 3e-9), 8.0e5,
              1.3e-11, alpha=0.02, Hext=(-24.6e-3 / MU0, 4.3e-3 / MU0, 0.0),
              terms=TERM_DEMAG | TERM_EXCHANGE | TERM_ZEEMAN, dtypes=("f64", "f32"),
              init="in_plane", seed=SEED0 + 2),
    3: Config("cfg3_block_256x256x64", (256, 256, 64), (2e-9, 2e-9, 2e-9), 1.0e6, 1.5e-11,
              Ku=5e5, alpha=0.1, terms=TERM_DEMAG | TERM_EXCHANGE | TERM_ANISOTROPY,
              dtypes=("f32",), init="smoothed", seed=SEED0 + 3),
    4: Config("cfg4_film_512x512x128", (512, 512, 128), (4e-9, 4e-9, 4e-9), 8.0e5, 1.3e-11,
              alpha=0.02, Hext=(0.0, 0.0, 50e-3 / MU0),
              terms=TERM_DEMAG | TERM_EXCHANGE | TERM_ZEEMAN, dtypes=("f32", "f64"),
              seed=SEED0 + 4),
    5: Config("cfg5_sweep", (64, 64, 64), (4e-9, 4e-9, 4e-9), 8.0e5, 1.3e-11, alpha=0.02,
              dtypes=("f32", "f64"), seed=SEED0 + 5),
}

SWEEP_MESHES = [(64, 64, 64), (128, 128, 128), (256, 256, 256), (512, 512, 64),
                (1024, 1024, 64), (1024, 1024, 128)]

# The paper's own benchmark meshes, none a power of two (cubes of side N = 100, 350, 400:
# PAPER.md:217, 225, 240; the 512 x 512 x 90 multilayer: PAPER.md:250).  "paper_ms": the paper's
# published demag time per evaluation in fp64 where it prints one for a single device
# (context, other hardware).
PAPER_MESHES = [(100, 100, 100), (350, 350, 350), (400, 400, 400), (512, 512, 90)]
PAPER_DEMAG_MS = {(350, 350, 350): (164.9, "1x H100 HBM3, fp64, PAPER.md:217"),
                  (100, 100, 100): (29.8, "2x Xeon 8490H, 8 MPI ranks NUMA-pinned, fp64, PAPER.md:240")}


def get_config(i: int) -> Config:
    return CONFIGS[i]
