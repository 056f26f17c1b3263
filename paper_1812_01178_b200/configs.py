"""The five BASELINE.json workloads (+ the paper's own 607M grid as number 6) as plain data.
Only dimensions, stretching, alpha = dt/(2 Re), seeds and RHS kind: no arithmetic of the method."""
from dataclasses import dataclass
import numpy as np
from . import inputs


@dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    stretch: str        # "two" | "one"
    gamma: float
    alpha: float
    rhs: str            # "uniform" | "gaussian" | "smooth"
    seed: int
    P: tuple            # partitions per line named by the config
    lz: float = 1.0
    ly: float = 1.0

    @property
    def lx(self):       # dx == dz (SURVEY 8(c) C1 reading)
        return self.lz * self.nx / self.nz

    @property
    def npts(self):
        return self.nx * self.ny * self.nz

    @property
    def nm(self):
        return self.nz // 2 + 1

    def faces(self):
        xf = inputs.faces_uniform(self.nx, self.lx)
        zf = inputs.faces_uniform(self.nz, self.lz)
        if self.stretch == "two":
            yf = inputs.faces_tanh_two_sided(self.ny, self.gamma, self.ly)
        else:
            yf = inputs.faces_tanh_one_sided(self.ny, self.gamma, self.ly)
        return xf, yf, zf

    def rhs_field(self):
        shape = (self.nz, self.ny, self.nx)
        if self.rhs == "uniform":
            return inputs.rhs_uniform(shape, self.seed)
        if self.rhs == "gaussian":
            return inputs.rhs_gaussian(shape, self.seed)
        return inputs.rhs_smooth_modes(shape, self.seed, self.lx, self.ly, self.lz)

    def rhs_helmholtz(self):
        return inputs.rhs_complex_uniform((self.nm, self.ny, self.nx), self.seed)

    def kz2(self):
        return inputs.modified_wavenumbers_z(self.nz, self.lz)


CONFIGS = (
    Config("cfg1_64x32x32", 64, 32, 32, "two", 2.0, 1e-3 / (2 * 1000.0), "uniform", 1, (4,)),
    Config("cfg2_256x128x128", 256, 128, 128, "two", 2.0, 1e-3 / (2 * 1000.0), "uniform", 2, (4, 8, 16)),
    Config("cfg3_512x256x256", 512, 256, 256, "two", 2.5, 5e-4 / (2 * 5000.0), "gaussian", 3, (8, 16, 32, 64)),
    Config("cfg4_1024x512x256", 1024, 512, 256, "one", 3.0, 5e-4 / (2 * 5000.0), "smooth", 4, (16, 32)),
    Config("cfg5_4096x288x512", 4096, 288, 512, "one", 3.0, 2e-4 / (2 * 20000.0), "smooth", 5, (16, 18)),
    # not a BASELINE.json config: the grid of the paper's own ~607M flat-plate run, 3072 x 256 x 768 cells (PAPER.md:L182,
    # L314) -- a factor 3 in x and z; cfg5's operator and right-hand side recipe.  `bench.py --config 6`.
    Config("paper607_3072x256x768", 3072, 256, 768, "one", 3.0, 2e-4 / (2 * 20000.0), "smooth", 6, (16, 32)),
)


def get(i):
    """1-based config number as in BASELINE.json / SURVEY.md."""
    return CONFIGS[i - 1]
