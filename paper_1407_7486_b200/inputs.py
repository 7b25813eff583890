"""Seeded, synthetic workload definitions shared by tests/ and bench.py.

This module holds NONE of the method's arithmetic: only the five workload
shapes of BASELINE.json `configs` and the (T, rho_cm, phi_cm) grids, computed in
FP64 on the host and handed as plain arrays to both the CUDA path and the
oracle (reading A10).  Loop ensembles are produced by
`wl_loops_generate` (product, CUDA) or by the oracle's own d-loop twin; neither
lives here.

The paper's own ensembles were Matlab-generated text files that are not
available; these seeded ensembles stand in for them.
"""
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

UNIFORM = 0
SECH2 = 1
FLUXTUBE = 2      # the paper's validation profile, eq. (68)


@dataclass(frozen=True)
class WLConfig:
    name: str
    n_loops: int
    n_ppl: int
    seed: int
    profile: int                 # UNIFORM or SECH2
    params: Tuple[float, ...]    # UNIFORM: (eB,), SECH2: (eB0, lambda)
    n_T: int
    T_min: float
    T_max: float
    n_rho: int
    rho_max: float               # rho_cm uniform in [0, rho_max] ...
    circle_radius: Optional[float]   # ... or n_rho points on a circle (config 2)
    n_groups: int
    loop_dtype: str              # storage of the loop coordinates: "f64" | "f32"
    compute: Tuple[str, ...]     # kernels run on it: subset of ("f64", "f32")

    @property
    def point_evals(self) -> int:
        return self.n_loops * self.n_ppl * self.n_T * self.n_rho

    def grids(self):
        """(T[n_T], rho_cm[n_rho], phi_cm[n_rho] or None), FP64, endpoints included."""
        k = np.arange(self.n_T, dtype=np.float64)
        T = self.T_min * (self.T_max / self.T_min) ** (k / (self.n_T - 1))
        T[0], T[-1] = self.T_min, self.T_max
        if self.circle_radius is None:
            rho = self.rho_max * np.arange(self.n_rho, dtype=np.float64) / (self.n_rho - 1)
            return T, rho, None
        rho = np.full(self.n_rho, self.circle_radius, dtype=np.float64)
        phi = 2.0 * np.pi * np.arange(self.n_rho, dtype=np.float64) / self.n_rho
        return T, rho, phi


# BASELINE.json `configs`, in order.
CONFIGS = (
    WLConfig("cfg1_small_sech2", 1024, 256, 1, SECH2, (1.0, 1.0),
             16, 0.01, 10.0, 16, 4.0, None, 16, "f64", ("f64",)),
    WLConfig("cfg2_uniform_validation", 4096, 1024, 2, UNIFORM, (1.0,),
             32, 0.01, 5.0, 8, 2.0, 2.0, 32, "f64", ("f64", "f32")),
    WLConfig("cfg3_paper_scale", 16384, 2048, 3, SECH2, (1.0, 1.0),
             64, 0.001, 20.0, 64, 5.0, None, 64, "f32", ("f32",)),
    WLConfig("cfg4_narrow_flux_tube", 32768, 8192, 4, SECH2, (10.0, 0.1),
             48, 1e-4, 10.0, 128, 1.0, None, 128, "f32", ("f64", "f32")),
    WLConfig("cfg5_large_sweep", 65536, 8192, 5, SECH2, (1.0, 1.0),
             64, 0.001, 20.0, 64, 5.0, None, 256, "f32", ("f32",)),
)


def config(i: int) -> WLConfig:
    """1-based index, as in BASELINE.json / SURVEY.md section 8(a)."""
    return CONFIGS[i - 1]
