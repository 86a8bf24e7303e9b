"""The five synthetic workloads of BASELINE.json (`configs[0..4]`) as plain data.

This module holds NO arithmetic of the method (no Eq.4/5/6 of PAPER.md): it only
names grid sizes, generator widths and the paper's free parameters
(T0, gamma, <F>, z, cosmology) for each configuration, so that the
CUDA path, the oracle tests and bench.py all describe the same problem.

Readings: C9 defaults omega_b_h2 = 0.024, Gamma_-12 = 1,
Y = 0.24; C12 config 4 has no T0 in BASELINE.json -> 1e4 K; C5 pivot 1+delta = 10 on.
"""
from __future__ import annotations

from dataclasses import dataclass, asdict

SEED_BASE = 11054747          # seed_c = 11054747 + c


@dataclass(frozen=True)
class Workload:
    cfg: int                  # 1..5 = BASELINE.json configs[cfg-1]
    n: int                    # grid is n^3, fp32, C order [iz][iy][ix]
    box_mpch: float           # comoving side L [h^-1 Mpc]
    z: float
    sigma_g: float            # rms of the Gaussian field g behind the lognormal delta
    sigma_v: float            # rms of v_pec [km/s]
    T0: float                 # Eq.5
    gamma: float              # Eq.5
    f_target: float           # observed mean flux to match
    axes: tuple               # sightline axes, 0=x (contiguous), 1=y, 2=z
    omega_m: float = 0.3
    h: float = 0.7
    omega_b_h2: float = 0.024
    gamma_m12: float = 1.0
    y_he: float = 0.24
    delta_pivot: float = 10.0
    smooth_r: float = 2.0      # Gaussian smoothing radius of the generator [cells]

    @property
    def seed(self) -> int:
        return SEED_BASE + self.cfg

    @property
    def name(self) -> str:
        return f"cfg{self.cfg}_{self.n}cubed_L{self.box_mpch:g}_z{self.z:g}"

    def as_dict(self) -> dict:
        d = asdict(self)
        d["axes"] = list(self.axes)
        return d


WORKLOADS = {
    1: Workload(1, 64, 20.0, 2.5, 1.0, 50.0, 1.0e4, 1.5, 0.80, (0,)),
    2: Workload(2, 256, 100.0, 2.5, 1.2, 80.0, 1.5e4, 1.3, 0.78, (0,)),
    3: Workload(3, 512, 200.0, 2.25, 1.3, 100.0, 1.2e4, 1.6, 0.82, (0, 1, 2)),
    4: Workload(4, 1024, 400.0, 2.5, 1.4, 120.0, 1.0e4, 1.5, 0.80, (0,)),
    5: Workload(5, 2048, 1000.0, 2.5, 1.5, 150.0, 1.0e4, 1.5, 0.80, (0,)),
}


def scaled(w: Workload, n: int) -> Workload:
    """Same physical cell size and parameters on a smaller n^3 grid (parity-test sizes)."""
    d = asdict(w)
    d["box_mpch"] = w.box_mpch * n / w.n
    d["n"] = n
    d["axes"] = tuple(w.axes)
    return Workload(**d)
