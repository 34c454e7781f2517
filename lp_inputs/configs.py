"""The five workloads of BASELINE.json `configs` (recipe: DESIGN.md section 4)."""
from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

BASE_SEED = 260223434

WORKLOAD_NAMES = {
    1: "synchrotron_16c_1k",
    2: "adiabatic_64c_64k",
    3: "turbulent_128c_1m",
    4: "large_256c_16m",
    5: "binsweep_512c_4m",
}


@dataclass(frozen=True)
class LPWorkload:
    index: int
    name: str
    n: int                      # cells per axis
    np: int                     # particles
    nbins: int
    e_min: float
    e_max: float
    periodic: Tuple[int, int, int]
    field_kind: str             # "uniform_b" | "homologous" | "turbulent"
    kmax: int = 0               # turbulent: 1 <= |k| <= kmax
    nmodes: int = 64
    p_index: float = 2.5        # initial power-law index (Eq. 13)
    support: Optional[Tuple[float, float]] = None   # power-law support; None = full range
    pos_box: Tuple[float, float] = (-1.0, 1.0)      # particles uniform in this cube
    xlo: Tuple[float, float, float] = (-1.0, -1.0, -1.0)   # domain [-1,1]^3
    xhi: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    kappa: float = 1.0
    u_rad_frac: float = 0.0     # u_rad = frac * <|B|^2/2>
    cfl_e: float = 0.5
    max_substeps: int = 4096
    sort_every: int = 0
    dt: float = 0.0             # 0 => derived (workload 1: loss CFL)
    steps: int = 1
    alpha: float = 0.0          # homologous flow rate
    b0: float = 0.0             # uniform_b: B = (0, 0, b0)
    vmax: float = 0.5
    brms: float = 1.0e-3
    sigma_rho: float = 0.5
    seed: int = BASE_SEED

    def scaled(self, n=None, np=None, nbins=None, steps=None, **kw):
        """A smaller (or different-bin) copy with dt rescaled to keep dt*vmax/dx fixed."""
        d = {}
        if n is not None and n != self.n:
            d["n"] = int(n)
            if self.field_kind == "turbulent":
                d["dt"] = self.dt * self.n / n
                d["kmax"] = max(1, min(self.kmax, n // 4))
        if np is not None:
            d["np"] = int(np)
        if nbins is not None:
            d["nbins"] = int(nbins)
        if steps is not None:
            d["steps"] = int(steps)
        d.update(kw)
        return replace(self, **d)


def workload(index: int) -> LPWorkload:
    """BASELINE.json configs[index-1]; readings R13, R18, R19 of DESIGN.md."""
    s = BASE_SEED + index
    if index == 1:   # pure synchrotron cooling; dt from the loss CFL (derived by the caller)
        return LPWorkload(1, WORKLOAD_NAMES[1], n=16, np=1024, nbins=64, e_min=1e1, e_max=1e6,
                          periodic=(1, 1, 1), field_kind="uniform_b", b0=1e-4, p_index=2.5,
                          support=(1e2, 1e5), steps=100, seed=s)
    if index == 2:   # homologous expansion, staged API with time-dependent fields
        return LPWorkload(2, WORKLOAD_NAMES[2], n=64, np=65536, nbins=128, e_min=1.0, e_max=1e7,
                          periodic=(0, 0, 0), field_kind="homologous", alpha=0.1, p_index=2.2,
                          pos_box=(-0.5, 0.5), dt=0.04, steps=200, seed=s)
    if index == 3:
        return LPWorkload(3, WORKLOAD_NAMES[3], n=128, np=1 << 20, nbins=128, e_min=1.0, e_max=1e7,
                          periodic=(1, 1, 1), field_kind="turbulent", kmax=8, p_index=2.5,
                          u_rad_frac=0.1, sort_every=50, dt=0.0125, steps=50, seed=s)
    if index == 4:
        return LPWorkload(4, WORKLOAD_NAMES[4], n=256, np=1 << 24, nbins=64, e_min=1.0, e_max=1e8,
                          periodic=(1, 1, 1), field_kind="turbulent", kmax=16, p_index=2.5,
                          u_rad_frac=0.1, sort_every=10, dt=0.00625, steps=20, seed=s)
    if index == 5:   # nbins is swept over 16..512 by the caller (scaled(nbins=...))
        return LPWorkload(5, WORKLOAD_NAMES[5], n=512, np=1 << 22, nbins=64, e_min=1.0, e_max=1e8,
                          periodic=(1, 1, 1), field_kind="turbulent", kmax=16, p_index=2.5,
                          u_rad_frac=0.1, sort_every=10, dt=0.003125, steps=10, seed=s)
    raise ValueError("workload index must be 1..5")
