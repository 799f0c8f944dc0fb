"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws particle positions, forces,
torques and noise.  It is the one module both the CUDA-path tests/bench and the oracle-side tests
use, so that both sides see byte-identical arrays.  numpy only.

Recipe: everything is drawn in fp64 from
``numpy.random.default_rng(seed)`` in the fixed order positions -> forces -> torques -> noise,
then cast ONCE to the run precision; the oracle promotes those already-rounded arrays back to
fp64 exactly (S11).  a = eta = 1.  Uniform configs: positions i.i.d. uniform in a cube whose side
follows from the volume fraction phi, L = a (N 4 pi / (3 phi))^(1/3); overlaps are allowed.
The paper's own timed workload (perturbed FCC lattice) gives its densities only
in a figure that is not available; these configs stand in for it.  ``fcc`` reproduces its shape.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np


@dataclasses.dataclass(frozen=True)
class Config:
    index: int               # 1-based position in BASELINE.json "configs"
    name: str
    op: str                  # "mdot" | "mdot_batch" | "sqrt+mdot"
    precision: str           # "f32" | "f64"
    N: int
    angular: bool
    nrhs: int
    geometry: str            # "cube_side" | "phi" | "clusters"
    geom_param: float        # cube side, volume fraction, or cluster-centre cube side
    seed: int
    tol: float = 0.0         # Lanczos tolerance (config 3)
    a: float = 1.0
    eta: float = 1.0


CONFIGS = {
    1: Config(1, "c1_f64_N1024_trans", "mdot", "f64", 1024, False, 1, "cube_side", 40.0, 0),
    2: Config(2, "c2_f32_N16384_angular", "mdot", "f32", 16384, True, 1, "phi", 0.10, 1),
    3: Config(3, "c3_f32_N131072_lanczos", "sqrt+mdot", "f32", 131072, False, 1, "phi", 0.05, 2, tol=1e-3),
    4: Config(4, "c4_f32_N1048576_rhs4", "mdot_batch", "f32", 1048576, False, 4, "phi", 0.01, 3),
    5: Config(5, "c5_f64_N262144_clusters_angular", "mdot", "f64", 262144, True, 1, "clusters", 400.0, 4),
}

N_CLUSTERS = 64
CLUSTER_SIGMA = 3.0


def np_dtype(precision: str):
    return {"f32": np.float32, "f64": np.float64}[precision]


def cube_side(N: int, phi: float, a: float = 1.0) -> float:
    return a * (N * 4.0 * math.pi / (3.0 * phi)) ** (1.0 / 3.0)


def positions(cfg: Config, rng: np.random.Generator, N: int | None = None) -> np.ndarray:
    """(N,3) fp64 positions.  ``N`` overrides cfg.N keeping the density / cluster structure."""
    N = cfg.N if N is None else N
    if cfg.geometry == "cube_side":
        # config 1 fixes the side at N = 1024; keep its number density when N is overridden
        L = cfg.geom_param * (N / cfg.N) ** (1.0 / 3.0)
        return rng.random((N, 3)) * L
    if cfg.geometry == "phi":
        return rng.random((N, 3)) * cube_side(N, cfg.geom_param, cfg.a)
    if cfg.geometry == "clusters":
        # 64 Gaussian clusters, sigma = 3a, centres uniform in a cube of side 400; contiguous
        # cluster id = i // (N/64) so overlapping pairs concentrate in diagonal tiles.
        centres = rng.random((N_CLUSTERS, 3)) * cfg.geom_param
        per = -(-N // N_CLUSTERS)
        cid = np.minimum(np.arange(N) // per, N_CLUSTERS - 1)
        return centres[cid] + rng.normal(0.0, CLUSTER_SIGMA * cfg.a, (N, 3))
    raise ValueError(cfg.geometry)


def generate(index: int, N: int | None = None, seed: int | None = None) -> dict:
    """All arrays of config ``index`` (optionally at a reduced N, or with another seed for a replica), already cast to its precision.

    Keys: cfg, N, pos (N,3), forces (nrhs,N,3) or (N,3), torques (N,3) or None, noise (dof,) or None.
    """
    cfg = CONFIGS[index]
    N = cfg.N if N is None else N
    dt = np_dtype(cfg.precision)
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    pos = positions(cfg, rng, N)
    if cfg.nrhs > 1:
        forces = rng.standard_normal((cfg.nrhs, N, 3))
    else:
        forces = rng.standard_normal((N, 3))
    torques = rng.standard_normal((N, 3)) if cfg.angular else None
    noise = None
    if cfg.op == "sqrt+mdot":
        noise = rng.standard_normal((6 if cfg.angular else 3) * N)
    cast = lambda v: None if v is None else np.ascontiguousarray(v.astype(dt))
    return dict(cfg=cfg, N=N, pos=cast(pos), forces=cast(forces), torques=cast(torques), noise=cast(noise))


def noise_for(index: int, N: int | None = None) -> np.ndarray:
    """A seeded N(0,1) noise vector W (dof entries, layout [3N linear | 3N angular]) for ANY config, in its precision:
    configs 1, 2, 4, 5 are M.F workloads, but lm_sqrt_mdot_w is tested on their particle configurations too."""
    cfg = CONFIGS[index]
    N = cfg.N if N is None else N
    rng = np.random.default_rng(10_000 + cfg.seed)
    return np.ascontiguousarray(rng.standard_normal((6 if cfg.angular else 3) * N).astype(np_dtype(cfg.precision)))


def random_case(N: int, side: float, seed: int, precision: str = "f64", angular: bool = False,
                with_noise: bool = False) -> dict:
    """Free-form small case for tests: uniform in a cube of the given side (many overlaps if small)."""
    dt = np_dtype(precision)
    rng = np.random.default_rng(seed)
    pos = rng.random((N, 3)) * side
    forces = rng.standard_normal((N, 3))
    torques = rng.standard_normal((N, 3)) if angular else None
    noise = rng.standard_normal((6 if angular else 3) * N) if with_noise else None
    cast = lambda v: None if v is None else np.ascontiguousarray(v.astype(dt))
    return dict(N=N, pos=cast(pos), forces=cast(forces), torques=cast(torques), noise=cast(noise))


def fcc(n_cells: int, number_density: float, jitter: float, seed: int) -> np.ndarray:
    """Perturbed FCC lattice (the paper's Fig. 7 workload shape): 4 n^3 sites at
    number density rho = N/V (units a^-3), each displaced uniformly by up to ``jitter``."""
    cell = (4.0 / number_density) ** (1.0 / 3.0)
    base = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    g = np.stack(np.meshgrid(*[np.arange(n_cells)] * 3, indexing="ij"), -1).reshape(-1, 1, 3)
    pos = ((g + base[None]) * cell).reshape(-1, 3)
    rng = np.random.default_rng(seed)
    return pos + (rng.random(pos.shape) - 0.5) * 2.0 * jitter


# ---------------------------------------------------------------- single-wall workloads
MICROROLLER_A = 0.656          # radius in micrometres
MICROROLLER_N = 32768          # N = 2^15


def wall_slab_case(N: int, side: float, z_lo: float, z_hi: float, seed: int, precision: str = "f64", angular: bool = False,
                   with_noise: bool = False, wall_z: float = 0.0) -> dict:
    """Free-form wall test case: x, y uniform in a square of the given side, heights above the wall uniform in
    [z_lo, z_hi] (z_lo < a: particles cutting the wall; z_lo < 0: particles under it)."""
    dt = np_dtype(precision)
    rng = np.random.default_rng(seed)
    pos = np.column_stack([rng.random(N) * side, rng.random(N) * side, wall_z + z_lo + rng.random(N) * (z_hi - z_lo)])
    forces = rng.standard_normal((N, 3))
    torques = rng.standard_normal((N, 3)) if angular else None
    noise = rng.standard_normal((6 if angular else 3) * N) if with_noise else None
    cast = lambda v: None if v is None else np.ascontiguousarray(v.astype(dt))
    return dict(N=N, pos=cast(pos), forces=cast(forces), torques=cast(torques), noise=cast(noise), wall_z=float(wall_z))


def microroller_monolayer(N: int = MICROROLLER_N, a: float = MICROROLLER_A, h_g_over_a: float = 1.5, seed: int = 5, precision: str = "f32",
                          with_noise: bool = False) -> dict:
    """The initial configuration of the paper's microroller suspension, synthetic: the x-y plane of a
    60a x 4915a strip (scaled with N so that the area fraction stays that of N = 2^15) is gridded in cells of side 2a,
    N distinct cells are drawn at random (no two particles overlap) and each particle sits at the centre of its cell;
    the height of each centre is a + an exponential of mean k_BT/mg = h_g - a (Gibbs-Boltzmann above the contact
    height; h_g = 1.5a or 6.1a in the paper).  Forces and torques ~ N(0,1) (the paper drives the rollers with one
    constant torque; random inputs exercise every block).  Wall at z = 0."""
    dt = np_dtype(precision)
    rng = np.random.default_rng(seed)
    nx = 30
    ny = max(-(-2457 * N // MICROROLLER_N), -(-N // nx) + 1)
    cells = rng.choice(nx * ny, size=N, replace=False)
    x = (cells % nx + 0.5) * 2.0 * a
    y = (cells // nx + 0.5) * 2.0 * a
    z = a + rng.exponential((h_g_over_a - 1.0) * a, N)
    pos = np.column_stack([x, y, z])
    forces = rng.standard_normal((N, 3))
    torques = rng.standard_normal((N, 3))
    noise = rng.standard_normal(6 * N) if with_noise else None
    cast = lambda v: None if v is None else np.ascontiguousarray(v.astype(dt))
    return dict(N=N, a=a, pos=cast(pos), forces=cast(forces), torques=cast(torques), noise=cast(noise), wall_z=0.0)
