"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path's callers and the oracle's tests.  It holds none of
the method's arithmetic: only sun-direction layouts, design-parameter draws and the
config table.  numpy only; importable without a GPU or the CUDA library.

The paper measures on TU Delft / GPS IIF meshes that are not available (PAPER.md:354-360,
396-404); these parametric workloads stand in for them.
"""
from dataclasses import dataclass

import numpy as np

FAMILY_PLATE, FAMILY_BOXWING, FAMILY_DETAILED, FAMILY_BOXWING6, FAMILY_SAIL, FAMILY_BOXWING_T = range(6)
N_PARAMS = {FAMILY_PLATE: 3, FAMILY_BOXWING: 2, FAMILY_DETAILED: 2, FAMILY_BOXWING6: 6,
            FAMILY_SAIL: 1, FAMILY_BOXWING_T: 2}
TRI_COUNT = {FAMILY_PLATE: 2, FAMILY_BOXWING: 16, FAMILY_DETAILED: 49840, FAMILY_BOXWING6: 16,
             FAMILY_SAIL: 1019698, FAMILY_BOXWING_T: 1280}
SOLAR_PRESSURE = 4.56e-6   # N/m^2 at 1 AU
MESH_SEED = 2
PARAM_SEED = 1


def fibonacci_sphere(S, front_hemisphere=False):
    """S unit vectors (body -> sun), fp64 then rounded to fp32.

    Full sphere: z_j = 1 - (2j+1)/S.  Front hemisphere (config 1): z_j = 1 - (j+1/2)/S > 0.
    phi_j = j * pi * (3 - sqrt 5).
    """
    j = np.arange(S, dtype=np.float64)
    z = 1.0 - (j + 0.5) / S if front_hemisphere else 1.0 - (2.0 * j + 1.0) / S
    phi = j * np.pi * (3.0 - np.sqrt(5.0))
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1).astype(np.float32)


def latlong_directions(n_lat, n_lon):
    """Force-map layout of the paper's figures (Fig. 5/6/12): a latitude-longitude image of sun
    directions, pixel centres, row r = polar angle theta = pi (r + 1/2) / n_lat from +z, column c = azimuth
    phi = 2 pi (c + 1/2) / n_lon.  Returns float32[n_lat * n_lon, 3] in row-major image order."""
    th = np.pi * (np.arange(n_lat, dtype=np.float64) + 0.5) / n_lat
    ph = 2.0 * np.pi * (np.arange(n_lon, dtype=np.float64) + 0.5) / n_lon
    st, ct = np.sin(th)[:, None], np.cos(th)[:, None]
    d = np.stack([st * np.cos(ph)[None, :], st * np.sin(ph)[None, :], np.broadcast_to(ct, (n_lat, n_lon))], axis=2)
    return np.ascontiguousarray(d.reshape(-1, 3), dtype=np.float32)


def draw_params(family, D, seed=PARAM_SEED):
    """float32[D, n_params] design parameters, uniform over the physical ranges of each family."""
    rng = np.random.default_rng([seed, family])
    u = rng.random((D, N_PARAMS[family]))
    if family == FAMILY_PLATE:
        th = np.tile(np.array([0.3, 0.5, 0.2]), (D, 1))                 # (alpha, rho_s, rho_d)
    elif family in (FAMILY_BOXWING, FAMILY_BOXWING_T):
        th = np.stack([2.0 + 6.0 * u[:, 0], np.pi * u[:, 1]], axis=1)   # (L, phi)
    elif family == FAMILY_DETAILED:
        th = np.pi * u                                                  # (theta_dish, phi_pan)
    elif family == FAMILY_BOXWING6:
        th = np.stack([np.pi * u[:, 0], np.pi * u[:, 1], 2.0 + 6.0 * u[:, 2],
                       0.5 + 1.5 * u[:, 3], 0.05 + 0.85 * u[:, 4], 0.05 + 0.75 * u[:, 5]], axis=1)
    elif family == FAMILY_SAIL:
        th = np.full((D, 1), 0.05)                                      # noise amplitude, m
    else:
        raise ValueError("unknown family")
    return np.ascontiguousarray(th, dtype=np.float32)


def random_directions(M, seed=3):
    """M unit vectors uniform on the sphere, fp64 then rounded to fp32: the light direction of each record of a
    per-sample-design batch ("a list of pairs consisting of light directions and design
    parameters")."""
    rng = np.random.default_rng([seed, 77])
    z = 2.0 * rng.random(M) - 1.0
    phi = 2.0 * np.pi * rng.random(M)
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1).astype(np.float32)


@dataclass(frozen=True)
class SampleConfig:
    """The paper's own workload shape: M records, each its own random design AND its own
    light direction, N Monte-Carlo samples per record, a ~1 k-face mesh, every ray tested against all triangles."""
    name: str
    family: int
    M: int
    N: int
    B: int
    seed: int = 0

    def params(self):
        return draw_params(self.family, self.M)

    def sun_dirs(self):
        return random_directions(self.M)


# "100 k light directions and/or designs x 1000 samples, ~1 k faces" (N = 2^10: the stratified grid)
SAMPLE_CONFIGS = {"paper_map": SampleConfig("paper_map", FAMILY_BOXWING_T, 100_000, 1 << 10, 4)}


@dataclass(frozen=True)
class Config:
    name: str
    family: int
    D: int
    S: int
    N: int              # rays (photons) per direction
    B: int              # max bounces (reflections followed)
    front_hemisphere: bool = False
    seed: int = 0

    def sun_dirs(self):
        return fibonacci_sphere(self.S, self.front_hemisphere)

    def params(self):
        return draw_params(self.family, self.D)

    @property
    def pairs(self):
        return self.D * self.S

    @property
    def primaries(self):
        return self.D * self.S * self.N


CONFIGS = {
    "cfg1_plate": Config("cfg1_plate", FAMILY_PLATE, 1, 64, 1 << 16, 1, front_hemisphere=True),
    "cfg2_boxwing": Config("cfg2_boxwing", FAMILY_BOXWING, 256, 1024, 1 << 18, 4),
    "cfg3_detailed": Config("cfg3_detailed", FAMILY_DETAILED, 16, 4096, 1 << 20, 8),
    "cfg4_sweep": Config("cfg4_sweep", FAMILY_BOXWING6, 4096, 256, 1 << 16, 4),
    "cfg5_sail": Config("cfg5_sail", FAMILY_SAIL, 1, 4096, 1 << 20, 8),
}


def icosphere(subdiv, radius=1.0):
    """Test mesh: subdivided icosahedron, float32[T,3,3], T = 20 * 4**subdiv (vertices on the sphere)."""
    t = (1.0 + np.sqrt(5.0)) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0], [0, -1, t], [0, 1, t],
                  [0, -1, -t], [0, 1, -t], [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], float)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11], [1, 5, 9], [5, 11, 4],
                  [11, 10, 2], [10, 7, 6], [7, 1, 8], [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8],
                  [3, 8, 9], [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]])
    tri = v[f]
    for _ in range(subdiv):
        a, b, c = tri[:, 0], tri[:, 1], tri[:, 2]
        ab, bc, ca = a + b, b + c, c + a
        ab /= np.linalg.norm(ab, axis=1, keepdims=True)
        bc /= np.linalg.norm(bc, axis=1, keepdims=True)
        ca /= np.linalg.norm(ca, axis=1, keepdims=True)
        tri = np.concatenate([np.stack([a, ab, ca], 1), np.stack([b, bc, ab], 1),
                              np.stack([c, ca, bc], 1), np.stack([ab, bc, ca], 1)])
    return np.ascontiguousarray(tri * radius, dtype=np.float32)


def dirichlet_materials(T, seed):
    """float32[T,3] (alpha, rho_s, rho_d) ~ Dirichlet(2,2,2), for user-supplied test meshes."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.dirichlet([2.0, 2.0, 2.0], size=T), dtype=np.float32)
