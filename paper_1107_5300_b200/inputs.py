"""Seeded synthetic workloads shaped like the paper's ribbons.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only draws on-site energies, vacancy flags and energy grids.
Recipe: numpy Generator(PCG64(seed)),
uniform(-W, W, size=(L, M)) float64 C order; t = -2.7 eV, eta = 1e-9 eV; energy grids are
inclusive linspaces (reading Q7).
"""
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

T_HOP = -2.7      # eV, nearest-neighbour hopping (BASELINE.json:configs[0])
ETA = 1e-9        # eV
VACANCY_ONSITE = 1e3   # eV, on-site energy written on a vacant site (BASELINE.json:configs[4])


@dataclass
class Workload:
    name: str
    M: int                       # atoms per slice (matrix size)
    L: int                       # number of slices
    onsite: np.ndarray           # [n_dev][L][M] float64
    vacancy: Optional[np.ndarray]  # [n_dev][L][M] uint8 or None
    energies: np.ndarray         # [n_E] float64
    t: float = T_HOP
    eta: float = ETA
    notes: dict = field(default_factory=dict)

    @property
    def n_dev(self):
        return self.onsite.shape[0]

    @property
    def n_E(self):
        return self.energies.shape[0]

    @property
    def slice_steps(self):
        return self.n_dev * self.n_E * self.L


def anderson(M, L, W, seed):
    """i.i.d. uniform on-site disorder in [-W, W] on every device site (reading Q13)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(-W, W, size=(L, M))


def edge_vacancies(M, L, prob, seed, edge_depth=1):
    """Each atom in the outermost `edge_depth` rows per edge is vacant with probability prob (Q16)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    vac = np.zeros((L, M), dtype=np.uint8)
    rows = list(range(edge_depth)) + list(range(M - edge_depth, M))
    draws = rng.random(size=(L, len(rows)))
    for k, j in enumerate(rows):
        vac[:, j] = (draws[:, k] < prob).astype(np.uint8)
    return vac


def config0(M=20, L=40, n_E=64):
    """Clean ribbon, closed-form check (BASELINE.json:configs[0])."""
    return Workload("configs[0] clean M=%d L=%d" % (M, L), M, L, np.zeros((1, L, M)), None,
                    np.linspace(-2.7, 2.7, n_E))


def config1(M=128, L=1000, n_E=256, seeds=(1107, 1108, 1109, 1110), W=0.25):
    """Anderson disorder +-0.25 eV, 4 disorder seeds batched (BASELINE.json:configs[1])."""
    on = np.stack([anderson(M, L, W, s) for s in seeds])
    return Workload("configs[1] M=%d L=%d x%d seeds" % (M, L, len(seeds)), M, L, on, None,
                    np.linspace(-1.0, 1.0, n_E), notes={"seeds": list(seeds), "W": W})


def config2(M=244, L=8000, n_E=512, seed=5300, W=0.1):
    """Paper-scale ribbon, the headline throughput config (BASELINE.json:configs[2])."""
    on = anderson(M, L, W, seed)[None]
    return Workload("configs[2] M=%d L=%d n_E=%d" % (M, L, n_E), M, L, on, None,
                    np.linspace(-1.0, 1.0, n_E), notes={"seed": seed, "W": W})


def config3(M=244, L=2000, n_half=512, seed=5301, W=0.1, disordered=True):
    """Precision study: half uniform in [-1,1], half clustered in [-0.05,0.05] (configs[3], Q7, Q14)."""
    on = anderson(M, L, W, seed)[None] if disordered else np.zeros((1, L, M))
    E = np.concatenate([np.linspace(-1.0, 1.0, n_half), np.linspace(-0.05, 0.05, n_half)])
    return Workload("configs[3] M=%d L=%d %s" % (M, L, "disordered" if disordered else "clean"), M, L, on, None, E,
                    notes={"seed": seed if disordered else None, "W": W if disordered else 0.0})


def config4(M=1024, L=2000, n_E=64, seed_onsite=5302, seed_vac=5303, W=0.1, prob=0.1, edge_depth=1):
    """Wide ribbon with edge roughness (BASELINE.json:configs[4], Q15, Q16)."""
    on = anderson(M, L, W, seed_onsite)
    vac = edge_vacancies(M, L, prob, seed_vac, edge_depth)
    on[vac != 0] = VACANCY_ONSITE
    return Workload("configs[4] M=%d L=%d" % (M, L), M, L, on[None], vac[None],
                    np.linspace(-0.5, 0.5, n_E), notes={"seeds": [seed_onsite, seed_vac], "W": W, "prob": prob})


NEAR_NEUTRALITY_CASES = ("clean_M20", "clean_M20_vacancy", "disordered_M128", "disordered_M128_vacancy")


def near_neutrality(case):
    """Conducting (metallic: M + 1 divisible by 3) ribbons probed at |E| = 1e-2 ... 1e-5 eV, the edge case of the method
    (PAPER.md:82): clean M = 20, L = 40 and Anderson +-0.25 eV M = 128, L = 200 (seed 4242), each also with two edge vacancies."""
    assert case in NEAR_NEUTRALITY_CASES, case
    if case.startswith("clean"):
        M, L = 20, 40
        on = np.zeros((L, M))
    else:
        M, L = 128, 200
        on = anderson(M, L, 0.25, 4242)
    vac = None
    if case.endswith("vacancy"):
        vac = np.zeros((L, M), dtype=np.uint8)
        vac[L // 2, 0] = 1
        vac[L // 3, M - 1] = 1
        on = on.copy()
        on[vac != 0] = VACANCY_ONSITE
    E = np.array([s * e for e in (1e-2, 1e-3, 1e-4, 1e-5) for s in (1.0, -1.0)])
    return Workload("near neutrality " + case, M, L, on[None], None if vac is None else vac[None], E)


def truncate(w: Workload, L: int, energy_index=None) -> Workload:
    """First L slices of the same arrays (leads then attach at slice L) and a subset of energies."""
    E = w.energies if energy_index is None else w.energies[np.asarray(energy_index)]
    vac = None if w.vacancy is None else np.ascontiguousarray(w.vacancy[:, :L])
    return Workload(w.name + " [first %d slices, %d energies]" % (L, len(E)), w.M, L,
                    np.ascontiguousarray(w.onsite[:, :L]), vac, np.ascontiguousarray(E), w.t, w.eta, dict(w.notes))


def shard(energies, world, rank):
    """Round-robin energy shard of rank `rank` ((seed, energy) pairs are independent)."""
    return np.ascontiguousarray(np.asarray(energies)[rank::world])


def unshard(parts, n_total):
    """Inverse of shard(): parts[r] holds the results of energies[r::world]."""
    world = len(parts)
    out = np.empty((parts[0].shape[0], n_total) if parts[0].ndim == 2 else n_total, dtype=parts[0].dtype)
    for r, p in enumerate(parts):
        out[..., r::world] = p
    return out
