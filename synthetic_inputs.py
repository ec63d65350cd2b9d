"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no MPO construction, no contraction, no
time evolution).  It only draws numbers from ``numpy.random.default_rng(seed)`` in a fixed,
documented order and packs them into arrays, so that ``oracle/`` and
``paper_1907_12044_b200/`` see bit-identical inputs without importing each other.

What stands in for what:
the paper measures on the 7-site FMO Frenkel-Holstein model with parameters from its refs
53, 72-74 (section II.C); those parameters are not available here, so
BASELINE.json's "FMO-like" random draws (same shapes: 7 electronic states, tens of modes per
state, d = 4..10, one exciton, vacuum start) stand in for them.

Draw order for a vibronic model:
``E[N_el]``, ``J`` (strict upper triangle, row-major), ``omega[N_el, n_modes]``,
``S[N_el, n_modes]`` (Huang-Rhys factors).  Energies are in cm^-1.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# 2*pi*c in rad fs^-1 per cm^-1: converts an energy in cm^-1 into an angular frequency in
# rad/fs (hbar = 1).  The library itself is unit free.
CM1_TO_RAD_PER_FS = 1.8836515673e-4


@dataclasses.dataclass(frozen=True)
class VibronicParams:
    """Raw Frenkel-Holstein parameters (Eq. 45), energies in cm^-1."""
    E: np.ndarray        # [N_el] site energies
    J: np.ndarray        # [N_el, N_el] symmetric, zero diagonal
    omega: np.ndarray    # [N_el, n_modes] mode frequencies
    S: np.ndarray        # [N_el, n_modes] Huang-Rhys factors (g = sqrt(S), reading c4)
    n_ph: int            # phonon levels kept per mode
    layout: str          # "A": one electronic site of dim N_el, then all modes site-major
                         # "B": 2-level electronic DOF followed by its own modes, repeated

    @property
    def n_el(self) -> int:
        return int(self.E.shape[0])

    @property
    def n_modes(self) -> int:
        return int(self.omega.shape[1])


@dataclasses.dataclass(frozen=True)
class ChainConfig:
    """One of BASELINE.json's chain workloads (configs 1, 3, 4, 5)."""
    name: str
    model_seed: int
    n_el: int
    n_modes: int
    n_ph: int
    e_range: tuple
    j_range: tuple
    nearest_neighbour: bool
    omega_range: tuple
    omega_log_uniform: bool
    s_range: tuple
    layout: str
    M: int
    pad_seed: int
    delta: float          # admixture added to the centre tensor (0 = none), reading c7/c8
    delta_seed: int
    krylov_dim: int
    dt_fs: float
    n_steps: int


CONFIGS = {
    # BASELINE.json configs[0]
    "tiny": ChainConfig("tiny", 1, 3, 2, 4, (-200.0, 200.0), (-100.0, 100.0), True,
                        (50.0, 500.0), False, (0.01, 0.1), "A", 16, 7, 0.0, 21, 10, 10.0, 20),
    # BASELINE.json configs[2]
    "fmo64": ChainConfig("fmo64", 5, 7, 10, 10, (-300.0, 300.0), (-100.0, 100.0), False,
                         (20.0, 1500.0), True, (0.001, 0.05), "A", 64, 7, 1e-6, 21, 10, 20.0, 50),
    # BASELINE.json configs[3]
    "fmo128": ChainConfig("fmo128", 5, 7, 10, 10, (-300.0, 300.0), (-100.0, 100.0), False,
                          (20.0, 1500.0), True, (0.001, 0.05), "A", 128, 7, 1e-6, 21, 10, 5.0, 20),
    # BASELINE.json configs[4]
    "fmo256": ChainConfig("fmo256", 6, 7, 20, 10, (-300.0, 300.0), (-100.0, 100.0), False,
                          (20.0, 1500.0), True, (0.001, 0.05), "B", 256, 7, 1e-6, 21, 10, 20.0, 20),
}


def draw_vibronic_params(cfg: ChainConfig) -> VibronicParams:
    rng = np.random.default_rng(cfg.model_seed)
    n = cfg.n_el
    E = rng.uniform(cfg.e_range[0], cfg.e_range[1], size=n)
    J = np.zeros((n, n))
    for m in range(n):
        for q in range(m + 1, n):
            v = rng.uniform(cfg.j_range[0], cfg.j_range[1])
            if cfg.nearest_neighbour and q != m + 1:
                v = 0.0
            J[m, q] = v
            J[q, m] = v
    if cfg.omega_log_uniform:
        lo, hi = math.log(cfg.omega_range[0]), math.log(cfg.omega_range[1])
        omega = np.exp(rng.uniform(lo, hi, size=(n, cfg.n_modes)))
    else:
        omega = rng.uniform(cfg.omega_range[0], cfg.omega_range[1], size=(n, cfg.n_modes))
    S = rng.uniform(cfg.s_range[0], cfg.s_range[1], size=(n, cfg.n_modes))
    return VibronicParams(E=E, J=J, omega=omega, S=S, n_ph=cfg.n_ph, layout=cfg.layout)


def complex_normal(rng: np.random.Generator, shape) -> np.ndarray:
    """Complex128 array with iid N(0,1) real and imaginary parts (drawn interleaved)."""
    raw = rng.standard_normal(tuple(shape) + (2,))
    return np.ascontiguousarray(raw[..., 0] + 1j * raw[..., 1])


def microbench_tensors(M: int, d: int = 10, D_W: int = 20, nnz: int = 6000,
                       seed: int | None = None):
    """BASELINE.json configs[1]: iid complex N(0,1) L, A, R and a W with exactly ``nnz``
    non-zero entries (positions from ``rng.choice`` without replacement).  Draw order:
    L, A, R, W positions, W values.  Seed defaults to 1000 + M."""
    rng = np.random.default_rng(1000 + M if seed is None else seed)
    L = complex_normal(rng, (M, D_W, M))
    A = complex_normal(rng, (M, d, M))
    R = complex_normal(rng, (M, D_W, M))
    total = D_W * d * d * D_W
    pos = rng.choice(total, size=min(nnz, total), replace=False)
    vals = complex_normal(rng, (pos.shape[0],))
    W = np.zeros(total, dtype=np.complex128)
    W[pos] = vals
    return L, W.reshape(D_W, d, d, D_W), A, R


def random_site_problem(Ml: int, Mr: int, d: int, Dl: int, Dr: int, density: float, seed: int):
    """A ragged single-site problem for parity tests: L[Ml,Dl,Ml], W[Dl,d,d,Dr] with the
    given element density, A[Ml,d,Mr], R[Mr,Dr,Mr]."""
    rng = np.random.default_rng(seed)
    L = complex_normal(rng, (Ml, Dl, Ml))
    A = complex_normal(rng, (Ml, d, Mr))
    R = complex_normal(rng, (Mr, Dr, Mr))
    W = complex_normal(rng, (Dl, d, d, Dr))
    mask = rng.uniform(size=W.shape) < density
    W = np.where(mask, W, 0.0).astype(np.complex128)
    return L, np.ascontiguousarray(W), A, R


def site_dims(params: VibronicParams) -> list:
    """Physical dimension of every MPS site for the model's layout (reading c1)."""
    if params.layout == "A":
        return [params.n_el] + [params.n_ph] * (params.n_el * params.n_modes)
    if params.layout == "B":
        dims = []
        for _ in range(params.n_el):
            dims += [2] + [params.n_ph] * params.n_modes
        return dims
    raise ValueError(params.layout)


def initial_occupations(params: VibronicParams, excited: int = 0) -> list:
    """Local basis index occupied on every site for 'exciton on electronic state `excited`,
    all modes in the vacuum' (BASELINE.json configs)."""
    if params.layout == "A":
        return [excited] + [0] * (params.n_el * params.n_modes)
    occ = []
    for m in range(params.n_el):
        occ += [1 if m == excited else 0] + [0] * params.n_modes
    return occ


def capped_bonds(dims, M: int) -> list:
    """Bond dimensions M_i = min(M, prod_{j<=i} d_j, prod_{j>i} d_j), i = 0..N (reading c7)."""
    n = len(dims)
    left = [1] * (n + 1)
    right = [1] * (n + 1)
    for i in range(n):
        left[i + 1] = min(left[i] * dims[i], 10 ** 12)
    for i in range(n - 1, -1, -1):
        right[i] = min(right[i + 1] * dims[i], 10 ** 12)
    return [int(min(M, left[i], right[i])) for i in range(n + 1)]


def padded_product_mps(dims, occ, M: int, pad_seed: int, delta: float = 0.0,
                       delta_seed: int = 21) -> list:
    """Right-canonical padded product state with the centre at site 0 (reading c7).

    Site i > 0 is a right isometry B_i[Ml, d, Mr] (rows orthonormal in the Ml x (d*Mr) view):
    row 0 is the product-state vector e_{occ_i} (x) e_0, rows 1.. are seeded complex-Gaussian
    vectors orthonormalised top-down by two passes of classical Gram-Schmidt.  Site 0 is the
    centre C_0[1, d_0, Mr] = e_{occ_0} (x) e_0, optionally with a `delta` complex-Gaussian
    admixture (then renormalised).  This is workload definition, not part of the paper's method
    (the paper warms up with P&C-RK4 instead)."""
    bonds = capped_bonds(dims, M)
    rng = np.random.default_rng(pad_seed)
    mps = []
    for i, d in enumerate(dims):
        Ml, Mr = bonds[i], bonds[i + 1]
        cols = d * Mr
        mat = np.zeros((Ml, cols), dtype=np.complex128)
        mat[0, occ[i] * Mr + 0] = 1.0
        if i > 0:
            for r in range(1, Ml):
                v = complex_normal(rng, (cols,))
                for _ in range(2):
                    v = v - (mat[:r].conj() @ v) @ mat[:r]
                mat[r] = v / np.linalg.norm(v)
        mps.append(np.ascontiguousarray(mat.reshape(Ml, d, Mr)))
    if delta > 0.0:
        drng = np.random.default_rng(delta_seed)
        c = mps[0] + delta * complex_normal(drng, mps[0].shape)
        mps[0] = np.ascontiguousarray(c / np.linalg.norm(c))
    return mps


def random_right_canonical_mps(dims, M: int, seed: int) -> list:
    """Random full-rank right-canonical MPS (centre at site 0, norm 1) for ragged parity cases."""
    bonds = capped_bonds(dims, M)
    rng = np.random.default_rng(seed)
    mps = []
    for i, d in enumerate(dims):
        Ml, Mr = bonds[i], bonds[i + 1]
        g = complex_normal(rng, (d * Mr, Ml))
        if i == 0:
            mps.append(np.ascontiguousarray((g / np.linalg.norm(g)).T.reshape(Ml, d, Mr)))
        else:
            q, _ = np.linalg.qr(g)
            mps.append(np.ascontiguousarray(q.T.reshape(Ml, d, Mr)))
    return mps
