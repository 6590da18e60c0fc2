"""Seeded synthetic inputs for the tetrahedron-DOS hot path.

This module holds *no* arithmetic of the tetrahedron method.  It only builds the
arrays the method consumes (band energies E, orbital weights W = |a_n^m|^2, the
energy grid omega), so that the CUDA path and the CPU oracle can be fed the very
same bits.  It is the only module both sides may import.

What the inputs stand in for: the paper benchmarks an eight-orbital FeSe
tight-binding model (Sec. II.A; Sec. IV.A) whose
hopping parameters are not available.  The seeded model below has the same
shapes and value ranges (8 bands, unitary eigenvectors -> weights in [0,1],
quasi-2D dispersion, ~8 eV bandwidth); recipe: SURVEY.md 8(d), DESIGN.md
"Input recipe".

Index conventions (part of the ABI, include/tetrados.h): ik = ix + N1*(iy + N2*iz),
k = 2*pi*(ix/N1, iy/N2, iz/N3).  Arrays are returned in the AoS layout
E[ik][n], W[ik][n][m]; `to_soa` gives E[n][ik], W[n][m][ik].
"""
from __future__ import annotations

import json
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
PARAMS_FILE = os.path.join(_HERE, "data", "tb8_params.json")

# hopping vectors R of the tetragonal model: three in-plane shells + weak interlayer
TB8_R = [(1, 0, 0), (0, 1, 0), (1, 1, 0), (1, -1, 0), (2, 0, 0), (0, 2, 0), (0, 0, 1)]
TB8_SIGMA = [0.3, 0.3, 0.3, 0.3, 0.3, 0.3, 0.1]  # eV
TB8_SEED = 1710
TB8_NORM_GRID = 16  # spectrum is normalised with min/max eigenvalue on this grid


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: grid, model, energy grid."""
    name: str
    nk: tuple          # (N1, N2, N3)
    model: str         # "cosine" | "tb8"
    nb: int
    norb: int
    nE: int
    omega_min: float
    omega_max: float
    host_inputs: bool = False  # config 5: inputs start in pinned host memory


# BASELINE.json `configs`, in order.  omega ranges not given there follow config 3
# ([-6, 4] eV), reading SURVEY.md 8 (table footnote).
CONFIGS = {
    "cfg1": Config("cfg1", (16, 16, 16), "cosine", 1, 1, 201, -6.5, 6.5),
    "cfg2": Config("cfg2", (32, 32, 32), "tb8", 8, 8, 1000, -6.0, 4.0),
    "cfg3": Config("cfg3", (64, 64, 64), "tb8", 8, 8, 2000, -6.0, 4.0),
    "cfg4": Config("cfg4", (128, 128, 128), "tb8", 8, 8, 4000, -6.0, 4.0),
    "cfg5": Config("cfg5", (192, 192, 192), "tb8", 8, 8, 1000, -6.0, 4.0, host_inputs=True),
    # the SHAPES of the paper's own largest benchmark (Table II
    # :320): anisotropic 60 x 60 x 10 grid (n_k = 36000), 8 bands, 1024 equidistant energies -- with the
    # seeded model standing in for FeSe (its hopping parameters are not available).
    "paper60": Config("paper60", (60, 60, 10), "tb8", 8, 8, 1024, -6.0, 4.0),
}


def omega_grid(omega_min: float, omega_max: float, nE: int) -> np.ndarray:
    """Equidistant grid, endpoints inclusive, evaluated in double then rounded to
    fp32 ("equidistantly spaced grid of 1024 energies")."""
    if nE == 1:
        return np.array([omega_min], dtype=np.float32)
    i = np.arange(nE, dtype=np.float64)
    return (omega_min + i * ((omega_max - omega_min) / (nE - 1))).astype(np.float32)


def kgrid(nk) -> np.ndarray:
    """k-vectors [nk_total][3] in units of radians, ix fastest."""
    n1, n2, n3 = nk
    iz, iy, ix = np.meshgrid(np.arange(n3), np.arange(n2), np.arange(n1), indexing="ij")
    k = np.stack([ix.ravel() / n1, iy.ravel() / n2, iz.ravel() / n3], axis=1)
    return 2.0 * np.pi * k


def cosine_band(nk, t: float = 1.0):
    """Config 1: E(k) = -2t(cos kx + cos ky + cos kz), one band, W == 1."""
    k = kgrid(nk)
    e = -2.0 * t * np.cos(k).sum(axis=1)
    E = e.astype(np.float32).reshape(-1, 1)
    W = np.ones((E.shape[0], 1, 1), dtype=np.float32)
    return E, W


def _draw_tb8_params() -> dict:
    """Draw onsite levels and hopping matrices in the documented order."""
    rng = np.random.default_rng(TB8_SEED)
    eps = rng.uniform(-2.0, 2.0, 8)
    hops = []
    for sigma in TB8_SIGMA:
        re = rng.normal(0.0, sigma / np.sqrt(2.0), (8, 8))
        im = rng.normal(0.0, sigma / np.sqrt(2.0), (8, 8))
        hops.append((re, im))
    return {
        "seed": TB8_SEED,
        "R": [list(r) for r in TB8_R],
        "sigma": TB8_SIGMA,
        "eps": eps.tolist(),
        "T_re": [h[0].tolist() for h in hops],
        "T_im": [h[1].tolist() for h in hops],
    }


def load_tb8_params() -> dict:
    """The committed parameter file is the authority (numpy does not promise
    bit-stable random streams across versions); it is drawn once if missing."""
    if not os.path.exists(PARAMS_FILE):
        os.makedirs(os.path.dirname(PARAMS_FILE), exist_ok=True)
        p = _draw_tb8_params()
        lo, hi = _tb8_raw_spectrum_range(p, (TB8_NORM_GRID,) * 3)
        p["norm_lo"], p["norm_hi"] = lo, hi
        with open(PARAMS_FILE, "w") as f:
            json.dump(p, f, indent=1)
    with open(PARAMS_FILE) as f:
        return json.load(f)


def _tb8_hraw(p: dict, k: np.ndarray) -> np.ndarray:
    """H_raw(k) = diag(eps) + sum_R [T_R e^{ik.R} + T_R^dagger e^{-ik.R}], complex128."""
    n = k.shape[0]
    H = np.zeros((n, 8, 8), dtype=np.complex128)
    H[:, np.arange(8), np.arange(8)] = np.asarray(p["eps"])
    for R, tre, tim in zip(p["R"], p["T_re"], p["T_im"]):
        T = np.asarray(tre) + 1j * np.asarray(tim)
        ph = np.exp(1j * (k @ np.asarray(R, dtype=np.float64)))
        H += ph[:, None, None] * T[None] + np.conj(ph)[:, None, None] * T.conj().T[None]
    return H


def _tb8_raw_spectrum_range(p: dict, nk):
    w = np.linalg.eigvalsh(_tb8_hraw(p, kgrid(nk)))
    return float(w.min()), float(w.max())


def _tb8_chunk(p: dict, k: np.ndarray):
    lo, hi = p["norm_lo"], p["norm_hi"]
    c, s = 0.5 * (lo + hi), 8.0 / (hi - lo)
    H = _tb8_hraw(p, k)
    H -= c * np.eye(8)
    H *= s
    H -= np.eye(8)
    w, U = np.linalg.eigh(H)           # ascending eigenvalues, U[m][n]
    Wt = (U.real ** 2 + U.imag ** 2)   # |U[m][n]|^2, shape [k][m][n]
    return w.astype(np.float32), np.ascontiguousarray(Wt.transpose(0, 2, 1)).astype(np.float32)


def tb8_hamiltonian(nk, chunk: int = 65536) -> np.ndarray:
    """The normalised Hamiltonian itself, H[ik][8][8] complex64 (exactly Hermitian after the cast): the input of the
    device-side eigensolver (Eq. 1).  tb8_bands diagonalises the same matrices on the host in complex128."""
    p = load_tb8_params()
    lo, hi = p["norm_lo"], p["norm_hi"]
    c, s = 0.5 * (lo + hi), 8.0 / (hi - lo)
    k = kgrid(nk)
    out = np.empty((k.shape[0], 8, 8), dtype=np.complex64)
    for s0 in range(0, k.shape[0], chunk):
        H = _tb8_hraw(p, k[s0:s0 + chunk])
        H -= c * np.eye(8)
        H *= s
        H -= np.eye(8)
        H = 0.5 * (H + H.conj().transpose(0, 2, 1))
        out[s0:s0 + chunk] = H.astype(np.complex64)
    return out


def random_tb_hamiltonian(nk, norb: int, seed: int, hop: float = 0.35) -> np.ndarray:
    """A seeded generic tight-binding Hamiltonian of any order (input generator for the eigensolver tests at orders
    above 8): H(k) = T0 + sum_d (T_d e^{2 pi i k_d} + h.c.), T0 Hermitian with a spread diagonal, T_d
    random complex nearest-neighbour hoppings.  Smooth and periodic in k; H[ik][norb][norb] complex64, exactly
    Hermitian after the cast."""
    rng = np.random.default_rng(seed)
    T0 = rng.normal(size=(norb, norb)) + 1j * rng.normal(size=(norb, norb))
    T0 = 0.25 * (T0 + T0.conj().T) + np.diag(np.linspace(-2.0, 2.0, norb))
    Td = hop * (rng.normal(size=(3, norb, norb)) + 1j * rng.normal(size=(3, norb, norb)))
    k = kgrid(nk)                                            # [nk][3] in units of the reciprocal lattice vectors
    ph = np.exp(2j * np.pi * k)                              # [nk][3]
    H = np.broadcast_to(T0, (k.shape[0], norb, norb)).copy()
    for d in range(3):
        hopd = ph[:, d, None, None] * Td[d][None]
        H += hopd + hopd.conj().transpose(0, 2, 1)
    H = 0.5 * (H + H.conj().transpose(0, 2, 1))
    return H.astype(np.complex64)


def tb8_bands(nk, threads: int | None = None, chunk: int = 16384):
    """Configs 2-5: E[ik][8] ascending (fp32), W[ik][n][m] = |U[m][n]|^2 (fp32).
    H(k) = s*(H_raw(k) - c) - 1 with c, s from the Nk=16 spectrum so that the
    spectrum sits in about [-5, 3] eV."""
    p = load_tb8_params()
    k = kgrid(nk)
    n = k.shape[0]
    E = np.empty((n, 8), dtype=np.float32)
    W = np.empty((n, 8, 8), dtype=np.float32)
    starts = list(range(0, n, chunk))
    threads = threads or min(len(starts), len(os.sched_getaffinity(0)))

    def work(s0):
        e, w = _tb8_chunk(p, k[s0:s0 + chunk])
        E[s0:s0 + chunk] = e
        W[s0:s0 + chunk] = w

    if threads <= 1:
        for s0 in starts:
            work(s0)
    else:
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(work, starts))
    return E, W


def random_bands(nk, nb: int, norb: int, seed: int, spread: float = 1.0):
    """Unstructured random E and W for adversarial / brute-force tests (not a
    paper workload): E ~ U(-spread, spread) sorted per k-point, W ~ U(0,1)."""
    rng = np.random.default_rng(seed)
    n = int(np.prod(nk))
    E = np.sort(rng.uniform(-spread, spread, (n, nb)), axis=1).astype(np.float32)
    W = rng.uniform(0.0, 1.0, (n, nb, norb)).astype(np.float32)
    return E, W


def make_inputs(cfg: Config | str, cache_dir: str | None = None):
    """Return (E[ik][nb], W[ik][nb][norb], omega[nE]) for a config, AoS, fp32.
    With cache_dir, the diagonalised arrays are cached as .npy (scratch only)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    om = omega_grid(cfg.omega_min, cfg.omega_max, cfg.nE)
    if cfg.model == "cosine":
        E, W = cosine_band(cfg.nk)
        return E, W, om
    if cache_dir:
        os.makedirs(cache_dir, exist_ok=True)
        tag = "tb8_%dx%dx%d" % tuple(cfg.nk)
        fe, fw = os.path.join(cache_dir, tag + "_E.npy"), os.path.join(cache_dir, tag + "_W.npy")
        if os.path.exists(fe) and os.path.exists(fw):
            return np.load(fe), np.load(fw), om
    E, W = tb8_bands(cfg.nk)
    if cache_dir:
        np.save(fe, E)
        np.save(fw, W)
    return E, W, om


def to_soa(E: np.ndarray, W: np.ndarray):
    """AoS E[ik][n], W[ik][n][m]  ->  SoA E[n][ik], W[n][m][ik] (k fastest)."""
    return np.ascontiguousarray(E.T), np.ascontiguousarray(W.transpose(1, 2, 0))
