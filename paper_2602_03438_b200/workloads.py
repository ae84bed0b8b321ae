"""Seeded synthetic NEGF workloads (inputs only).

This module serves BOTH the oracle-side tests and the CUDA path.  It holds none of
the method's arithmetic: no Green's functions, no decimation, no RGF, no observables.
It only draws the block-tridiagonal inputs H, S, Sigma_S of `BASELINE.json:configs[0..4]`
with the distributions fixed in SURVEY.md section 8(c-3), readings R1-R10
(restated in DESIGN.md "Input recipe").  It imports numpy only.

Structure kept from the paper: block-tridiagonal ("a block tri-diagonal
(BT) shape is imposed on all A and B matrices"), complex Hermitian H, optional
non-orthogonal S (localized basis), contact blocks repeated into the
leads, BT scattering self-energies for the GW-like case.

Deviation from R10 (stated in DESIGN.md): instead of ONE generator stream with a fixed
draw order, every array family has its own child stream
``PCG64(SeedSequence([26020343800 + config, family_id, energy_index]))`` so that the
per-energy Sigma_S of configs[3] can be drawn batch by batch (all 32 energies do not fit
in HBM at once) and any energy can be regenerated alone for sampled parity checks.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional

import numpy as np

BASE_SEED = 26020343800

# family ids for the child streams
_F_HDIAG, _F_HUP, _F_SDIAG, _F_SUP, _F_OFFS, _F_SIG_L, _F_SIG_G, _F_SIG_P = range(8)


def _rng(config: int, family: int, sub: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([BASE_SEED + config, family, sub])))


def complex_normal(rng: np.random.Generator, shape, variance: float = 1.0) -> np.ndarray:
    """CN(0, variance): E|x|^2 = variance; re and im each N(0, variance/2)  (reading R4).
    One `standard_normal(shape + (2,))` draw per complex array (reading R10)."""
    x = rng.standard_normal(tuple(shape) + (2,))
    return (x[..., 0] + 1j * x[..., 1]) * np.sqrt(variance / 2.0)


def hermitian_blocks(rng, n: int, b: int, variance: float = 1.0) -> np.ndarray:
    """n Hermitian b x b blocks (R + R^H)/sqrt(2)/sqrt(b), R ~ CN(0, variance) (reading R4)."""
    r = complex_normal(rng, (n, b, b), variance)
    return (r + np.conj(np.swapaxes(r, -1, -2))) / np.sqrt(2.0) / np.sqrt(b)


def fermi_input(e: np.ndarray, mu: float, kt: float) -> np.ndarray:
    """Occupation used ONLY to scale the synthetic scalar Sigma^<_S of configs[1]
    (reading R5).  Input recipe, overflow-safe."""
    x = (np.asarray(e, dtype=np.float64) - mu) / kt
    out = np.empty_like(x)
    pos = x > 0
    out[pos] = np.exp(-x[pos]) / (1.0 + np.exp(-x[pos]))
    out[~pos] = 1.0 / (1.0 + np.exp(x[~pos]))
    return out


@dataclass
class Workload:
    """One synthetic device + energy grid.  Arrays are C-contiguous complex128,
    blocks row-major [.., b, b] (the layout of include/negf.h)."""

    config: int
    name: str
    n_blocks: int
    block_size: int
    energies: np.ndarray            # [N_E] float64
    eta: float
    H_diag: np.ndarray              # [n, b, b]
    H_upper: np.ndarray             # [n-1, b, b]; lower = upper^H
    S_diag: Optional[np.ndarray]    # None => S = I
    S_upper: Optional[np.ndarray]
    mu_L: float = 0.1
    mu_R: float = -0.1
    kT: float = 0.025
    tol: float = 1e-12
    max_iter: int = 64
    sigma_kind: str = "none"        # "none" | "scalar" | "bt"
    want_lesser: bool = True
    want_greater: bool = False
    weights: np.ndarray = field(default=None)  # trapezoid weights (reading R8)

    @property
    def n_energy(self) -> int:
        return int(self.energies.shape[0])

    def sigma_s(self, e_lo: int = 0, e_hi: Optional[int] = None) -> Dict[str, Optional[dict]]:
        """Scattering self-energies for energies [e_lo, e_hi).

        Returns {"r": .., "l": .., "g": ..}; each value is None (absent),
        {"kind": "scalar", "value": [ne] complex} (value * I on every diagonal block) or
        {"kind": "bt", "diag": [ne,n,b,b], "upper": [ne,n-1,b,b], "lower": [ne,n-1,b,b]}
        (for "l"/"g" lower = -upper^H is implied and "lower" is omitted).
        """
        e_hi = self.n_energy if e_hi is None else e_hi
        ne = e_hi - e_lo
        n, b = self.n_blocks, self.block_size
        if self.sigma_kind == "none":
            return {"r": None, "l": None, "g": None}
        if self.sigma_kind == "scalar":
            # reading R5: Sigma^R_S = -i*0.01*I ; Sigma^<_S = +i*0.01*f_0(E)*I (mu = 0);
            # Sigma^>_S := Sigma^<_S + Sigma^R_S - Sigma^A_S.
            f0 = fermi_input(self.energies[e_lo:e_hi], 0.0, self.kT)
            sr = np.full(ne, -0.01j, dtype=np.complex128)
            sl = (0.01j * f0).astype(np.complex128)
            sg = sl + sr - np.conj(sr)
            return {"r": {"kind": "scalar", "value": sr},
                    "l": {"kind": "scalar", "value": sl},
                    "g": {"kind": "scalar", "value": sg}}
        # "bt": reading R6.  M_<, M_>, P independent Hermitian BT, entries CN(0,1e-3)/sqrt(b).
        var = 1e-3
        out = {k: {"kind": "bt",
                   "diag": np.empty((ne, n, b, b), np.complex128),
                   "upper": np.empty((ne, max(n - 1, 0), b, b), np.complex128)} for k in "rlg"}
        out["r"]["lower"] = np.empty((ne, max(n - 1, 0), b, b), np.complex128)
        for k in range(ne):
            e = e_lo + k
            fam = {}
            for tag, fid in (("l", _F_SIG_L), ("g", _F_SIG_G), ("p", _F_SIG_P)):
                rng = _rng(self.config, fid, e)
                d = hermitian_blocks(rng, n, b, var)
                u = complex_normal(rng, (max(n - 1, 0), b, b), var) / np.sqrt(b)
                fam[tag] = (d, u)
            (ld, lu), (gd, gu), (pd, pu) = fam["l"], fam["g"], fam["p"]
            out["l"]["diag"][k] = 1j * ld
            out["l"]["upper"][k] = 1j * lu
            out["g"]["diag"][k] = -1j * gd
            out["g"]["upper"][k] = -1j * gu
            # Sigma^R = P + (Sigma^> - Sigma^<)/2
            out["r"]["diag"][k] = pd - 0.5j * (gd + ld)
            out["r"]["upper"][k] = pu - 0.5j * (gu + lu)
            h = lambda a: np.conj(np.swapaxes(a, -1, -2))
            out["r"]["lower"][k] = h(pu) - 0.5j * (h(gu) + h(lu))
        return out


_CONFIG_TABLE = {
    # config: (name, N_E, n, b)
    0: ("config0_single_energy_b16", 1, 8, 16),
    1: ("config1_64E_n32_b64_scalar_scattering", 64, 32, 64),
    2: ("config2_256E_n64_b256_nonorthogonal", 256, 64, 256),
    3: ("config3_32E_n40_b1024_bt_scattering", 32, 40, 1024),
    4: ("config4_8E_n20_b2048_offsets", 8, 20, 2048),
}


def trapezoid_weights(e: np.ndarray) -> np.ndarray:
    e = np.asarray(e, dtype=np.float64)
    if e.size == 1:
        return np.ones(1)
    w = np.zeros_like(e)
    de = np.diff(e)
    w[:-1] += 0.5 * de
    w[1:] += 0.5 * de
    return w


def make_workload(config: int, n_blocks: Optional[int] = None, block_size: Optional[int] = None,
                  n_energy: Optional[int] = None) -> Workload:
    """Workload of BASELINE.json:configs[config]; the size overrides give the SAME recipe
    at reduced (or ragged) sizes for tests."""
    name, ne0, n0, b0 = _CONFIG_TABLE[config]
    n = n0 if n_blocks is None else int(n_blocks)
    b = b0 if block_size is None else int(block_size)
    ne = ne0 if n_energy is None else int(n_energy)
    if (n, b, ne) != (n0, b0, ne0):
        name = f"{name}[n={n},b={b},NE={ne}]"

    # energies: configs[0] single E = 0.3; others linspace(-1, 1, N_E) inclusive (reading R8)
    if config == 0 and ne == 1:
        energies = np.array([0.3])
    elif ne == 1:
        energies = np.array([0.3])
    else:
        energies = np.linspace(-1.0, 1.0, ne)

    coupling = 0.7 if config == 2 else 1.0
    H_diag = hermitian_blocks(_rng(config, _F_HDIAG), n, b, 1.0)
    onsite = _rng(config, _F_HDIAG, 1).uniform(-1.0, 1.0, size=(n, b))
    idx = np.arange(b)
    H_diag[:, idx, idx] += onsite
    H_upper = coupling * complex_normal(_rng(config, _F_HUP), (max(n - 1, 0), b, b), 0.5) / np.sqrt(b)
    if config == 4:
        # reading R7: one scalar offset v_i ~ U[-2,2] per block, H_ii += v_i I
        v = _rng(config, _F_OFFS).uniform(-2.0, 2.0, size=n)
        H_diag[:, idx, idx] += v[:, None]

    S_diag = S_upper = None
    if config == 2:
        S_diag = 0.05 * hermitian_blocks(_rng(config, _F_SDIAG), n, b, 1.0)
        S_diag[:, idx, idx] += 1.0
        S_upper = 0.02 * complex_normal(_rng(config, _F_SUP), (max(n - 1, 0), b, b), 1.0) / np.sqrt(b)

    sigma_kind = {0: "none", 1: "scalar", 2: "none", 3: "bt", 4: "none"}[config]
    want_greater = config in (3, 4)
    return Workload(config=config, name=name, n_blocks=n, block_size=b, energies=energies, eta=1e-6,
                    H_diag=np.ascontiguousarray(H_diag), H_upper=np.ascontiguousarray(H_upper),
                    S_diag=S_diag, S_upper=S_upper, sigma_kind=sigma_kind,
                    want_lesser=True, want_greater=want_greater,
                    weights=trapezoid_weights(energies))


def chain_lead(b: int, seed: int = 7):
    """Lead with a known closed-form surface Green's function (SURVEY.md 8(c) pin P5):
    H_d = U diag(eps_k) U^H, H_u = U diag(-t_k) U^H with a random unitary U.
    Returns (H_d, H_u, U, eps, t).  Input construction only; the closed form itself
    lives in the tests."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([BASE_SEED, 99, seed, b])))
    q, _ = np.linalg.qr(complex_normal(rng, (b, b)))
    eps = rng.uniform(-0.5, 0.5, size=b)
    t = rng.uniform(0.3, 0.8, size=b)
    H_d = (q * eps) @ q.conj().T
    H_u = (q * (-t)) @ q.conj().T
    return H_d, H_u, q, eps, t


def shard_energies(wl: Workload, rank: int, world: int) -> Workload:
    """Energy sharding for multi-GPU runs ("Each E is independent of the other"): the
    job's grid is `world` times as dense as the config's and rank r takes every world-th point
    starting at r, so that every rank keeps N_E energies of the same range (weak scaling) and the
    union over ranks is one uniform grid.  No data-path collective is needed; only the density
    would be summed over ranks by a caller that wants the total."""
    import copy
    if world <= 1:
        return wl
    ne = wl.n_energy
    if ne == 1:
        lo, hi = float(wl.energies[0]), float(wl.energies[0]) + 1e-3 * world
    else:
        lo, hi = float(wl.energies[0]), float(wl.energies[-1])
    dense = np.linspace(lo, hi, ne * world)
    out = copy.copy(wl)
    out.energies = np.ascontiguousarray(dense[rank::world])
    w_dense = trapezoid_weights(dense)
    out.weights = np.ascontiguousarray(w_dense[rank::world])
    out.name = f"{wl.name}[rank {rank}/{world}]"
    return out
