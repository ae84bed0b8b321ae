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
_F_HDIAG, _F_HUP, _F_SDIAG, _F_SUP, _F_OFFS, _F_SIG_L, _F_SIG_G, _F_SIG_P, _F_KPT = range(9)


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


def make_phonon_workload(n_blocks: int, block_size: int, n_omega: int, periodic: bool = False,
                         seed: int = 0, eta: float = 1e-4) -> Workload:
    """Phonon-like inputs for the same Eqs. 1-2 (A "made of the Hamiltonian, dynamical,
    or bare Coulomb matrices"): A(w) = (w^2 + i eta) I - Phi with the dynamical
    matrix Phi of a network of unit masses and positive springs, block tridiagonal, real symmetric,
    positive semi-definite (acoustic sum rule inside the device).  Mapping onto include/negf.h:
    H := Phi, S := I, energy := w^2.  `periodic` repeats one cell and one inter-cell coupling, which makes
    the device a piece of a perfect wire.  Inputs only; the frequencies sit inside the band."""
    n, b = int(n_blocks), int(block_size)
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([BASE_SEED, 201, seed, n, b])))
    cells = 1 if periodic else n
    K = rng.uniform(0.2, 1.0, size=(cells, b, b)) / max(b - 1, 1)
    K = np.triu(K, 1)
    K = K + np.swapaxes(K, -1, -2)                                 # springs inside a cell
    C = rng.uniform(0.2, 1.0, size=(max(cells - 1, 1), b, b)) / b   # springs cell i (row) <-> cell i+1 (column)
    if periodic:
        K = np.repeat(K, n, axis=0)
        C = np.repeat(C[:1], max(n - 1, 0), axis=0)
        left = right = C[0] if n > 1 else C[0]
    else:
        C = C[:max(n - 1, 0)]
        left = right = None
    idx = np.arange(b)
    Phi_d = -K.copy()
    Phi_d[:, idx, idx] += K.sum(axis=2)
    for i in range(n - 1):
        Phi_d[i, idx, idx] += C[i].sum(axis=1)
        Phi_d[i + 1, idx, idx] += C[i].sum(axis=0)
    if periodic and n > 1:      # the springs to the lead cells, so that every cell of the wire is the same
        Phi_d[0, idx, idx] += C[0].sum(axis=0)
        Phi_d[n - 1, idx, idx] += C[0].sum(axis=1)
    elif not periodic and n > 1:   # leads are periodic copies of the contact blocks (reading R2): tie them too
        Phi_d[0, idx, idx] += C[0].sum(axis=0)
        Phi_d[n - 1, idx, idx] += C[n - 2].sum(axis=1)
    Phi_u = -C
    wmax2 = 0.6 * float(np.max(np.linalg.eigvalsh(Phi_d[0])))
    omega2 = np.linspace(0.05 * wmax2, wmax2, int(n_omega)) if n_omega > 1 else np.array([0.4 * wmax2])
    return Workload(config=100, name=f"phonon[n={n},b={b},Nw={n_omega}]", n_blocks=n, block_size=b,
                    energies=omega2, eta=eta, H_diag=np.ascontiguousarray(Phi_d.astype(np.complex128)),
                    H_upper=np.ascontiguousarray(Phi_u.astype(np.complex128)), S_diag=None, S_upper=None,
                    sigma_kind="none", want_lesser=True, want_greater=True, weights=trapezoid_weights(omega2))


def make_coulomb_workload(n_blocks: int, block_size: int, n_omega: int, seed: int = 0):
    """Screened-Coulomb-like inputs for the same Eqs. 1-2 (C = W, B = P):
    W^R(w) = (V^-1 - P^R(w))^-1 with a block-tridiagonal Hermitian positive definite inverse bare
    interaction V^-1 and block-tridiagonal polarisations P^R, P^<, P^> per frequency, P^> - P^< = P^R - P^A.
    Mapping onto include/negf.h: H := -V^-1, S := I, energy := 0, eta := 0 (z = 0), Sigma := P, no leads.
    Returns (workload, sigma) with sigma in the layout of Workload.sigma_s().  Inputs only."""
    n, b, nw = int(n_blocks), int(block_size), int(n_omega)
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([BASE_SEED, 202, seed, n, b])))
    Vd = 0.3 * hermitian_blocks(rng, n, b, 1.0)
    idx = np.arange(b)
    Vd[:, idx, idx] += 2.0
    Vu = 0.3 * complex_normal(rng, (max(n - 1, 0), b, b), 1.0) / np.sqrt(b)
    wl = Workload(config=101, name=f"coulomb[n={n},b={b},Nw={nw}]", n_blocks=n, block_size=b,
                  energies=np.zeros(nw), eta=0.0, H_diag=np.ascontiguousarray(-Vd), H_upper=np.ascontiguousarray(-Vu),
                  S_diag=None, S_upper=None, sigma_kind="bt", want_lesser=True, want_greater=True,
                  weights=np.ones(nw))
    h = lambda a: np.conj(np.swapaxes(a, -1, -2))
    var = 1e-2
    sig = {k: {"kind": "bt", "diag": np.empty((nw, n, b, b), np.complex128),
               "upper": np.empty((nw, max(n - 1, 0), b, b), np.complex128)} for k in "rlg"}
    sig["r"]["lower"] = np.empty((nw, max(n - 1, 0), b, b), np.complex128)
    for k in range(nw):
        ld, gd, pd = (hermitian_blocks(rng, n, b, var) for _ in range(3))
        lu, gu, pu = (complex_normal(rng, (max(n - 1, 0), b, b), var) / np.sqrt(b) for _ in range(3))
        sig["l"]["diag"][k], sig["l"]["upper"][k] = 1j * ld, 1j * lu            # anti-Hermitian P^<
        sig["g"]["diag"][k], sig["g"]["upper"][k] = -1j * gd, -1j * gu          # anti-Hermitian P^>
        sig["r"]["diag"][k] = pd - 0.5j * (gd + ld)                             # P^R = Re + (P^> - P^<)/2
        sig["r"]["upper"][k] = pu - 0.5j * (gu + lu)
        sig["r"]["lower"][k] = h(pu) - 0.5j * (h(gu) + h(lu))
    return wl, sig


def make_kpoint_workloads(config: int, n_k: int, transverse: float = 0.3, **size_overrides):
    """Momentum-resolved inputs ("the momentum dependence is omitted for simplicity"; SURVEY.md 8(f)
    item 2): the device of `make_workload(config, ...)` made periodic in one transverse direction with coupling
    blocks V to the neighbouring transverse cell, Bloch-summed at n_k momenta k_j = -pi + 2 pi (j + 1/2) / n_k:
        H_ii(k)     = H_ii     + e^{ik} V_ii + e^{-ik} V_ii^H              (Hermitian for every k)
        H_{i,i+1}(k) = H_{i,i+1} + e^{ik} V+_i + e^{-ik} V-_i,   H_{i+1,i}(k) = H_{i,i+1}(k)^H
    with V_ii ~ CN(0, 1)/sqrt(b), V+-_i ~ CN(0, 0.5)/sqrt(b), all scaled by `transverse`; for non-orthogonal configs
    S(k) gets the same construction at a tenth of the overlap's own scale.  Returns (list of n_k Workloads that
    share the energy grid, k values, k weights 1/n_k).  Inputs only."""
    base = make_workload(config, **size_overrides)
    n, b = base.n_blocks, base.block_size
    rng = _rng(config, _F_KPT)
    Vd = transverse * complex_normal(rng, (n, b, b), 1.0) / np.sqrt(b)
    Vp = transverse * complex_normal(rng, (max(n - 1, 0), b, b), 0.5) / np.sqrt(b)
    Vm = transverse * complex_normal(rng, (max(n - 1, 0), b, b), 0.5) / np.sqrt(b)
    if base.S_diag is not None:
        Td = 0.005 * complex_normal(rng, (n, b, b), 1.0) / np.sqrt(b)
        Tp = 0.002 * complex_normal(rng, (max(n - 1, 0), b, b), 1.0) / np.sqrt(b)
        Tm = 0.002 * complex_normal(rng, (max(n - 1, 0), b, b), 1.0) / np.sqrt(b)
    h = lambda a: np.conj(np.swapaxes(a, -1, -2))
    ks = -np.pi + 2.0 * np.pi * (np.arange(n_k) + 0.5) / n_k
    out = []
    import copy
    for j, k in enumerate(ks):
        ph = np.exp(1j * k)
        wl = copy.copy(base)
        wl.name = f"{base.name}[k{j}/{n_k}]"
        wl.H_diag = np.ascontiguousarray(base.H_diag + ph * Vd + np.conj(ph) * h(Vd))
        wl.H_upper = np.ascontiguousarray(base.H_upper + ph * Vp + np.conj(ph) * Vm)
        if base.S_diag is not None:
            wl.S_diag = np.ascontiguousarray(base.S_diag + ph * Td + np.conj(ph) * h(Td))
            wl.S_upper = np.ascontiguousarray(base.S_upper + ph * Tp + np.conj(ph) * Tm)
        out.append(wl)
    return out, ks, np.full(n_k, 1.0 / n_k)


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
