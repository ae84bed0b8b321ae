"""The whole LSE+OBC path for a workload, energy by energy (what bench.py's cpu_baseline times).

TEST INFRASTRUCTURE (see oracle/__init__.py).  Chains S1-S7 of SURVEY.md 8(a) for each energy
("Each E is independent of the other"): decimation of both leads, assembly,
retarded sweeps, lesser/greater sweeps, observables.
"""
import numpy as np

from . import assemble, obc, observables, rgf


def _slice_sigma(sig, k):
    if sig is None:
        return None
    if sig["kind"] == "scalar":
        return {"kind": "scalar", "value": sig["value"][k]}
    out = {"kind": "bt", "diag": sig["diag"][k], "upper": sig["upper"][k]}
    if "lower" in sig:
        out["lower"] = sig["lower"][k]
    return out


def obc_one_energy(E, eta, H_diag, H_upper, S_diag, S_upper, mu, kT, side, tol=1e-12, max_iter=64,
                   extended=False, cond_trace=None):
    z = complex(E, eta)
    Hd, Hu, Sd, Su = obc.contact_blocks(H_diag, H_upper, S_diag, S_upper, side)
    a_d, a_u, a_l = obc.lead_blocks(z, Hd, Hu, Sd, Su)
    g_s, iters, conv = obc.sancho_rubio(a_d, a_u, a_l, side, tol, max_iter, extended=extended,
                                           cond_trace=cond_trace)
    if extended:
        a_u, a_l = a_u.astype(np.clongdouble), a_l.astype(np.clongdouble)
    sig = obc.boundary_self_energy(a_u, a_l, g_s, side)
    gam = obc.broadening(sig)
    f = obc.fermi(E, mu, kT)
    sl, sg = obc.boundary_lesser_greater(gam, f)
    return {"sigma_r": sig, "gamma": gam, "sigma_l": sl, "sigma_g": sg, "g_s": g_s,
            "iters": iters, "converged": conv, "f": f}


def solve_energy(wl, k, sigma=None, obc_in=None, want_greater=None, corner=True):
    """Full path for energy index k of Workload `wl`.
    sigma: result of wl.sigma_s(k, k+1) (computed if None).
    obc_in: optional (left, right) dicts with sigma_r/gamma/sigma_l/sigma_g to use INSTEAD of
    running the decimation (used to feed identical Sigma_B to oracle and GPU, hazard H2)."""
    E = float(wl.energies[k])
    z = complex(E, wl.eta)
    n, b = wl.n_blocks, wl.block_size
    if sigma is None:
        sigma = wl.sigma_s(k, k + 1)
    sr, sl, sg = (_slice_sigma(sigma[t], 0) for t in "rlg")
    if obc_in is None:
        left = obc_one_energy(E, wl.eta, wl.H_diag, wl.H_upper, wl.S_diag, wl.S_upper,
                              wl.mu_L, wl.kT, 0, wl.tol, wl.max_iter)
        right = obc_one_energy(E, wl.eta, wl.H_diag, wl.H_upper, wl.S_diag, wl.S_upper,
                               wl.mu_R, wl.kT, 1, wl.tol, wl.max_iter)
    else:
        left, right = obc_in
    A_diag, A_upper, A_lower = assemble.a_blocks(z, wl.H_diag, wl.H_upper, wl.S_diag, wl.S_upper,
                                                 sr, left["sigma_r"], right["sigma_r"])
    ret = rgf.rgf_retarded(A_diag, A_upper, A_lower, corner=corner)
    out = {"left": left, "right": right, "ret": ret, "A": (A_diag, A_upper, A_lower)}
    want_greater = wl.want_greater if want_greater is None else want_greater
    BL = assemble.b_blocks(n, b, sl, left["sigma_l"], right["sigma_l"])
    out["BL"] = BL
    out["les"] = rgf.rgf_lesser_greater(A_upper, A_lower, BL[0], BL[1], ret)
    if want_greater:
        BG = assemble.b_blocks(n, b, sg, left["sigma_g"], right["sigma_g"])
        out["BG"] = BG
        out["gtr"] = rgf.rgf_lesser_greater(A_upper, A_lower, BG[0], BG[1], ret)
    # observables
    obs = {"ldos": observables.ldos(ret["GR_diag"], ret["GR_upper"], ret["GR_lower"], wl.S_diag, wl.S_upper),
           "density_integrand": observables.density_integrand(out["les"]["GX_diag"], out["les"]["GX_upper"],
                                                              wl.S_diag, wl.S_upper),
           "bond_current": observables.bond_current(E, wl.H_upper, wl.S_upper, out["les"]["GX_upper"])}
    if corner:
        obs["transmission"] = observables.transmission(ret["GR_corner"][0], left["gamma"], right["gamma"])
    if want_greater:
        obs["contact_current"] = np.array([
            observables.contact_current(left["sigma_l"], left["sigma_g"],
                                        out["les"]["GX_diag"][0], out["gtr"]["GX_diag"][0]),
            observables.contact_current(right["sigma_l"], right["sigma_g"],
                                        out["les"]["GX_diag"][n - 1], out["gtr"]["GX_diag"][n - 1])])
    out["obs"] = obs
    return out


def density(wl, integrands):
    """n_k = sum_E w_E * integrand_k(E)  (R12; trapezoid weights, R8)."""
    return np.tensordot(wl.weights, np.asarray(integrands), axes=(0, 0))
