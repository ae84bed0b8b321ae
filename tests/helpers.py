"""Shared test helpers (no method arithmetic beyond norms)."""
import numpy as np


def rel_fro(x, ref):
    """Relative Frobenius error per block, no floor (reading R14); returns the max over blocks."""
    x = np.asarray(x)
    ref = np.asarray(ref)
    if x.ndim == 2:
        x, ref = x[None], ref[None]
    x = x.reshape(-1, x.shape[-2], x.shape[-1])
    ref = ref.reshape(-1, ref.shape[-2], ref.shape[-1])
    if x.shape[0] == 0:
        return 0.0
    num = np.linalg.norm(x - ref, axis=(1, 2))
    den = np.linalg.norm(ref, axis=(1, 2))
    return float(np.max(num / den))


def fp64_oracle_ensemble(E, eta, H_diag, H_upper, S_diag, S_upper, side, tol, max_iter, k_perm=7, seed=0):
    """Sigma^R_B of one lead and energy from the fp64 oracle run as it stands AND on k_perm exactly permuted copies
    of the lead blocks (a -> P a P^T for a_d, a_u, a_l; the result is un-permuted afterwards).  A permutation
    similarity is exact in floating point, so every member solves the SAME mathematical problem with another pivot
    and summation order: the members are independent draws of the rounding error of a correct fp64 evaluation
    (SURVEY 8(c) H2 measured two such runs to differ by up to 5e-10).  The yardstick of rule H2-ii, "the FP64
    oracle's own error", is the largest error over this ensemble."""
    from oracle import obc
    Hd, Hu, Sd, Su = obc.contact_blocks(H_diag, H_upper, S_diag, S_upper, side)
    a_d, a_u, a_l = obc.lead_blocks(complex(E, eta), Hd, Hu, Sd, Su)
    b = a_d.shape[0]
    rng = np.random.default_rng(seed)
    out = []
    for j in range(k_perm + 1):
        p = np.arange(b) if j == 0 else rng.permutation(b)
        ix = np.ix_(p, p)
        g, _, _ = obc.sancho_rubio(a_d[ix], a_u[ix], a_l[ix], side, tol, max_iter)
        s_p = obc.boundary_self_energy(a_u[ix], a_l[ix], g, side)
        s = np.empty_like(s_p)
        s[ix] = s_p
        out.append(s)
    return out


def rgf_oracle_ensemble(A, B_list, members=("mirror", "perm", "mirror+perm"), seed=0):
    """The fp64 RGF oracle (oracle/rgf.py as it stands) run on exactly equivalent copies of the same block
    tridiagonal system: the chain mirrored (block i -> n-1-i, upper and lower blocks exchanged: the sweeps then run
    from the other end), every block conjugated by the same permutation (P A_ij P^T: another pivot and summation
    order), or both.  Mirroring and permuting are exact in floating point, so every member evaluates the SAME
    mathematical G^R and G^x through other rounding errors; their deviation from the run as it stands is the
    yardstick for "conditioning-limited at the 1e-10 bar".
    A = (A_diag, A_upper, A_lower), B_list = [(B_diag, B_upper), ...].  Returns a list of dicts with GR_diag,
    GR_upper, GR_lower and GX = [(GX_diag, GX_upper), ...] in the ORIGINAL labelling."""
    from oracle import rgf
    from oracle.assemble import dagger
    Ad, Au, Al = A
    n, b = Ad.shape[0], Ad.shape[1]
    rng = np.random.default_rng(seed)
    out = []
    for m in members:
        mir, perm = "mirror" in m, "perm" in m
        p = rng.permutation(b) if perm else np.arange(b)
        ix = np.ix_(p, p)
        P = lambda x: x[:, p][:, :, p]
        ad, au, al = P(Ad), P(Au), P(Al)
        bl = [(P(Bd), P(Bu)) for Bd, Bu in B_list]
        if mir:
            ad, au, al = ad[::-1].copy(), al[::-1].copy(), au[::-1].copy()
            bl = [(Bd[::-1].copy(), (-dagger(Bu))[::-1].copy()) for Bd, Bu in bl]
        ret = rgf.rgf_retarded(ad, au, al)
        gx = [rgf.rgf_lesser_greater(au, al, Bd, Bu, ret) for Bd, Bu in bl]
        Gd, Gu, Gl = ret["GR_diag"], ret["GR_upper"], ret["GR_lower"]
        X = [(x["GX_diag"], x["GX_upper"], x["GX_lower"]) for x in gx]
        if mir:
            Gd, Gu, Gl = Gd[::-1], Gl[::-1], Gu[::-1]
            X = [(xd[::-1], xl[::-1], xu[::-1]) for xd, xu, xl in X]
        inv = np.empty(b, dtype=int); inv[p] = np.arange(b)
        U = lambda x: np.ascontiguousarray(x[:, inv][:, :, inv])
        out.append({"GR_diag": U(Gd), "GR_upper": U(Gu), "GR_lower": U(Gl),
                    "GX": [(U(xd), U(xu)) for xd, xu, _ in X]})
    return out
