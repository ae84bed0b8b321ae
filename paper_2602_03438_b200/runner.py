"""Device-side driver of the hot path for a `workloads.Workload`: uploads inputs, owns output and
workspace tensors, and calls negf_obc_decimate -> negf_rgf_retarded -> negf_rgf_lesser_greater ->
negf_observables through the C ABI.  Marshalling and memory plumbing only (torch = device memory
+ streams); no arithmetic of the method happens here.
"""
from __future__ import annotations

from typing import Dict, Optional

import numpy as np
import torch

from . import negf
from .workloads import Workload

_KIND = {"none": negf.SIGMA_NONE, "scalar": negf.SIGMA_SCALAR, "bt": negf.SIGMA_BT}


def _dev(a, device):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(device)


class DevicePath:
    """One energy batch [e_lo, e_hi) of a workload resident on one GPU."""

    def __init__(self, wl: Workload, e_lo: int = 0, e_hi: Optional[int] = None, device: str = "cuda:0",
                 ctx: Optional[negf.Context] = None, want_greater: Optional[bool] = None,
                 sigma: Optional[dict] = None, alloc_outputs: bool = True, kpoints=None, k_weights=None):
        """kpoints: optional list of Workloads (one per momentum, same shape and energy grid as `wl`, e.g. from
        workloads.make_kpoint_workloads): the batch then holds every (k, E) pair in k-major order, entry
        j * N_E + e, as ONE lock-step batch (negf_problem.n_k / k_index); the quadrature weights become w_k w_E."""
        self.wl = wl
        self.device = torch.device(device)
        self.e_lo, self.e_hi = e_lo, wl.n_energy if e_hi is None else e_hi
        ne1 = self.e_hi - self.e_lo
        self.n_k = 1 if kpoints is None else len(kpoints)
        self.ne = ne1 * self.n_k
        self.n, self.b = wl.n_blocks, wl.block_size
        self.want_greater = wl.want_greater if want_greater is None else want_greater
        self.ctx = ctx or negf.Context(self.device.index or 0)
        d = self.device
        devs = [wl] if kpoints is None else list(kpoints)
        stack = lambda name: (None if getattr(devs[0], name) is None else
                              np.concatenate([getattr(w, name) for w in devs]) if kpoints is not None else getattr(wl, name))
        self.H_diag, self.H_upper = _dev(stack("H_diag"), d), _dev(stack("H_upper"), d)
        self.S_diag, self.S_upper = _dev(stack("S_diag"), d), _dev(stack("S_upper"), d)
        kw = np.ones(self.n_k) if k_weights is None else np.asarray(k_weights, dtype=np.float64)
        self.energy = _dev(np.tile(wl.energies[self.e_lo:self.e_hi].astype(np.float64), self.n_k), d)
        self.weights = _dev(np.concatenate([kw[j] * wl.weights[self.e_lo:self.e_hi].astype(np.float64)
                                            for j in range(self.n_k)]), d)
        self.k_index = None if kpoints is None else _dev(np.repeat(np.arange(self.n_k, dtype=np.int32), ne1), d)
        self.problem = negf.make_problem(self.n, self.b, self.ne, self.H_diag, self.H_upper, self.S_diag,
                                         self.S_upper, self.energy, wl.eta, self.n_k, self.k_index)
        if sigma is None:
            per_k = [w.sigma_s(self.e_lo, self.e_hi) for w in devs]
            sig = {t: (None if per_k[0][t] is None else
                       {kk: (vv if kk == "kind" else np.concatenate([p[t][kk] for p in per_k]))
                        for kk, vv in per_k[0][t].items()}) for t in "rlg"}
        else:
            sig = sigma
        self.sig_dev: Dict[str, Optional[dict]] = {}
        for t in "rlg":
            s = sig[t]
            if s is None:
                self.sig_dev[t] = None
            elif s["kind"] == "scalar":
                self.sig_dev[t] = {"kind": "scalar", "scalar": _dev(s["value"], d)}
            else:
                self.sig_dev[t] = {"kind": "bt", "diag": _dev(s["diag"], d), "upper": _dev(s["upper"], d),
                                   "lower": _dev(s.get("lower"), d)}
        kind_r = _KIND[self.sig_dev['r']['kind']] if self.sig_dev['r'] is not None else negf.SIGMA_NONE
        ws_bytes = negf.Context.workspace_bytes(self.problem, kind_r)
        self.workspace = torch.empty(ws_bytes, dtype=torch.uint8, device=d)
        self.ctx.set_workspace(self.workspace)
        self.ctx.set_stream(torch.cuda.current_stream(d).cuda_stream)
        self.out: Dict[str, torch.Tensor] = {}
        if alloc_outputs:
            self._alloc()

    def _alloc(self):
        ne, n, b, d = self.ne, self.n, self.b, self.device
        z = lambda *shape: torch.empty(shape, dtype=torch.complex128, device=d)
        r = lambda *shape: torch.empty(shape, dtype=torch.float64, device=d)
        i = lambda *shape: torch.empty(shape, dtype=torch.int32, device=d)
        o = self.out
        for side in "LR":
            for k in ("sigma_r", "gamma", "sigma_l", "sigma_g", "g_s"):
                o[f"{k}_{side}"] = z(ne, b, b)
            o[f"fermi_{side}"] = r(ne)
            o[f"iters_{side}"] = i(ne)
            o[f"status_{side}"] = i(ne)
        o["GR_diag"], o["GR_upper"], o["GR_lower"] = z(ne, n, b, b), z(ne, n - 1, b, b), z(ne, n - 1, b, b)
        o["GR_corner"] = z(ne, b, b)
        o["GL_diag"], o["GL_upper"] = z(ne, n, b, b), z(ne, n - 1, b, b)
        if self.want_greater:
            o["GG_diag"], o["GG_upper"] = z(ne, n, b, b), z(ne, n - 1, b, b)
        o["info_r"], o["info_x"] = i(ne), i(ne)
        o["density"], o["ldos"], o["transmission"] = r(n * b), r(ne, n), r(ne)
        o["bond_current"], o["contact_current"] = r(ne, max(n - 1, 1)), r(ne, 2)

    # -- the four calls -----------------------------------------------------------------------
    def _sigma(self, t: str, left=None, right=None) -> negf.Sigma:
        s = self.sig_dev[t]
        if s is None:
            return negf.make_sigma(negf.SIGMA_NONE, left=left, right=right)
        if s["kind"] == "scalar":
            return negf.make_sigma(negf.SIGMA_SCALAR, scalar=s["scalar"], left=left, right=right)
        return negf.make_sigma(negf.SIGMA_BT, diag=s["diag"], upper=s["upper"], lower=s["lower"],
                               left=left, right=right)

    def obc(self, pair: bool = True):
        wl, o = self.wl, self.out
        if pair:
            d = lambda t: {"sigma_r": o[f"sigma_r_{t}"], "gamma": o[f"gamma_{t}"], "sigma_lesser": o[f"sigma_l_{t}"],
                           "sigma_greater": o[f"sigma_g_{t}"], "g_surface": o[f"g_s_{t}"], "fermi": o[f"fermi_{t}"],
                           "iters": o[f"iters_{t}"], "status": o[f"status_{t}"]}
            self.ctx.obc_decimate_pair(self.problem, wl.mu_L, wl.mu_R, wl.kT, wl.tol, wl.max_iter, d("L"), d("R"))
            return
        for side, tag, mu in ((0, "L", wl.mu_L), (1, "R", wl.mu_R)):
            self.ctx.obc_decimate(self.problem, side, mu, wl.kT, wl.tol, wl.max_iter, o[f"sigma_r_{tag}"],
                                  o[f"gamma_{tag}"], o[f"sigma_l_{tag}"], o[f"sigma_g_{tag}"], o[f"g_s_{tag}"],
                                  o[f"fermi_{tag}"], o[f"iters_{tag}"], o[f"status_{tag}"])

    def set_boundary(self, left: dict, right: dict):
        """Overwrite the boundary blocks with given host arrays (feeding the oracle's Sigma_B, H2)."""
        for tag, src in (("L", left), ("R", right)):
            for k in ("sigma_r", "gamma", "sigma_l", "sigma_g"):
                self.out[f"{k}_{tag}"].copy_(torch.from_numpy(np.ascontiguousarray(src[k])))

    def retarded(self, corner: bool = True, keep: bool = True):
        o = self.out
        self._sr = self._sigma("r", o["sigma_r_L"], o["sigma_r_R"])
        self.ctx.rgf_retarded(self.problem, self._sr, o["GR_diag"], o["GR_upper"] if self.n > 1 else None,
                              o["GR_lower"] if self.n > 1 else None, o["GR_corner"] if corner else None,
                              negf.KEEP_SWEEP if keep else 0, o["info_r"])

    def lesser_greater(self):
        o = self.out
        sl = self._sigma("l", o["sigma_l_L"], o["sigma_l_R"])
        sg = self._sigma("g", o["sigma_g_L"], o["sigma_g_R"]) if self.want_greater else None
        self.ctx.rgf_lesser_greater(self.problem, self._sr, sl, sg, o["GR_diag"], o["GL_diag"],
                                    o["GL_upper"] if self.n > 1 else None, o.get("GG_diag"),
                                    o.get("GG_upper") if self.n > 1 else None, o["info_x"])

    def observables(self):
        o = self.out
        g = self.want_greater
        self.ctx.observables(self.problem, o["GR_diag"], o["GR_upper"], o["GR_lower"], o["GR_corner"], o["GL_diag"],
                             o["GL_upper"], o.get("GG_diag"), o["gamma_L"], o["gamma_R"],
                             o["sigma_l_L"] if g else None, o["sigma_g_L"] if g else None,
                             o["sigma_l_R"] if g else None, o["sigma_g_R"] if g else None,
                             self.weights, o["density"], o["ldos"], o["transmission"],
                             o["bond_current"] if self.n > 1 else None, o["contact_current"] if g else None)

    def run_four_calls(self):
        """One pass of the whole hot path (S1-S7) as the four C-ABI calls, one after the other on this context."""
        self.obc()
        self.retarded()
        self.lesser_greater()
        self.observables()

    def run(self):
        """One pass of the whole hot path (S1-S7) over this energy batch through negf_pipeline_device: the same
        four steps, scheduled by the library (concurrent energy groups in the small-block regime)."""
        o, wl, g = self.out, self.wl, self.want_greater
        if not hasattr(self, "_dev_out"):
            obc = lambda t: negf.ObcOut(*[negf._ptr(o[f"{k}_{t}"]) for k in
                                          ("sigma_r", "gamma", "sigma_l", "sigma_g", "g_s", "fermi", "iters", "status")])
            m = self.n > 1
            self._dev_out = negf.DeviceOutputs(
                obc("L"), obc("R"), negf._ptr(o["GR_diag"]), negf._ptr(o["GR_upper"] if m else None),
                negf._ptr(o["GR_lower"] if m else None), negf._ptr(o["GR_corner"]), negf._ptr(o["GL_diag"]),
                negf._ptr(o["GL_upper"] if m else None), negf._ptr(o.get("GG_diag")),
                negf._ptr(o.get("GG_upper") if m else None), negf._ptr(o["density"]), negf._ptr(o["ldos"]),
                negf._ptr(o["transmission"]), negf._ptr(o["bond_current"] if m else None),
                negf._ptr(o["contact_current"] if g else None), negf._ptr(o["info_r"]), negf._ptr(o["info_x"]))
        self._sr = self._sigma("r", o["sigma_r_L"], o["sigma_r_R"])
        self.ctx.pipeline_device(self.problem, self._sigma("r"), self._sigma("l"), self._sigma("g") if g else None,
                                 self.weights, wl.mu_L, wl.mu_R, wl.kT, wl.tol, wl.max_iter, self._dev_out)

    def host(self, name: str) -> np.ndarray:
        return self.out[name].cpu().numpy()


class HostPath:
    """The whole path through negf_pipeline_host: HOST (pinned) inputs and outputs, host<->device copies
    inside the call (what bench.py times as the end-to-end number)."""

    def __init__(self, wl: Workload, n_energy: Optional[int] = None, device: str = "cuda:0",
                 ctx: Optional[negf.Context] = None, want_greater: Optional[bool] = None, blocks: bool = True,
                 kpoints=None, k_weights=None):
        """blocks=False: the G block outputs are NULL (only the observables come back to the host).
        kpoints / k_weights: as for DevicePath (every (k, E) pair in k-major order as one batch)."""
        self.wl = wl
        self.device = torch.device(device)
        ne1 = wl.n_energy if n_energy is None else min(n_energy, wl.n_energy)
        self.n_k = 1 if kpoints is None else len(kpoints)
        self.ne = ne1 * self.n_k
        self.n, self.b = wl.n_blocks, wl.block_size
        self.want_greater = wl.want_greater if want_greater is None else want_greater
        self.ctx = ctx or negf.Context(self.device.index or 0)
        ne, n, b = self.ne, self.n, self.b
        pin = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        devs = [wl] if kpoints is None else list(kpoints)
        stack = lambda name: (None if getattr(devs[0], name) is None else np.concatenate([getattr(w, name) for w in devs]))
        kw = np.ones(self.n_k) if k_weights is None else np.asarray(k_weights, dtype=np.float64)
        self._keep = [pin(stack("H_diag")), pin(stack("H_upper")), pin(stack("S_diag")), pin(stack("S_upper")),
                      pin(np.tile(wl.energies[:ne1].astype(np.float64), self.n_k)),
                      pin(np.concatenate([kw[j] * wl.weights[:ne1].astype(np.float64) for j in range(self.n_k)]))]
        Hd, Hu, Sd, Su, en, self.weights = self._keep
        kidx = None if kpoints is None else np.repeat(np.arange(self.n_k, dtype=np.int32), ne1)
        self._keep.append(kidx)
        self.problem = negf.make_problem(n, b, ne, Hd, Hu, Sd, Su, en, wl.eta, self.n_k, kidx)
        per_k = [w.sigma_s(0, ne1) for w in devs]
        sig = {t: (None if per_k[0][t] is None else
                   {kk: (vv if kk == "kind" else np.concatenate([p[t][kk] for p in per_k]))
                    for kk, vv in per_k[0][t].items()}) for t in "rlg"}
        self.sig = {}
        for t in "rlg":
            s = sig[t]
            if t == "g" and not self.want_greater:
                self.sig[t] = None
            elif s is None:
                self.sig[t] = negf.make_sigma(negf.SIGMA_NONE)
            elif s["kind"] == "scalar":
                v = pin(s["value"]); self._keep.append(v)
                self.sig[t] = negf.make_sigma(negf.SIGMA_SCALAR, scalar=v)
            else:
                d, u, l = pin(s["diag"]), pin(s["upper"]), pin(s.get("lower")); self._keep += [d, u, l]
                self.sig[t] = negf.make_sigma(negf.SIGMA_BT, diag=d, upper=u, lower=l)
        kind = _KIND[wl.sigma_kind]
        self.scratch = torch.empty(negf.Context.pipeline_host_bytes(self.problem, kind, self.want_greater),
                                   dtype=torch.uint8, device=self.device)
        z = lambda *s: torch.empty(s, dtype=torch.complex128).pin_memory() if blocks else None
        r = lambda *s: torch.empty(s, dtype=torch.float64).pin_memory()
        g = self.want_greater
        self.out = {"GR_diag": z(ne, n, b, b), "GR_upper": z(ne, n - 1, b, b), "GR_lower": z(ne, n - 1, b, b),
                    "GL_diag": z(ne, n, b, b), "GL_upper": z(ne, n - 1, b, b),
                    "GG_diag": z(ne, n, b, b) if g else None, "GG_upper": z(ne, n - 1, b, b) if g else None,
                    "density": r(n * b), "ldos": r(ne, n), "transmission": r(ne), "bond_current": r(ne, n - 1),
                    "contact_current": r(ne, 2) if g else None, "info": torch.empty(ne, dtype=torch.int32).pin_memory()}
        self._ho = negf.HostOutputs(*[negf._ptr(self.out[k]) for k in
                                      ("GR_diag", "GR_upper", "GR_lower", "GL_diag", "GL_upper", "GG_diag", "GG_upper",
                                       "density", "ldos", "transmission", "bond_current", "contact_current", "info")])

    def run(self):
        """One synchronising call; returns (h2d_bytes, d2h_bytes)."""
        wl = self.wl
        return self.ctx.pipeline_host(self.problem, self.sig["r"], self.sig["l"], self.sig["g"], self.weights,
                                      wl.mu_L, wl.mu_R, wl.kT, wl.tol, wl.max_iter, self.scratch, self._ho)
