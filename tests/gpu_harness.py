"""Helpers shared by the `-m gpu` parity tests: move a seeded WaterBox to the device, run the CUDA
path through the C ABI (via the thin binding) and compare with the CPU fp64 oracle.

Tolerances (BASELINE.json north_star, restated in DESIGN.md "Parity bar"):
  neighbour set  bit-exact as a sorted (i,j) set, ignoring pairs within 1e-5 nm of r_cut + skin
  fp32 / mixed   |E - E_orc| / |E_orc| <= 1e-5 ;  max_i |dF_i| <= 1e-4 * RMS(F) (+ allow_i, reading C-10)
  fp64           both 1e-10
"""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos

BAND = 1e-5  # nm, half-width of the ambiguity band around r_nl (sets) and r_c (forces, C-10)
TOL = {"f32": (1e-5, 1e-4), "mixed": (1e-5, 1e-4), "f64": (1e-10, 1e-10)}
METHOD = {"rf": oracle.METHOD_RF, "ewald": oracle.METHOD_EWALD_REAL}


def real_of(precision):
    return torch.float64 if precision == "f64" else torch.float32


def lj_table_np(wb):
    return oracle.lorentz_berthelot(wb.sigma, wb.epsilon)


class DeviceBox:
    """Device copies of one WaterBox in the element type of `precision`."""

    def __init__(self, wb, precision, box=None, pos=None):
        dev = torch.device("cuda", 0)
        real = real_of(precision)
        self.wb = wb
        self.box = np.asarray(wb.box if box is None else box, dtype=np.float64)
        p = wb.pos if pos is None else pos
        self.pos_np = np.ascontiguousarray(p)
        self.pos = torch.from_numpy(np.ascontiguousarray(p)).to(dev, real).contiguous()
        self.charge = torch.from_numpy(wb.charge).to(dev, real).contiguous()
        self.type = torch.from_numpy(wb.type).to(dev).contiguous()
        self.excl = torch.from_numpy(wb.excl_pairs).to(dev).contiguous()
        self.lj_np = lj_table_np(wb)
        self.lj = torch.from_numpy(self.lj_np).to(dev).contiguous()


def pair_keys(pairs, n):
    pairs = np.asarray(pairs, dtype=np.int64).reshape(-1, 2)
    return pairs[:, 0] * n + pairs[:, 1]


def check_neighbor_set(gpu_pairs, pos, box, r_nl, excl_pairs):
    """GPU pair set == oracle pair set outside the +-BAND shell around r_nl (north_star, reading C-9)."""
    n = pos.shape[0]
    gp = np.asarray(gpu_pairs, dtype=np.int64).reshape(-1, 2)
    assert np.all(gp[:, 0] < gp[:, 1]), "exported pairs must have i < j"
    gk = np.sort(pair_keys(gp, n))
    assert np.all(np.diff(gk) > 0), "duplicate pair in the exported neighbour set"
    must = pair_keys(oracle.neighbor_pairs(pos, box, r_nl - BAND, excl_pairs, "celllist"), n)
    may = pair_keys(oracle.neighbor_pairs(pos, box, r_nl + BAND, excl_pairs, "celllist"), n)
    missing = np.setdiff1d(must, gk)
    extra = np.setdiff1d(gk, may)
    assert missing.size == 0, f"{missing.size} oracle pairs missing from the GPU list, first (i,j)={divmod(int(missing[0]), n)}"
    assert extra.size == 0, f"{extra.size} GPU pairs not in the oracle set, first (i,j)={divmod(int(extra[0]), n)}"
    return len(gk), len(must), len(may)


def check_neighbor_set_device(gpu_pairs, pos, box, r_nl, excl_pairs):
    """check_neighbor_set for lists of 1e7 ... 3e8 pairs: the same comparison (sorted int64 keys i * n + j; every oracle
    pair with r < r_nl - BAND is in the GPU set, every GPU pair has r < r_nl + BAND in the oracle) with the sorting and
    the membership tests done by torch on the device.  gpu_pairs: (m, 2) int32 CUDA tensor."""
    n = pos.shape[0]
    assert bool((gpu_pairs[:, 0] < gpu_pairs[:, 1]).all()), "exported pairs must have i < j"
    gk = torch.sort(gpu_pairs[:, 0].long() * n + gpu_pairs[:, 1].long()).values
    assert bool((gk[1:] > gk[:-1]).all()), "duplicate pair in the exported neighbour set"
    counts = {}
    for name, radius in (("must", r_nl - BAND), ("may", r_nl + BAND)):
        op = torch.from_numpy(oracle.neighbor_pairs(pos, box, radius, excl_pairs, "celllist")).to(gk.device)
        ok = torch.sort(op[:, 0].long() * n + op[:, 1].long()).values
        del op
        counts[name] = int(ok.numel())
        if name == "must":  # every oracle pair is in the GPU set
            idx = torch.searchsorted(gk, ok).clamp_(max=gk.numel() - 1)
            bad = ok[gk[idx] != ok]
            assert bad.numel() == 0, f"{bad.numel()} oracle pairs missing from the GPU list, first (i,j)={divmod(int(bad[0]), n)}"
        else:  # every GPU pair is in the oracle's wider set
            idx = torch.searchsorted(ok, gk).clamp_(max=ok.numel() - 1)
            bad = gk[ok[idx] != gk]
            assert bad.numel() == 0, f"{bad.numel()} GPU pairs not in the oracle set, first (i,j)={divmod(int(bad[0]), n)}"
        del ok, idx, bad
    return int(gk.numel()), counts["must"], counts["may"]


def check_nonbonded(F, E, W, orc, precision, use_allow=True, e_floor=0.0):
    """Element-by-element force comparison + energy components + virial against an oracle result.
    e_floor: lower bound of the energy scale the relative error refers to -- along a trajectory the total energy of the
    relaxing box passes through zero, where |dE| / |E| has no meaning; the trajectory test passes |E| of its first frame."""
    e_tol, f_tol = TOL[precision]
    F = np.asarray(F, dtype=np.float64)
    E = np.asarray(E, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64).reshape(3, 3)
    rms = float(np.sqrt((orc.F ** 2).sum(axis=1).mean()))
    dF = np.sqrt(((F - orc.F) ** 2).sum(axis=1))
    allow = orc.allow if (use_allow and orc.allow is not None and precision != "f64") else np.zeros_like(dF)
    # reading C-10: the allowance is rare (SURVEY expects ~2.8 % of atoms own a pair within 1e-5 nm of r_c)
    # in a uniform fluid: 2 atoms per pair in the shell r_c +- BAND, i.e. a fraction 2 (n_pairs / N) 6 BAND / r_c with r_c ~ 1 nm
    # (2.5 % for water); the bound is twice that, and never below the 5 % that holds for every water box
    expect = 2.0 * orc.n_pairs / max(len(dF), 1) * 6.0 * BAND
    assert (allow > 0).mean() <= max(0.05, 2.0 * expect), f"{(allow > 0).mean():.3f} of the atoms carry a cutoff-band allowance"
    excess = dF - allow
    worst = int(np.argmax(excess))
    assert excess[worst] <= f_tol * rms, (
        f"force mismatch atom {worst}: |dF|={dF[worst]:.3e} allow={allow[worst]:.3e} tol={f_tol * rms:.3e} rms={rms:.3e}")
    e_err = abs(E[0] - orc.E[0]) / max(abs(orc.E[0]), e_floor) if max(abs(orc.E[0]), e_floor) != 0 else abs(E[0])
    assert e_err <= e_tol, f"energy mismatch: gpu {E[0]!r} oracle {orc.E[0]!r} rel {e_err:.3e}"
    # components relative to the sum of magnitudes (reading C-11); virial likewise
    comp_scale = np.abs(orc.E[1:]).sum()
    assert np.abs(E[1:] - orc.E[1:]).max() <= max(e_tol * comp_scale * 10, 1e-9), (E, orc.E)
    assert abs(E[0] - E[1:].sum()) <= 1e-9 * max(1.0, comp_scale)
    w_scale = np.abs(orc.W).max()
    w_tol = (1e-4 if precision != "f64" else 1e-9) * w_scale
    assert np.abs(W - orc.W).max() <= w_tol, f"virial mismatch {np.abs(W - orc.W).max():.3e} > {w_tol:.3e}"
    return {"max_dF_over_rms": float(dF.max() / rms), "n_allow": int((allow > 0).sum()), "e_rel": float(e_err)}


def run_case(wb, precision, r_cut, skin, method, box=None, pos=None, eps_rf=78.5, alpha=3.12, oracle_alg="celllist",
             check_set=True, r_switch=0.0, exceptions=None, on_device=False):
    """Build + export + nonbonded on the GPU, compare all of it with the oracle.  Returns a small report.
    on_device: sort / compare the pair keys with torch on the GPU (the 1e8-pair sets of the full-size configs), and
    compare the in-cutoff pair count dimos_nl_count_within(r_cut) -- the numerator of bench.py's metric -- with the
    oracle's, up to the pairs within BAND of r_cut."""
    db = DeviceBox(wb, precision, box=box, pos=pos)
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, r_cut, skin, db.excl)
        rep = {"stats": nl.stats()}
        assert torch.equal(nl.pos_at_build, db.pos)
        pos64 = db.pos.double().cpu().numpy()
        if check_set and on_device:
            gp = dimos.dimos_nl_export_pairs(ctx, nl)
            rep["set"] = check_neighbor_set_device(gp, pos64, db.box, r_cut + skin, wb.excl_pairs)
            del gp
            torch.cuda.empty_cache()
        elif check_set:
            gp = dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy()
            rep["set"] = check_neighbor_set(gp, pos64, db.box, r_cut + skin, wb.excl_pairs)
        if exceptions is not None:
            dimos.dimos_nl_set_exceptions(ctx, nl, torch.from_numpy(np.ascontiguousarray(exceptions[0], dtype=np.int32)).to(db.pos.device),
                                          torch.from_numpy(np.ascontiguousarray(exceptions[1], dtype=np.float64)).to(db.pos.device))
        F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, method=method, eps_rf=eps_rf, alpha=alpha,
                                        r_switch=r_switch)
        torch.cuda.synchronize()
        orc = oracle.nonbonded(pos64, db.charge.double().cpu().numpy(), wb.type, db.lj_np, db.box, r_cut, method=METHOD[method],
                               eps_rf=eps_rf, alpha=alpha, excl_pairs=wb.excl_pairs, band=BAND, algorithm=oracle_alg,
                               r_switch=r_switch, exceptions=exceptions)
        rep.update(check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision))
        rep["n_pairs_cut"] = orc.n_pairs
        if on_device:
            lo = oracle.count_pairs(pos64, db.box, r_cut - BAND, wb.excl_pairs)
            hi = oracle.count_pairs(pos64, db.box, r_cut + BAND, wb.excl_pairs)
            got = ctx.nl_count_within(nl, r_cut)
            assert lo <= orc.n_pairs <= hi
            assert lo <= got <= hi, f"dimos_nl_count_within(r_cut) = {got}, oracle {orc.n_pairs} (band [{lo}, {hi}])"
            rep["count_within"] = (got, lo, hi)
        return rep
    finally:
        ctx.close()
