"""Parity statistics between the oracle's maps and the maps of the implementation under test (TEST INFRASTRUCTURE).

Pure numpy, no method arithmetic: it only compares.  The gates are BASELINE.json's (north_star):
  - winning plane index equal on >= 99.9 % of the oracle-valid pixels, a differing index counting as equal only when
    it is a floating-point tie in the ORACLE's own cost vector: c_oracle[k_test] - c_oracle[k*] <= tie_tol (2e-4);
  - best cost within 1e-4 absolute;
  - refined depth within 1e-3 relative wherever the indices are equal;
  - validity bit-exact away from ties (pixels the oracle marks fragile: a geometric or threshold margin below its
    epsilon, or an argmin tie).
"""
from __future__ import annotations

import numpy as np

TIE_TOL = 2e-4
COST_TOL = 1e-4
DEPTH_RTOL = 1e-3


def depth_conditioning(orc: dict, plane_s, pden=None, kbest=None) -> np.ndarray:
    """(|ds|/s) / pden per pixel: how strongly an error of the three costs around the minimum moves the refined
    depth.  With |error| <= eps on each cost, |d delta| <= 3 eps / pden, and d depth / depth = d delta * |ds| / s
    ("Tolerances").  inf where the parabola was not applied is replaced by 0 (no refinement -> no
    sensitivity)."""
    k = (orc["kbest"] if kbest is None else kbest).astype(np.int64)
    pd = orc["pden"] if pden is None else pden
    plane_s = np.asarray(plane_s, dtype=np.float64)
    ks = np.clip(k & 0x3FFF, 0, len(plane_s) - 1)
    kn = np.clip(ks + 1, 0, len(plane_s) - 1)
    ds = np.abs(plane_s[kn] - plane_s[ks])
    s = plane_s[ks]
    with np.errstate(divide="ignore", invalid="ignore"):
        cond = np.where(pd > 0, (ds / s) / pd, 0.0)
    return np.where(k >= 0, cond, 0.0)


def compare_maps(orc: dict, test: dict, cost_volumes=None, index_flag_mask: int = 0x3FFF, depth_cond=None) -> dict:
    """orc: dict from oracle.compute_depth / compute_depth_multires (float64 maps, 'reason', 'kbest', 'c2raw' ...).
    test: dict of numpy arrays depth, best_cost, second_cost, plane_index, valid_reason.
    cost_volumes: oracle cost volume [P,H,W] (single pass), or a pair (cost_lo at half resolution, cost_hi) for the
    multi-resolution call, used for the oracle-side tie rule; None = exact equality only."""
    o_valid = orc["reason"] == 0
    t_valid = np.asarray(test["valid_reason"]) == 0
    o_raw = orc["raw_valid"] != 0
    t_k_full = np.asarray(test["plane_index"]).astype(np.int64)
    t_raw = t_k_full >= 0
    o_k_full = orc["kbest"].astype(np.int64)
    o_k = np.where(o_k_full >= 0, o_k_full & index_flag_mask, -1)
    t_k = np.where(t_k_full >= 0, t_k_full & index_flag_mask, -1)
    same_source = (o_k_full >> 14) == (t_k_full >> 14)

    # fragility: geometry, thresholds, argmin ties
    fragile = (orc.get("fragile_geom", np.zeros_like(o_valid, dtype=np.uint8)) != 0)
    fragile |= (orc.get("fragile_thr", np.zeros_like(o_valid, dtype=np.uint8)) != 0)
    c2raw = orc.get("c2raw")
    tie = np.zeros_like(o_valid)
    if c2raw is not None:
        with np.errstate(invalid="ignore"):
            tie = o_raw & (np.abs(orc["c1"] - c2raw) < TIE_TOL)
    # a tie excuses the validity of a pixel only where the test really took another plane than the oracle
    tie_excuse = tie & (o_k != t_k)
    fragile_all = fragile | tie_excuse

    both = o_valid & t_raw
    n_valid = int(o_valid.sum())
    exact = both & (o_k == t_k) & same_source
    matched = exact.copy()
    if cost_volumes is not None:
        diff = both & ~exact
        ys, xs = np.nonzero(diff)
        if ys.size:
            if isinstance(cost_volumes, (tuple, list)):
                cost_lo, cost_hi = cost_volumes
                ok = np.zeros(ys.size, dtype=bool)
                for n, (y, x) in enumerate(zip(ys, xs)):
                    if not same_source[y, x]:
                        continue
                    vol, yy, xx = (cost_hi, y, x) if (o_k_full[y, x] >> 14) else (cost_lo, y >> 1, x >> 1)
                    kt, ko = t_k[y, x], o_k[y, x]
                    if 0 <= kt < vol.shape[0]:
                        ok[n] = vol[kt, yy, xx] - vol[ko, yy, xx] <= TIE_TOL
            else:
                vol = cost_volumes
                kt = np.clip(t_k[ys, xs], 0, vol.shape[0] - 1)
                ok = (vol[kt, ys, xs] - vol[o_k[ys, xs], ys, xs] <= TIE_TOL) & same_source[ys, xs]
            matched[ys[ok], xs[ok]] = True

    with np.errstate(invalid="ignore", divide="ignore"):
        dc1 = np.abs(np.asarray(test["best_cost"], dtype=np.float64) - orc["c1"])
        dc2 = np.abs(np.asarray(test["second_cost"], dtype=np.float64) - orc["c2"])
        # relative to |depth|: with FSW_DEPTH_Z (range * r_z, reading Q16) the depth of a ray more than 90 degrees off
        # the axis is negative; validity is the reason code, not the sign
        ddepth = np.abs(np.asarray(test["depth"], dtype=np.float64) - orc["depth"]) / np.maximum(np.abs(orc["depth"]), 1e-30)
    cost_set = o_raw & t_raw & (o_k == t_k) & same_source
    depth_set = o_valid & t_valid & (o_k == t_k) & same_source
    max_dc1 = float(dc1[cost_set].max()) if cost_set.any() else 0.0
    eps_run = min(COST_TOL, max(1.5 * max_dc1, 2e-5))   # the cost error this run shows, not the 1e-4 it is allowed
    if depth_cond is not None:
        # the bound assumes that the three costs around the minimum carry the run's cost error; on a geometrically
        # fragile pixel (a window sample within its margin of a view border) a NEIGHBOUR plane may be a mean over
        # another set of views in one of the two implementations (the same exclusion as for the second best below),
        # so those pixels only count toward the plain 1e-3 share
        geom = (orc.get("fragile_geom", np.zeros_like(o_valid, dtype=np.uint8)) != 0)
        allowed = DEPTH_RTOL + 3.0 * eps_run * depth_cond
        cond_set = depth_set & ~geom
        depth_cond_viol = int((ddepth[cond_set] > allowed[cond_set]).sum())
        worst_ratio = float((ddepth[cond_set] / allowed[cond_set]).max()) if cond_set.any() else 0.0
    else:
        depth_cond_viol, worst_ratio = -1, -1.0
    raw_mismatch = (o_raw != t_raw)
    valid_mismatch = (o_valid != t_valid)
    stats = dict(
        n_pixels=int(o_valid.size),
        n_oracle_valid=n_valid,
        n_oracle_raw_valid=int(o_raw.sum()),
        n_test_valid=int(t_valid.sum()),
        index_exact_frac=float(exact.sum()) / max(n_valid, 1),
        index_match_frac=float(matched.sum()) / max(n_valid, 1),
        max_dc1=max_dc1,
        p999_dc1=float(np.quantile(dc1[cost_set], 0.999)) if cost_set.any() else 0.0,
        frac_dc1_over_tol=float((dc1[cost_set] > COST_TOL).mean()) if cost_set.any() else 0.0,
        # equal index => same candidate planes for c2, unless the finiteness of one of them is itself fragile (a
        # window sample on a border: the plane then averages over another set of views in one of the two)
        max_dc2=float(dc2[cost_set & ~fragile].max()) if (cost_set & ~fragile).any() else 0.0,
        max_dc2_all=float(dc2[cost_set].max()) if cost_set.any() else 0.0,
        frac_dc2_over_tol=float((dc2[cost_set & ~fragile] > COST_TOL).mean()) if (cost_set & ~fragile).any() else 0.0,
        max_ddepth_rel=float(ddepth[depth_set].max()) if depth_set.any() else 0.0,
        frac_ddepth_over_tol=float((ddepth[depth_set] > DEPTH_RTOL).mean()) if depth_set.any() else 0.0,
        depth_violations_conditioned=depth_cond_viol,
        depth_worst_ratio_to_bound=worst_ratio,
        depth_bound_cost_eps=eps_run,
        fragile_frac=float(fragile_all.mean()),
        fragile_frac_of_raw=float((fragile_all & o_raw).sum()) / max(int(o_raw.sum()), 1),
        tie_frac_of_raw=float(tie.sum()) / max(int(o_raw.sum()), 1),
        raw_valid_mismatch_nonfragile=int((raw_mismatch & ~(fragile)).sum()),
        valid_mismatch_nonfragile=int((valid_mismatch & ~fragile_all).sum()),
        valid_mismatch_total=int(valid_mismatch.sum()),
    )
    return stats


def to_numpy(out: dict) -> dict:
    """torch tensors (any device) -> numpy arrays, dropping private keys."""
    res = {}
    for k, v in out.items():
        if k.startswith("_"):
            continue
        res[k] = v.detach().cpu().numpy() if hasattr(v, "detach") else np.asarray(v)
    return res
