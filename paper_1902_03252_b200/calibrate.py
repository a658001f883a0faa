"""Empirical calibration of the paper's mixed-precision rule for a given catalogue.

The paper derives its rule for the SIE analytically (Appendix A): an SP error bound E_SP = 2.3e-3" outside DP
centre patches of 400 x 400 / 20 x 20 pixels, hence SP suffices where the magnification along an axis is
M_i <= (dx/4)/E_SP = 3.26, and says that for other models the SP-safe fraction "has to be computed for each
model independently".  This tool does that computation by measurement, for BOTH single precision versions:
  * "plain":       the paper's own SP version, "identical up to the change in precision" -- pixel coordinates,
                   lens centres and their difference in fp32 (lt_set_tuning, single_launch bit 4);
  * "tile_centre": the product's fp32 mode, which forms the lens-frame position of each tile centre
                   in fp64 and adds the in-tile offset in fp32.
For each it runs the mixed mode (fp32 pass, rule) and the fp64 mode through the C ABI and hands the maps to
lt_rule_audit, which evaluates on the device
  * the SP error |fp32 - fp64| (arcsec): overall, inside / outside the rule's centre patches, and against the distance to
    the nearest lens centre (pixels) -- the table form of Fig. 9: the plain version shows the growth towards the
    centres that the patches exist for ((A.65)), the tile-centre version shows what is left of it;
  * the magnification bound M_max = (dx/4)/E_SP the measured error implies (the paper's 3.26);
  * the pixels that violate the paper's criterion |err_i| <= dx/(4 M_i) (M_i from the fp64 map, eq. 24-26) and
    how many of them the rule flags / misses;
and the same for a calibrated rule (M_max = half the implied value, c28 = (1 - 1/M_max)/2 -- the relation of the paper's
own 0.0104 and 0.0092 -- and minimal patches).

    python -m paper_1902_03252_b200.calibrate --config 2 [--paper-regime] [--model sie|nfw]

Marshalling only: every map and every number comes from the CUDA library (checked against oracle/calibrate_ref.py by
tests/test_gpu_audit.py).  Needs a GPU.
"""
import argparse
import json

PLAIN_SP = 16          # lt_set_tuning: single_launch bit 4


def _scheme(lt, torch, W, model, mixed, plain):
    grid = {"sie": lt.lt_gradient_grid_sie, "nfw": lt.lt_gradient_grid_nfw}.get(model, lt.lt_gradient_grid)
    scale_col = {"sie": 4, "nfw": None}.get(model, 6)
    L = torch.from_numpy(W.lenses).cuda()
    centres = torch.zeros((len(W.lenses), 3), dtype=torch.float64, device="cuda")
    centres[:, :2] = L[:, :2]
    if scale_col is not None:
        centres[:, 2] = L[:, scale_col]
    n = len(W.lenses)
    g64 = grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, lt.LT_FP64)
    ws = lt.alloc_workspace(n, W.nx, W.ny, lt.LT_MIXED)
    lt.lt_set_tuning(single_launch=PLAIN_SP if plain else 0)
    try:
        def audit(params):
            grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, lt.LT_MIXED, mixed=params, workspace=ws)
            sp = lt.lt_mixed_last_sp_map(ws, n, W.nx, W.ny)
            flags = lt.lt_mixed_last_flags(ws, n, W.nx, W.ny)
            d_res, _ = lt.lt_rule_audit(sp, g64, W.x_min, W.y_min, W.dx, centres=centres, flags=flags)
            return lt.lt_rule_audit_result(d_res, W.dx)
        r = audit(mixed)
        n_pix = r["n_pixels"]
        edges = list(lt.AUDIT_BIN_EDGES_PX) + ["inf"]
        out = {"sp_error_arcsec": {"max": r["max_err"], "max_inside_default_patches": r["max_err_in_patch"],
                                   "max_outside_default_patches": r["max_err_outside_patch"]},
               "max_sp_error_by_distance_px": {"%s-%s" % (lo, hi): v for lo, hi, v in
                                               zip(edges[:-1], edges[1:], r["max_err_by_distance"])},
               "implied_m_max_no_patches": r["implied_m_max"],
               "implied_m_max_outside_default_patches": r["implied_m_max_outside_patch"],
               "criterion": {"pixels_violating": r["n_violating"], "fraction_violating": r["n_violating"] / n_pix,
                             "violating_and_flagged_by_rule": r["n_violating_flagged"],
                             "violating_and_missed_by_rule": r["n_violating_missed"],
                             "flagged_fraction": r["n_flagged"] / n_pix}}
        # the calibrated rule: M_max from the measured SP error with a safety factor of 2, eq. 28's constant re-derived the
        # way the paper's own numbers are related (0.0104 = (0.03 - 0.0092)/2, i.e. c28 = (1 - 1/M_max)/2), minimal patches
        m_cal = max(1.5, 0.5 * r["implied_m_max"])
        cal = (m_cal, 0.5 * (1.0 - 1.0 / m_cal), 0.0, 0.0, 1e300)
        rc = audit(cal)
        out["calibrated_rule"] = {"m_max": m_cal, "c28": cal[1], "patch_halfwidths": [0.0, 0.0],
                                  "flagged_fraction": rc["n_flagged"] / n_pix,
                                  "violating_and_missed": rc["n_violating_missed"]}
    finally:
        lt.lt_set_tuning()
    return out


def calibrate(W, model="dpie", mixed=None):
    import torch
    from . import lt
    return {"workload": W.name, "dx": W.dx,
            "plain": _scheme(lt, torch, W, model, mixed, True),
            "tile_centre": _scheme(lt, torch, W, model, mixed, False)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--paper-regime", action="store_true")
    ap.add_argument("--model", default="dpie", choices=["dpie", "sie", "nfw"])
    args = ap.parse_args()
    from . import workloads
    if args.model == "sie":
        W, mixed = workloads.make_sie("paper"), (3.26, 0.0104 / 0.03, 6.0, 0.3, 1.0)
    elif args.model == "nfw":
        W, mixed = workloads.make_nfw(n_override=2048), None
    else:
        W, mixed = workloads.make(args.config, paper_regime=args.paper_regime), None
    print(json.dumps(calibrate(W, args.model, mixed)))


if __name__ == "__main__":
    main()
