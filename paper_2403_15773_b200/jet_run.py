"""Long jet run with the library: the paper's production set-up (Table 1) from rest,
time averages on the mid x-z plane (tslb_stats_*), and the diagnostics the paper reports for them
(Figs. 5-6): inverse centre-line velocity and phase field against z/D, their linear
fits beyond the potential core, and the Gaussian exponent of the radial profile of <u_z> at 12 D.

    python -m paper_2403_15773_b200.jet_run --grid 400 400 800 --D 40 --We 2000 --steps 100000 \
        --avg-from 50000 --out jet_we2000.json

Everything that advances the flow runs in libtslb.so; this file only drives it and post-processes the
two (nz, nx) averages on the host (numpy).  Prints one JSON object (and writes it to --out).
"""
import argparse
import json
import time

import numpy as np

from . import diagnostics, inputs, tslb


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--grid", type=int, nargs=3, default=[400, 400, 800])
    ap.add_argument("--D", type=float, default=40.0)
    ap.add_argument("--U", type=float, default=0.05)
    ap.add_argument("--Re", type=float, default=5000.0)
    ap.add_argument("--We", type=float, default=2000.0)
    ap.add_argument("--steps", type=int, default=100000)
    ap.add_argument("--avg-from", type=int, default=50000)
    ap.add_argument("--every", type=int, default=10, help="sample the averages every this many steps")
    ap.add_argument("--chunk", type=int, default=2000, help="steps between finiteness checks")
    ap.add_argument("--order", type=int, default=3, help="hermite_order (3: eqs. 16/19, 2: eq. 8)")
    ap.add_argument("--forcing", default="kick", choices=["kick", "guo"],
                    help="reading A9 (all kernels) or A18 (Guo-type, generic kernel; include/tslb.h)")
    ap.add_argument("--precision", default="f32")
    ap.add_argument("--perturbation", type=float, default=0.05)
    ap.add_argument("--seed", type=int, default=2024)
    ap.add_argument("--out", default="")
    return ap.parse_args()


linear_fit = diagnostics.linear_fit


def main():
    args = parse()
    import torch
    nx, ny, nz = args.grid
    D, U = args.D, args.U
    prm = inputs.jet_params(nx, ny, nz, D, U=U, Re=args.Re, We=args.We, perturbation=args.perturbation,
                            seed=args.seed)
    kw = {k: v for k, v in prm.items() if k not in ("nx", "ny", "nz", "omega")}
    prec = tslb.F32 if args.precision == "f32" else tslb.F64
    tdt = torch.float32 if prec == tslb.F32 else torch.float64
    dev = torch.device("cuda", 0)
    if args.forcing == "guo":
        kw["forcing"] = tslb.FORCING_GUO
    sim = tslb.Tslb(nx, ny, nz, prm["omega"], precision=prec, hermite_order=args.order, **kw)
    one = torch.ones((nz, ny, nx), dtype=tdt, device=dev)
    zero = torch.zeros((nz, ny, nx), dtype=tdt, device=dev)
    sim.init_fields(one, zero, zero.clone(), zero.clone(), zero.clone())
    del one, zero
    out = {"grid": [nx, ny, nz], "D": D, "U": U, "Re": args.Re, "We": args.We, "omega": prm["omega"],
           "sigma": prm["sigma"], "hermite_order": args.order, "forcing": args.forcing, "precision": args.precision,
           "kernel": sim.kernel_name, "steps": args.steps, "avg_from": args.avg_from, "every": args.every}
    t0 = time.time()
    done, blew_up = 0, None
    history = []
    while done < args.steps:
        n = min(args.chunk, args.steps - done)
        if done < args.avg_from < done + n:
            n = args.avg_from - done
        if done == args.avg_from:
            sim.stats_begin(args.every)
        sim.step(n)
        done += n
        m = sim.get_moments(device=True, want=("uz", "phi"))
        finite = bool(torch.isfinite(m["uz"]).all().item())
        umax = float(m["uz"].abs().max().item()) if finite else float("nan")
        axis = m["phi"][:, ny // 2 - 1:ny // 2 + 1, nx // 2 - 1:nx // 2 + 1].mean(dim=(1, 2))
        below = (axis < 0.5).nonzero()
        tip = int(below[0].item()) if below.numel() else nz
        if done % (10 * args.chunk) == 0 or not finite:
            history.append({"step": done, "max_uz": umax, "axis_phi_first_below_half": tip})
        del m
        if not finite or umax > 0.4:          # Mach ~ 0.7: the run has left the method's range
            blew_up = done
            break
    torch.cuda.synchronize()
    out["wall_s"] = time.time() - t0
    out["glups_incl_checks"] = nx * ny * nz * done / out["wall_s"] / 1e9
    out["steps_done"] = done
    out["blew_up_at_step"] = blew_up
    out["history"] = history
    if blew_up is None:
        m = sim.get_moments(device=True, want=("rho", "phi"))
        out["rho_range"] = [float(m["rho"].min()), float(m["rho"].max())]
        out["phi_range"] = [float(m["phi"].min()), float(m["phi"].max())]
        del m
        st = sim.stats_get()
        out["nsamples"] = st["nsamples"]
        if st["nsamples"] > 0:
            zD = np.arange(nz) / D
            uc = diagnostics.centerline(st["uz"]) / U
            pc = diagnostics.centerline(st["phi"])
            sub = slice(0, nz, max(1, nz // 100))
            out["z_over_D"] = zD[sub].tolist()
            out["uc_over_U"] = uc[sub].tolist()
            out["phi_c"] = pc[sub].tolist()
            # U/<u_c> grows linearly beyond the potential core, slope ~ 1/6.5 per D
            lo, hi = 8.0, min(16.0, 0.8 * nz / D)
            sel = (zD >= lo) & (zD <= hi) & (uc > 1e-6)
            if sel.sum() > 8:
                s, i0, rms = linear_fit(zD[sel], 1.0 / uc[sel])
                out["inv_uc_fit"] = {"range_z_over_D": [lo, hi], "slope_per_D": s, "intercept": i0, "rms": rms,
                                     "paper_slope_per_D": 1.0 / 6.5, "virtual_origin_z0_over_D": -i0 / s if s else None}
                sel2 = sel & (pc > 1e-6)
                if sel2.sum() > 8:
                    s2, i2, rms2 = linear_fit(zD[sel2], 1.0 / pc[sel2])
                    out["inv_phic_fit"] = {"range_z_over_D": [lo, hi], "slope_per_D": s2, "intercept": i2, "rms": rms2}
                # <u_z>(r)/<u_c> at z = 12 D falls on exp(-K (r/(z - z0))^2), K = 75
                z12 = int(round(12 * D))
                if z12 < nz and s > 0:
                    z0 = -i0 / s * D
                    r, q = diagnostics.radial_profile(st["uz"], z12)
                    K = diagnostics.gaussian_exponent(r, q, z12 - z0)
                    if K is not None:
                        out["gaussian_K_at_12D"] = {"K": K, "paper_K": 75.0, "z0": z0}
                    r, q = diagnostics.radial_profile(st["phi"], z12)
                    Kp = diagnostics.gaussian_exponent(r, q, z12 - z0)
                    if Kp is not None:
                        out["gaussian_Kint_phi_at_12D"] = {"K": Kp, "paper_K_We2000": 80.0}
    sim.close()
    s = json.dumps(out)
    print(s)
    if args.out:
        with open(args.out, "w") as f:
            f.write(s + "\n")


if __name__ == "__main__":
    main()
