"""The paper's physical application (section 5): decaying 2.5-D relativistic MHD turbulence on an n x n
grid, run with the full scheme (UCT=HO=YES) to t = 20 in the paper's units (box side 2 pi; the unit box used here
makes one paper time unit 1/(2 pi)), with the isotropised spectra of Fig. 5 at the end.

    python -m paper_2401_03008_b200.turb2d --n 4096 --t 20 --out gpurun_out/turb2d_4096

Everything on the time-stepping path is the CUDA library (binding.Echo); this module only drives it and
post-processes the final state (spectra.py).  Writes <out>.json (history of the rms fluctuations, spectra in
logarithmic bins, fitted slopes, wall-clock time) and prints a short summary.
"""
import argparse
import json
import math
import time


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--n", type=int, default=1024)
    ap.add_argument("--t", type=float, default=20.0, help="final time in the paper's units (L = 2 pi)")
    ap.add_argument("--samples", type=int, default=40, help="history samples between 0 and t")
    ap.add_argument("--seed", type=int, default=2401)
    ap.add_argument("--out", default="turb2d")
    ap.add_argument("--fit", type=int, nargs=2, default=None, help="shell range of the slope fit (default 8 .. n/32)")
    args = ap.parse_args(argv)

    import numpy as np
    import torch
    from . import binding, inputs, spectra

    n = args.n
    w = inputs.turbulence_2d(n, seed=args.seed)
    e = binding.Echo(n, n, 1, w["gamma"], 0.3)
    faces = e.faces_from_potential(*[torch.as_tensor(w[k], device="cuda") for k in ("ax", "ay", "az")], w["b0"])
    e.set_primitives(*[torch.as_tensor(w[k], device="cuda") for k in ("rho", "vx", "vy", "vz", "p")], *faces)
    del faces

    def sample():
        q = e.get_primitives()
        d = e.diagnostics()
        vperp = torch.sqrt(q["vx"] ** 2 + q["vy"] ** 2)
        bperp = torch.sqrt(q["bx"] ** 2 + q["by"] ** 2)
        rec = {"t": d["t"] * 2.0 * math.pi, "steps": int(d["steps"]),
               "rms_v_perp_over_vA": float(torch.sqrt((vperp ** 2).mean())) / w["vA"],
               "rms_b_perp_over_B0": float(torch.sqrt((bperp ** 2).mean())) / w["B0"],
               "mean_v_perp_over_vA": float(vperp.mean()) / w["vA"],
               "mean_b_perp_over_B0": float(bperp.mean()) / w["B0"],
               "max_W": d["max_W"], "min_rho": d["min_rho"], "min_p": d["min_p"], "max_div_b": d["max_div_b"],
               "c2p_failures": d["c2p_failures"], "c2p_max_iters": d["c2p_max_iters"],
               "sum_U": d["sum_U"], "sum_D": d["sum_D"]}
        return q, rec

    t_end = args.t / (2.0 * math.pi)
    hist = [sample()[1]]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for s in range(1, args.samples + 1):
        try:
            e.run_until(t_end * s / args.samples)      # echo_run_until: chunks sized from a_max, stops on t_end
        except binding.EchoError as err:
            if err.code != binding.ECHO_EC2P:
                raise
        q, rec = sample()
        hist.append(rec)
        if rec["c2p_failures"] or not math.isfinite(rec["max_W"]):
            break
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    steps = hist[-1]["steps"]

    spec = {"v_perp": spectra.spectrum_of_vector(q["vx"], q["vy"]), "b_perp": spectra.spectrum_of_vector(q["bx"], q["by"]),
            "v_z": spectra.isotropic_spectrum_2d(q["vz"]), "b_z": spectra.isotropic_spectrum_2d(q["bz"] - q["bz"].mean())}
    lo, hi = args.fit if args.fit else (8, max(16, n // 32))
    slopes = {k: spectra.fit_slope(v, lo, hi) for k, v in spec.items()}
    out = {"n": n, "t_final_paper_units": hist[-1]["t"], "steps": steps, "wall_seconds": wall,
           "cell_updates_per_s": n * n * steps / wall, "seconds_per_paper_time_unit": wall / max(hist[-1]["t"], 1e-30),
           "fit_shells": [lo, hi], "slopes": slopes, "history": hist,
           "spectra_log_bins": {k: spectra.log_bins(v) for k, v in spec.items()},
           "scheme": "MP5+HLL+UCT+DER6/INT6+SSPRK3 (UCT=HO=YES)", "seed": args.seed}
    with open(args.out + ".json", "w") as fh:
        json.dump(out, fh, indent=1)
    print(json.dumps({k: out[k] for k in ("n", "t_final_paper_units", "steps", "wall_seconds", "cell_updates_per_s",
                                          "seconds_per_paper_time_unit", "fit_shells", "slopes")}))
    last = hist[-1]
    print("final: rms dv/vA %.4f  rms dB/B0 %.4f  max W %.4f  min rho %.4f  min p %.3f  max div B %.2e  c2p failures %d"
          % (last["rms_v_perp_over_vA"], last["rms_b_perp_over_B0"], last["max_W"], last["min_rho"], last["min_p"],
             last["max_div_b"], last["c2p_failures"]))
    return 0 if not last["c2p_failures"] else 1


if __name__ == "__main__":
    raise SystemExit(main())
