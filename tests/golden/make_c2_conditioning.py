"""Writes tests/golden/c2_conditioning.txt: how fast two runs of the CPU ORACLE of config C2
(BASELINE.json configs[1]: 64^3, static droplet R=16, W=4, sigma=0.01, omega=1) drift apart when their
inputs differ by one ulp (relative 2^-52 noise, seeded).  n = G/(|G|+eps) (eq. 21, reading
A7) is not Lipschitz where grad(phi) passes through zero while phi(1-phi) != 0, so ANY two correct
implementations diverge at this rate; tests/test_parity_gpu.py::test_c2_static_droplet_fp64 gates the
GPU against max(1e-12, FACTOR x these numbers).  Calls nothing but oracle/ and the input generators.

    python tests/golden/make_c2_conditioning.py        (~1 min)
"""
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import ref                      # noqa: E402
from paper_2403_15773_b200 import inputs    # noqa: E402

STEPS = (10, 30, 50, 100)


def n2(a, b):
    """per field group, max |a - b| / max |b|."""
    e = {}
    for k in ("rho", "phi"):
        e[k] = np.abs(a[k] - b[k]).max() / np.abs(b[k]).max()
    num = max(np.abs(a[k] - b[k]).max() for k in ("ux", "uy", "uz"))
    e["u"] = num / max(max(np.abs(b[k]).max() for k in ("ux", "uy", "uz")), 1e-300)
    e["pineq"] = np.abs(a["pineq"] - b["pineq"]).max() / max(np.abs(b["pineq"]).max(), 1e-300)
    return e


def main():
    n, R, W, sigma, omega = 64, 16.0, 4.0, 0.01, 1.0
    d = inputs.static_droplet(n, R, W)
    rng = np.random.default_rng(1)
    dp = {k: (None if v is None else v * (1.0 + 2.0 ** -52 * rng.integers(-1, 2, size=v.shape))) for k, v in d.items()}
    runs = []
    for x in (d, dp):
        o = ref.Oracle(n, n, n, omega, two_component=True, sigma=sigma, interface_width=W)
        o.init_fields(x["rho"], x["ux"], x["uy"], x["uz"], x["phi"])
        runs.append(o)
    rows, t = [], 0
    for s in STEPS:
        for o in runs:
            o.step(s - t)
        t = s
        rows.append((s, n2(runs[1].get_moments(), runs[0].get_moments())))
    try:
        rev = subprocess.run(["git", "-C", ROOT, "log", "-1", "--format=%h %cs", "--", "oracle"], capture_output=True,
                             text=True).stdout.strip()
    except Exception:
        rev = "unknown"
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c2_conditioning.txt")
    with open(out, "w") as f:
        f.write("# C2 static droplet (64^3, R=16, W=4, sigma=0.01, omega=1): N2 distance between two CPU-oracle runs\n")
        f.write("# whose inputs differ by seeded one-ulp noise (relative 2^-52), after the given number of steps\n")
        f.write("# written by tests/golden/make_c2_conditioning.py (oracle only); oracle/ at commit %s\n" % rev)
        f.write("# steps rho u pineq phi\n")
        for s, e in rows:
            f.write("%d %.3e %.3e %.3e %.3e\n" % (s, e["rho"], e["u"], e["pineq"], e["phi"]))
    print(open(out).read())


if __name__ == "__main__":
    main()
