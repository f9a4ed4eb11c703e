"""Writes tests/golden/laplace_c2_oracle.txt: the Young-Laplace pressure jump of config C2
(BASELINE.json configs[1]) as computed by the CPU ORACLE ONLY (calls nothing but
oracle/ and the input generators).  ~8 min on 8 cores.

    python tests/golden/make_laplace_c2.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import ref                      # noqa: E402
from paper_2403_15773_b200 import inputs    # noqa: E402

n, R, W, sigma, omega, steps, navg = 64, 16.0, 4.0, 0.01, 1.0, 2000, 222
d = inputs.static_droplet(n, R, W)
o = ref.Oracle(n, n, n, omega, two_component=True, sigma=sigma, interface_width=W)
o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
x, y, z = inputs.grid(n, n, n)
c = (n - 1) / 2
r = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
inside, outside = r < R / 2, r > R + (n / 2 - R) / 2
o.step(steps - navg)
dps = []
for _ in range(navg):
    o.step(1)
    m = o.get_moments()
    dps.append((m["rho"][inside].mean() - m["rho"][outside].mean()) / 3.0)
dp = float(np.mean(dps))
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "laplace_c2_oracle.txt")
with open(out, "w") as f:
    f.write("# C2 static droplet, 64^3, R=16, W=4, sigma=0.01, omega=1, rho0=1, u0=0; CPU oracle fp64\n")
    f.write("# dp = c_s^2 (<rho>_{r<R/2} - <rho>_{r>R+(n/2-R)/2}) averaged over steps 1779..2000\n")
    f.write("# written by tests/golden/make_laplace_c2.py (oracle only); 2 sigma / R = 1.25e-3\n")
    f.write("dp_mean %.17g\n" % dp)
    f.write("dp_over_2sigmaR %.17g\n" % (dp / (2 * sigma / R)))
    f.write("dp_min %.17g\ndp_max %.17g\n" % (min(dps), max(dps)))
    f.write("max_abs_u %.17g\n" % max(np.abs(m[k]).max() for k in ("ux", "uy", "uz")))
    f.write("phi_sum_drift %.17g\n" % (m["phi"].sum() - d["phi"].sum()))
    f.write("mass_drift %.17g\n" % (m["rho"].sum() - d["rho"].sum()))
print(open(out).read())
