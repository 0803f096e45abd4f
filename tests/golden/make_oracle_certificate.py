"""Writes tests/golden/oracle_certificate.json from long runs of the CPU oracle ONLY.

Run:  python tests/golden/make_oracle_certificate.py          (about 15 minutes on one core)

Stored values are the oracle's own measurements of quantities the paper fixes (contact angle on
a cylinder, §III.B; Laplace law).  Nothing here calls the CUDA path.
"""
import json
import math
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
sys.path.insert(0, os.path.dirname(HERE))

import numpy as np  # noqa: E402

import _measure as ms  # noqa: E402
from oracle import ref  # noqa: E402
from paper_2605_30878_b200 import workloads as wl  # noqa: E402


def main():
    cert = {"source": "oracle/lbmref.c via tests/golden/make_oracle_certificate.py",
            "contact_angle": [], "laplace": []}
    # config 2 geometry at half scale (128^2, R = 20, drop 17.5, W = 5), 20,000 steps; at 30 deg the
    # cap is so flat that no contour point lies farther than 2W from the solid at that scale, so
    # that angle runs at full scale (256^2, R = 40)
    for theta, n in ((30.0, 256), (60.0, 128), (90.0, 128), (120.0, 128), (150.0, 128)):
        w = wl.config2(seed=0, theta_deg=theta, n=n)
        s = ref.RefLBM(ref.RefParams(**w.param_dict()), w.mask, w.disks)
        s.init(w.phi0)
        m0 = s.diag()["sum_phi"]
        s.step(20000)
        g, d = s.get(), s.diag()
        th, Rc, dist, hmax = ms.contact_angle_on_cylinder(g["phi"], w.mask, w.disks[0], w.W)
        R = w.disks[0][2]
        area = math.pi * Rc * Rc - ms.lens_area(R, Rc, dist)
        h_an = ms.analytic_drop_on_cylinder(R, area, theta)[2]
        cert["contact_angle"].append(dict(
            workload=w.name, steps=20000, theta_set=theta, theta_measured=th, tol_deg=4.0,
            hmax_over_R=hmax / R, hmax_over_R_analytic=h_an / R, umax=d["umax"],
            mass_drift_rel=(d["sum_phi"] - m0) / m0))
        print(cert["contact_angle"][-1], flush=True)
    for n, R in ((96, 24.0),):
        mask, disks, phi0 = wl.free_droplet(n, R, 4.0)
        prm = ref.RefParams(nx=n, ny=n, rho_l=1.0, rho_g=1.0, nu_l=1 / 6, nu_g=1 / 6, sigma=0.01, W=4.0)
        s = ref.RefLBM(prm, mask, disks); s.init(phi0); s.step(6000)
        g, d = s.get(), s.diag()
        ph = g["rho"] * g["p"]
        ratio = (ph[n // 2, n // 2] - ph[2, 2]) / (0.01 / math.sqrt(d["sum_phi"] / math.pi))
        cert["laplace"].append(dict(n=n, R=R, W=4.0, steps=6000, ratio=ratio, tol=0.03, umax=d["umax"]))
        print(cert["laplace"][-1], flush=True)
    with open(os.path.join(HERE, "oracle_certificate.json"), "w") as f:
        json.dump(cert, f, indent=1)


if __name__ == "__main__":
    main()
