"""Writes tests/golden/laplace_config1.txt by running ONLY the CPU oracle.

Config 1 of BASELINE.json (32^3 periodic, D3Q15+D3Q19, heavy droplet R=8, rho_H=1,
rho_L=1e-3, xi=5, sigma=1e-4, M=0.02, nu=1/60) run for 10 000 steps; records
dp/(2 sigma/R) with dp = p(centre cell) - p(corner cell), R the nominal radius, and the
sum(phi) drift.  Laplace's law (north_star; sigma enters via beta, kappa P:139) asks for
dp = 2 sigma / R within 3 % once the acoustic ringing has decayed (>= 8000 steps).

Usage: python tests/golden/make_laplace.py      (about half an hour on 8 cores)
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import Oracle  # noqa: E402
from paper_2012_06144_b200 import inputs  # noqa: E402

STEPS = [100, 500, 1000, 2000, 4000, 6000, 8000, 9000, 10000]


def main():
    p, phi, u = inputs.config1()
    R = 8.0
    o = Oracle.from_params(p)
    o.init(phi, u)
    m0 = o.phi_mass()
    lines = ["# config 1 (32^3, R=8): step  dp/(2 sigma/R)  (sum(phi)-m0)/m0  max|u|   -- written by make_laplace.py (oracle only)"]
    done = 0
    for s in STEPS:
        o.step(s - done)
        done = s
        ph, uu, pr = o.fields()
        c = p.nx // 2
        dp = pr[c, c, c] - pr[0, 0, 0]
        lines.append(f"{s} {dp / (2 * p.sigma / R):.15e} {(o.phi_mass() - m0) / m0:.3e} {abs(uu).max():.6e}")
        print(lines[-1], flush=True)
        with open(os.path.join(HERE, "laplace_config1.txt"), "w") as f:
            f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
