"""Writes tests/golden/sp3_oracle_energies.txt: reduced energies E / (Km V) of the relaxed twisted-flower
and vortex states of standard problem 3 (script L930-L955) at edge lengths 8.44 and
8.50 exchange lengths, computed by the fp64 oracle alone (about 25 minutes on one core; too slow for the
test suite, hence stored). Calls only oracle/ and synth/.

    python tests/golden/make_sp3_oracle.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import RefSim          # noqa: E402
from synth import Params           # noqa: E402

N, MS, A = 16, 500e3, 20e-12
KM = 0.5 * 4e-7 * np.pi * MS * MS
LEX = np.sqrt(A / KM)


def start(kind):
    z, y, x = np.meshgrid(*(np.arange(N) - 7.5,) * 3, indexing="ij")
    v = np.zeros((3, N, N, N))
    if kind == "twisted":                       # swirl about the easy axis: relaxes to the twisted flower
        r = np.sqrt(x * x + y * y) + 1e-9
        v[0] = -y / r; v[1] = x / r; v[2] = np.exp(-(r / 3) ** 2) + 0.2
    else:                                        # vortex with its core perpendicular to the easy axis
        r = np.sqrt(z * z + y * y) + 1e-9
        v[1] = -z / r; v[2] = y / r; v[0] = np.exp(-(r / 3) ** 2) + 0.2
    return v


def main():
    lines = ["# written by tests/golden/make_sp3_oracle.py (oracle only): L  state  E/(Km V)  <mx> <my> <mz>"]
    for L in (8.44, 8.50):
        c = L * LEX / N
        for kind in ("twisted", "vortex"):
            sim = RefSim((N, N, N), (c, c, c), demag_method="fft")
            sim.set_params(Params.uniform(1, Msat=MS, Aex=A, alpha=0.5, Ku1=0.1 * KM, anisU=(0, 0, 1)))
            sim.set_m(start(kind))
            sim.relax()
            e = sim.energy() / (KM * (c * N) ** 3)
            a = sim.avg_m()
            lines.append("%.2f %s %.10f %.6f %.6f %.6f" % (L, kind, e, a[0], a[1], a[2]))
            print(lines[-1], flush=True)
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "sp3_oracle_energies.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
