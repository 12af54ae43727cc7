"""Writes tests/golden/kinetic_spectrum_cfg0.txt from the ORACLE only (never from the CUDA path):
lowest eigenvalues and the largest one of 1/2 M_D^{-1/2} K M_D^{-1/2} on the config-0 mesh."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as O  # noqa: E402


def main():
    ref = O.RefCtx((3, 3, 3), (6.0, 6.0, 6.0), 3, (0, 0, 0))
    ref.set_potential(np.zeros(ref.M), None)
    H = ref.dense_H()
    lam = np.linalg.eigvalsh(H[0::2, 0::2].real)          # spin-up block = the scalar kinetic operator
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "kinetic_spectrum_cfg0.txt"), "w") as f:
        f.write("# eigenvalues of 1/2 M_D^{-1/2} K M_D^{-1/2}, 3x3x3 cells of order 3, box 6 bohr, periodic (oracle; SURVEY.md 9)\n")
        f.write("# index value   (plane-wave reference for levels 1..6: 0.5*(2*pi/6)**2 = %.9f)\n" % (0.5 * (2 * np.pi / 6) ** 2))
        for i in list(range(8)) + [len(lam) - 1]:
            f.write("%d %.9f\n" % (i, lam[i]))


if __name__ == "__main__":
    main()
