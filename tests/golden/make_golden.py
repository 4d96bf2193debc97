"""Writes the stored expected values under tests/golden/.  Calls neither the CUDA path nor
(for these closed forms) the oracle: every number is the paper's (cited) or a closed form.

    python tests/golden/make_golden.py
"""
import json
import math
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    # PAPER.md:220 (§4): "liquid and gas densities are 1000 and 1.2 kg/m^3 ... density ratio of 833"
    # 192x192x768 grid, 864 bubbles, d = 2 mm = 8 cells of 0.25 mm,
    # regular 6x6x24 array, void fraction "approximately 0.82 %".
    paper = {
        "_cite": "PAPER.md:199 (grid), PAPER.md:218 (864 bubbles, 6x6x24, void 0.82 %), "
                 "PAPER.md:220 (rho_l, rho_g, ratio 833, d = 2 mm)",
        "rho_l": 1000.0, "rho_g": 1.2, "density_ratio_rounded": 833,
        "grid": [192, 192, 768], "bubbles": 864, "array": [6, 6, 24],
        "diameter_cells": 8, "void_fraction_percent": 0.82,
    }
    with open(os.path.join(HERE, "paper_constants.json"), "w") as f:
        json.dump(paper, f, indent=1)
        f.write("\n")

    # Closed-form eigenvalue of the constant-density operator with Neumann x,y / periodic z
    # (SURVEY.md §8.c P1): lambda = -(1/rho) sum_d (4/h_d^2) sin^2(theta_d),
    # theta = pi kx/(2 nx), pi ky/(2 ny), pi kz/nz.  BASELINE.json configs[1]: 64x64x128, rho = 1000.
    nx, ny, nz, rho, h = 64, 64, 128, 1000.0, 1.0 / 64
    lam = -(1.0 / rho) * (4.0 / h ** 2) * (math.sin(math.pi * 1 / (2 * nx)) ** 2
                                           + math.sin(math.pi * 2 / (2 * ny)) ** 2
                                           + math.sin(math.pi * 3 / nz) ** 2)
    eig = {"_cite": "closed form, SURVEY.md §8.c P1 (operator: PAPER.md:111, BCs PAPER.md:195); "
                    "grid of BASELINE.json configs[1]",
           "nx": nx, "ny": ny, "nz": nz, "rho": rho, "mode": [1, 2, 3], "lambda_1_2_3": lam}
    with open(os.path.join(HERE, "eigenvalue_config2.json"), "w") as f:
        json.dump(eig, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
