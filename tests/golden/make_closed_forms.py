"""Writes tests/golden/closed_forms.json from formulas only (no simulation, no CUDA).

Formulas (SURVEY.md 8c "pins"; kinetic theory of SRD, refs [27-29] of the paper,
PAPER.md:23 -- the paper prints only the resulting viscosity 8.7):

  one-step decorrelation, i.i.d. velocities, Poisson occupancy (P0 = exp(-M)):
    SRD: <v.v'>/<v.v> = 1 - (2/3)(1 - cos a)(M - 1 + P0)/M
    AT : <v.v'>/<v.v> = (1 - P0)/M
  nu_col = a^2/(18 dt) (1 - cos a)(M - 1 + e^-M)/M
  nu_kin = (kT dt / 2m) [5M / ((M - 1 + e^-M)(2 - cos a - cos 2a)) - 1]
  D      = (kT dt / 2m) [3M / ((1 - cos a)(M - 1 + e^-M)) - 1]
"""
import json
import math
import os


def forms(M, alpha_deg, dt, kT=1.0, m=1.0, a=1.0):
    al = math.radians(alpha_deg)
    c, c2 = math.cos(al), math.cos(2 * al)
    P0 = math.exp(-M)
    g = M - 1 + P0
    return {
        "M": M, "alpha_deg": alpha_deg, "dt": dt,
        "srd_decorrelation": 1 - (2.0 / 3.0) * (1 - c) * g / M,
        "at_decorrelation": (1 - P0) / M,
        "nu_col": a * a / (18 * dt) * (1 - c) * g / M,
        "nu_kin": kT * dt / (2 * m) * (5 * M / (g * (2 - c - c2)) - 1),
        "D": kT * dt / (2 * m) * (3 * M / ((1 - c) * g) - 1),
    }


if __name__ == "__main__":
    out = {"_cite": __doc__, "cases": [forms(10, 130, 0.1), forms(5, 130, 0.1), forms(10, 130, 1.0), forms(5, 130, 1.0)]}
    for case in out["cases"]:
        case["nu"] = case["nu_col"] + case["nu_kin"]
        case["eta"] = case["M"] * case["nu"]
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_forms.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out["cases"], indent=1))
