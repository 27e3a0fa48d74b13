"""SURROGATE electron form-factor coefficient table (NOT Kirkland's, NOT physical data).

PAPER.md:81 (§2.2 "Atomic Scattering Potentials") says the coefficients {a_i,b_i,c_i,d_i} of
    f(q) = sum_i a_i/(q^2+b_i) + sum_i c_i exp(-d_i q^2)
"are tabulated" (ref. [33]) but prints none, and no third-party table may be transcribed
from memory.  The library takes coefficients through its ABI (`ps_set_form_factors`) in the
general (n_lorentz, n_gauss) form, so any real table can be supplied by a user.  What is
committed here is a clearly-labelled stand-in produced by the seeded recipe below, with
Kirkland-like magnitudes only:

  * sum_i a_i = Z / (2 pi^2 a0)   (the Mott/Rutherford 1/q^2 tail, a0 = 0.529177 Angstrom),
  * f(0) = 1.2 * Z**0.66 Angstrom  (right order of magnitude for light/medium elements),
  * half of f(0) carried by the Lorentzians, half by the Gaussians,
  * b_i, d_i log-uniform over the ranges such tables span.

Two kinds: "kirkland33" -> (n_lorentz, n_gauss) = (3, 3)   [configs 2-5]
           "gauss5"     -> (0, 5)                           [config 1, "5-Gaussian"]
q is |k| in 1/Angstrom (k = m/L, no 2 pi).

Run `python -m workloads.form_factors` to rewrite `surrogate_form_factors.json`.
"""
from __future__ import annotations

import json
import os

import numpy as np

_TABLE_PATH = os.path.join(os.path.dirname(__file__), "surrogate_form_factors.json")
_SEED = 260210064
ELEMENTS = (5, 6, 7, 8, 12, 13, 14, 22, 32, 38)  # B C N O Mg Al Si Ti Ge Sr
_A0 = 0.529177211


def _recipe(Z: int, kind: str) -> list[float]:
    rng = np.random.default_rng([_SEED, Z, 0 if kind == "kirkland33" else 1])
    f0 = 1.2 * Z ** 0.66
    if kind == "kirkland33":
        w = rng.uniform(0.5, 1.5, 3)
        a = Z / (2.0 * np.pi ** 2 * _A0) * w / w.sum()
        b = np.sort(np.exp(rng.uniform(np.log(0.2), np.log(20.0), 3)))
        b *= (a / b).sum() / (0.5 * f0)
        v = rng.uniform(0.5, 1.5, 3)
        c = 0.5 * f0 * v / v.sum()
        d = np.sort(np.exp(rng.uniform(np.log(0.05), np.log(5.0), 3)))
        return [float(x) for x in np.concatenate([a, b, c, d])]
    if kind == "gauss5":
        v = rng.uniform(0.5, 1.5, 5)
        c = f0 * v / v.sum()
        d = np.sort(np.exp(rng.uniform(np.log(0.03), np.log(6.0), 5)))
        return [float(x) for x in np.concatenate([c, d])]
    raise ValueError(kind)


def generate_table() -> dict:
    return {
        "_label": "SURROGATE coefficients from a seeded recipe (workloads/form_factors.py); "
                  "not Kirkland's table, not physical data",
        "kirkland33": {str(Z): _recipe(Z, "kirkland33") for Z in ELEMENTS},
        "gauss5": {str(Z): _recipe(Z, "gauss5") for Z in ELEMENTS},
    }


def _load() -> dict:
    with open(_TABLE_PATH) as fh:
        return json.load(fh)


def form_factor_coefficients(Zs, kind: str = "kirkland33"):
    """Return (n_lorentz, n_gauss, coef[len(Zs)][2*n_lorentz+2*n_gauss]) for the listed Z.

    Row layout: a_1..a_nl, b_1..b_nl, c_1..c_ng, d_1..d_ng  (a: Angstrom^-1, b: Angstrom^-2,
    c: Angstrom, d: Angstrom^2).
    """
    tab = _load()[kind]
    nl, ng = (3, 3) if kind == "kirkland33" else (0, 5)
    coef = np.array([tab[str(int(Z))] for Z in Zs], dtype=np.float64)
    assert coef.shape[1] == 2 * nl + 2 * ng
    return nl, ng, coef


if __name__ == "__main__":
    with open(_TABLE_PATH, "w") as fh:
        json.dump(generate_table(), fh, indent=1)
    print("wrote", _TABLE_PATH)
