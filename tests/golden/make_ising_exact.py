"""Writes tests/golden/ising_exact.json from closed forms only (tests/exact_ising.py: Kaufman's finite-lattice
partition function, brute-force enumeration at L=4, Onsager's limit), in 30 significant digits.
Calls neither oracle/ nor the CUDA path.  The same numbers are quoted in SURVEY.md section 8(c)
("Reference values (survey check, mpmath 60 digits)"), which tests/test_oracle_pins.py cross-checks.

    python tests/golden/make_ising_exact.py
"""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
from exact_ising import brute_force_dos, kaufman_lnZ, onsager_lnZ_per_site  # noqa: E402
from mpmath import nstr  # noqa: E402

out = {
    "_cite": "Kaufman 1949 closed form for the LxL torus; PAPER.md:33 eq.1 (Z), :78 eq.6 (H); SURVEY.md 8(c)",
    "dos_L4": {str(k): v for k, v in brute_force_dos(4)[0].items()},
    "lnZ": {},
    "onsager_lnZ_per_site": {},
}
for L, betas in {4: [0.005, 0.1, 0.4407, 0.5, 0.6, 1.0], 8: [0.5, 0.6, 1.0], 16: [0.5, 0.6, 1.0], 32: [1.0],
                 64: [0.5], 128: [0.6]}.items():
    for b in betas:
        out["lnZ"]["L%d_beta%g" % (L, b)] = nstr(kaufman_lnZ(L, b), 30)
for b in [0.5, 0.6, 1.0]:
    out["onsager_lnZ_per_site"]["beta%g" % b] = nstr(onsager_lnZ_per_site(b), 30)
with open(os.path.join(HERE, "ising_exact.json"), "w") as f:
    json.dump(out, f, indent=1, sort_keys=True)
    f.write("\n")
print("wrote", os.path.join(HERE, "ising_exact.json"))
