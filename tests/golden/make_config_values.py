"""Writes tests/golden/config_values.json: the observables BASELINE.json's configs 1 and 2 ask to report
(plaquette, kinetic energy, dH), computed by the CPU ORACLE ONLY (oracle/, serial build) from the seeded
start of DESIGN.md section 4.  Never calls the CUDA path.

    python tests/golden/make_config_values.py

These are regression values for the oracle itself (tests/test_oracle_pins.py checks that the oracle still
reproduces them) and the numbers the GPU trajectory tests are compared with; their correctness rests on the
pins of the oracle's functions, not on this file."""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle.oracle import Oracle  # noqa: E402
from tests import inputs  # noqa: E402


def main():
    orc = Oracle(omp=False)
    out = {}
    for n in (1, 2):
        c = inputs.CONFIGS[n]
        dims, beta, eps, nsteps = c["dims"], c["beta"], c["eps"], c["nsteps"]
        seed = inputs.config_seed(n)
        U0, P0 = orc.hot_start(dims, seed, c["sigma"]), orc.mom_refresh(dims, seed)
        K0, S0 = orc.hamiltonian(dims, beta, U0, P0)
        U1, P1 = orc.leapfrog(dims, beta, eps, nsteps, U0, P0)
        K1, S1 = orc.hamiltonian(dims, beta, U1, P1)
        out[str(n)] = {"dims": list(dims), "beta": beta, "eps": eps, "nsteps": nsteps, "sigma": c["sigma"],
                       "seed": hex(seed), "plaq0": orc.plaquette(dims, U0)[0], "K0": K0, "S0": S0,
                       "plaq1": orc.plaquette(dims, U1)[0], "K1": K1, "S1": S1, "dH": (K1 + S1) - (K0 + S0)}
    with open(os.path.join(HERE, "config_values.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out, indent=1))


if __name__ == "__main__":
    main()
