"""Writes stev_inputs/data/relaxed_pool_cfg2.npy -- the near-equilibrium pool of config 2.

BASELINE.json config 2: "60% of cells near equilibrium at 1000 K so they retire early".  The pool is 512
random compositions (Dirichlet(1), seed below) that the CPU ORACLE relaxes isothermally at 1000 K and
3 atm for 20 dt_cfd; the field generator jitters copies of them.  This script calls only oracle/ and
stev_inputs/ (never the CUDA path).  Run:  python -m oracle.make_relaxed_pool
"""
import os

import numpy as np

from oracle import stev_oracle as O
from stev_inputs.configs import BASE_SEED, DT_CFD, default_params, make_mechanism
from stev_inputs.mechanisms import P_ATM


def main() -> None:
    mech = make_mechanism(2)
    rng = np.random.default_rng(BASE_SEED + 29)
    n = 512
    Y = np.ascontiguousarray(rng.dirichlet(np.ones(mech.n_species), n).T)
    prm = default_params()
    prm["energy_mode"] = 1
    r = O.integrate(mech, None, prm, np.full(n, 1000.0), np.full(n, 3.0 * P_ATM), Y, 20.0 * DT_CFD[2])
    assert (r["status"] == 0).all()
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "stev_inputs", "data", "relaxed_pool_cfg2.npy")
    np.save(out, np.ascontiguousarray(r["Y"].T))
    print("wrote", os.path.normpath(out), "steps median", int(np.median(r["steps"])))


if __name__ == "__main__":
    main()
