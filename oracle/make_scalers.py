"""Write qnep_inputs/scalers.json: the frozen descriptor scaler s_nu of each config.

s_nu = 1 / (max_i D_nu - min_i D_nu), evaluated ONCE by the oracle on a step-0 structure of the
config's own construction, with the config's own random descriptor coefficients, then frozen as a
model parameter.  Calls only oracle/ and the input generators.

    python -m oracle.make_scalers
"""
import json
import os

import numpy as np

import qnep_inputs as I
from oracle import oracle as O


def main():
    out = {}
    samples = {
        "config0": lambda: I.config0(),
        "config1": lambda: I.config1(),
        "config2": lambda: I.config2(),
        # same construction at 8^3 cells (2560 atoms), same parameters as the 40^3 system
        "config3": lambda: I.config3(n_cells=8, grid=32),
        # config 4's parameters on a 10^3-molecule box of the same construction
        "config4": lambda: I.config4(n_side=10, grid=32),
        # configs 0-2 with NEP4's 4- and 5-body terms switched on (35 descriptors)
        "config0_45body": lambda: I.with_higher_body_terms(I.config0(), "config0_45body"),
        "config1_45body": lambda: I.with_higher_body_terms(I.config1(), "config1_45body"),
        "config2_45body": lambda: I.with_higher_body_terms(I.config2(), "config2_45body"),
    }
    for key, make in samples.items():
        w = make()
        D = O.descriptors(w.model, w.params.astype(np.float64), w.pos, w.types, w.box, use_bins=True)
        rng = D.max(axis=0) - D.min(axis=0)
        s = (1.0 / rng).astype(np.float32)          # stored at float32 precision, like all parameters
        out[key] = [float(x) for x in s]
        print(key, w.n_atoms, "atoms; scaler range", float(s.min()), float(s.max()))
    path = os.path.join(os.path.dirname(os.path.abspath(I.__file__)), "scalers.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
