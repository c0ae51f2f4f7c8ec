r"""Writes paper_1702_01106_b200/data/linear_modes.json: the linear eigenmodes used as INITIAL DATA by the
synthetic workloads of BASELINE.json configs 1 and 3.  ORACLE-SIDE, TEST INFRASTRUCTURE.

    python oracle/write_mode_tables.py

Calls only oracle/ (linear_modes.py -> grim_oracle.c point functions).  The table holds inputs, not expected
results: background state, wave vector, eigenvalue and unit-norm eigenvector of each mode (P = P0 +
A Re[dP exp(i(k.x + phase))]).  Config 1: the fast magnetosonic mode of ideal MHD at
k = (2 pi, 2 pi) (the paper prints no ideal-MHD eigenvector; closed-form check in tests/test_oracle_linear.py).
Config 3: four EMHD modes, wave vectors 2 pi x integers in {-2..2}^3 \ 0 and the choice among the
non-zero-frequency eigenvectors drawn from numpy PCG64(1106).
"""
import json
import os

import numpy as np

import linear_modes as lm
import oracle as og

HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(os.path.dirname(HERE), "paper_1702_01106_b200", "data", "linear_modes.json")


def mode_record(k, w, v):
    v = lm.normalise_phase(v, comp=int(np.argmax(abs(v))))
    return {"k": [float(x) for x in k], "omega": [float(w.real), float(w.imag)],
            "dP_re": [float(x) for x in v.real], "dP_im": [float(x) for x in v.imag]}


def main():
    out = {"comment": "written by oracle/write_mode_tables.py; inputs for configs 1 and 3, not expected values"}
    # config 1: ideal MHD, fast mode, omega = +i 4.4145848550 (SURVEY P-3)
    P0 = np.array([1.0, 2.0, 0.0, 0.0, 0.0, 0.1, 0.3, 0.0])
    m8 = og.model(nvar=8)
    A, GP = lm.pencil(m8, P0)
    k = np.array([2 * np.pi, 2 * np.pi, 0.0])
    w, v = lm.eigenmodes(A, GP, k)
    j = int(np.argmax(w.imag))
    rec = mode_record(k, w[j], lm.normalise_phase(v[:, j], 0))
    # keep d(rho) real and positive for this one (SURVEY P-3 convention)
    vv = lm.normalise_phase(v[:, j], 0)
    rec["dP_re"], rec["dP_im"] = [float(x) for x in vv.real], [float(x) for x in vv.imag]
    out["config1"] = {"P0": [float(x) for x in P0], "gamma": 4.0 / 3.0, "modes": [rec]}
    # config 3: EMHD, four seeded modes
    P0e = np.array([1.0, 2.0, 0.0, 0.0, 0.0, 0.1, 0.3, 0.0, 0.0, 0.0])
    m10 = og.model(nvar=10)
    A, GP = lm.pencil(m10, P0e)
    rng = np.random.Generator(np.random.PCG64(1106))
    modes = []
    while len(modes) < 4:
        kint = rng.integers(-2, 3, size=3)
        if not np.any(kint):
            continue
        k = 2 * np.pi * kint.astype(float)
        w, v = lm.eigenmodes(A, GP, k)
        cand = [i for i in range(len(w)) if abs(w[i].imag) > 1e-6]
        i = cand[int(rng.integers(0, len(cand)))]
        rec = mode_record(k, w[i], v[:, i])
        rec["phase"] = float(rng.uniform(0.0, 2 * np.pi))
        modes.append(rec)
    out["config3"] = {"P0": [float(x) for x in P0e], "gamma": 4.0 / 3.0, "phi": 1.0, "psi": 1.0, "tau": 1.0,
                      "modes": modes}
    with open(OUT, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", OUT)


if __name__ == "__main__":
    main()
