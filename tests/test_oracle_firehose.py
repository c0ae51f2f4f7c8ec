"""Pin P-14: the firehose-unstable Alfven mode the paper prints (L583-601: growth rate Gamma = 0.1036, amplitudes
A = 0.1628, B = 0.9867 of u^2 and B^2; tests/golden/firehose_mode.txt).  It exercises what the Table-1 mode does not:
a background with non-zero pressure anisotropy (the dP terms of the stress tensor carry the instability, eqs 33-34)
and a slow relaxation time.  (a) linear theory of the oracle's point functions; (b) the oracle's time stepping grows
the mode at that rate."""
import numpy as np

import linear_modes as lm
import oracle as og
from common import oracle_grid
from conftest import read_golden_table


def golden():
    r = read_golden_table("firehose_mode.txt")
    return {k: v[0] for k, v in r.items()}


def background(t):
    return np.array([t["rho"], t["u"], 0.0, 0.0, 0.0, t["B1"], 0.0, 0.0, 0.0, t["dP"]])


def test_firehose_growth_rate_and_eigenvector_from_linear_theory():
    t = golden()
    m = og.model(nvar=10)
    A, GP = lm.pencil(m, background(t), tau=t["tau"])
    w, v = lm.eigenmodes(A, GP, np.array([t["k1"], 0.0, 0.0]))
    uns = [i for i in range(len(w)) if w[i].real > 1e-3]
    assert len(uns) == 2                                   # the two transverse polarisations of the Alfven mode
    for i in uns:
        assert abs(w[i].real - t["Gamma"]) < 1e-4          # the paper prints four digits
        assert abs(w[i].imag) < 1e-9                       # purely growing
        vv = v[:, i]
        up, bp = np.linalg.norm(vv[3:5]), np.linalg.norm(vv[6:8])
        assert abs(up - t["A"]) < 2e-4 and abs(bp - t["B"]) < 2e-4
        assert np.linalg.norm(vv[[0, 1, 2, 5, 8, 9]]) < 1e-8
        # u^2 ~ sin, B^2 ~ cos: a quarter period apart
        j = 3 if abs(vv[3]) > abs(vv[4]) else 4
        ratio = vv[j] / vv[j + 3]
        assert abs(ratio.real) < 1e-6 * abs(ratio)


def test_firehose_mode_grows_at_the_printed_rate_in_the_scheme():
    """The paper's initial data (eqs 58-65, workloads.firehose) evolved by the oracle's time stepping: the amplitude
    of B^2 grows as exp(0.1036 t) over 0 < t < 3 (Fig. 9's first regime)."""
    from paper_1702_01106_b200 import workloads
    t = golden()
    gk, P = workloads.firehose(n=64, alpha=1e-6)
    assert gk["tau"] == t["tau"] and P[9].max() == t["dP"] and P[5].max() == t["B1"]
    g = oracle_grid(gk)
    g.fill_ghosts(P)
    dt = g.choose_dt(P)

    def amp(P):
        return np.sqrt(2 * np.mean(g.interior(P)[6] ** 2))

    a0, tt = amp(P), 0.0
    while tt < 3.0:
        st = g.timestep(P, dt)
        assert st.unconverged[1] == 0
        tt += dt
    rate = np.log(amp(P) / a0) / tt
    assert abs(rate - t["Gamma"]) < 2e-3, rate
