"""Linear theory of the oracle's equations about a uniform Minkowski background.  ORACLE-SIDE, TEST INFRASTRUCTURE.

Plays the role of the paper's linear-analysis package (L482): it builds the characteristic matrix of

    d_t U(P) + d_j F^j(P) - S(P, d_mu P) = 0                                    (eq 4, eqs 30-32, 39-40)

numerically from the oracle's own point functions (og_prim_to_U, og_prim_to_F, og_derived, og_emhd_targets,
og_rescale_factors), for plane waves  P = P0 + dP exp(i k.x + w t)  (L499).  Used to
  * pin the oracle against Table 1 (L484-499): M(w,k) dP = 0 and w an eigenvalue (pin P-1),
  * pin the ideal-MHD sector against the textbook magnetosonic / Alfven closed forms (P-3, P-13),
  * supply eigenvectors for the synthetic linear-mode inputs of configs 1 and 3 (written to
    paper_1702_01106_b200/data/linear_modes.json by oracle/write_mode_tables.py).
"""
import numpy as np

import oracle as og


def _dir_deriv(f, P, v, h):
    """4th-order central directional derivative of f at P along v."""
    return (8.0 * (f(P + h * v) - f(P - h * v)) - (f(P + 2 * h * v) - f(P - 2 * h * v))) / (12.0 * h)


def residual_density(m, P, d4, tau=1.0, h=1e-3):
    """G(P, d_mu P) = d_t U + d_j F^j - S, with d4[mu] = d_mu P (mu = t,1,2,3), Minkowski."""
    g = og.minkowski()
    n = m.nvar
    out = _dir_deriv(lambda p: og.prim_to_U(m, g, tau, p), P, d4[0], h)
    for j in (1, 2, 3):
        if np.any(d4[j] != 0):
            out = out + _dir_deriv(lambda p, j=j: og.prim_to_F(m, g, tau, j, p), P, d4[j], h)
    if n == 10:
        def der(p):
            th, ucon, ucov = og.derived(m, g, p)
            return np.concatenate([[th], ucov, ucon])
        dD = [(_dir_deriv(der, P, d4[mu], h) if np.any(d4[mu] != 0) else np.zeros(9)) for mu in range(4)]
        dTheta = np.array([dD[mu][0] for mu in range(4)])
        ducov = np.array([dD[mu][1:5] for mu in range(4)])
        ducon = np.array([dD[mu][5:9] for mu in range(4)])
        divu = sum(ducon[mu][mu] for mu in range(4))           # nabla_mu u^mu, flat space
        q0, dP0 = og.emhd_targets(m, g, np.zeros((4, 4, 4)), tau, P, dTheta, ducov, divu)
        fq, fd = og.rescale_factors(m, tau, P)
        qt, dpt = P[8] * fq, P[9] * fd
        out[8] -= -(qt - fq * q0) / tau + 0.5 * qt * divu       # eq 39
        out[9] -= -(dpt - fd * dP0) / tau + 0.5 * dpt * divu    # eq 40
    return out


def pencil(m, P0, tau=1.0):
    """Blocks A[mu] = dG/d(d_mu P) (mu = t,1,2,3) and GP = dG/dP at the uniform background P0."""
    n = m.nvar
    P0 = np.asarray(P0, dtype=np.float64)
    z = np.zeros((4, n))
    G0 = residual_density(m, P0, z, tau)
    A = []
    for mu in range(4):
        Am = np.zeros((n, n))
        for c in range(n):
            d4 = z.copy()
            d4[mu, c] = 1.0
            Am[:, c] = residual_density(m, P0, d4, tau) - G0
        A.append(Am)
    GP = np.zeros((n, n))
    hp = 1e-3
    for c in range(n):
        e = np.zeros(n)
        e[c] = 1.0
        GP[:, c] = _dir_deriv(lambda p: residual_density(m, p, z, tau), P0, e, hp)
    return A, GP


def char_matrix(A, GP, w, k):
    return w * A[0] + 1j * (k[0] * A[1] + k[1] * A[2] + k[2] * A[3]) + GP


def eigenmodes(A, GP, k):
    """All (w, dP) with (w A^t + i k_j A^j + G_P) dP = 0; eigenvectors as columns, unit 2-norm."""
    Cm = 1j * (k[0] * A[1] + k[1] * A[2] + k[2] * A[3]) + GP
    w, v = np.linalg.eig(np.linalg.solve(A[0], -Cm))
    v = v / np.linalg.norm(v, axis=0, keepdims=True)
    return w, v


def normalise_phase(v, comp=0):
    """Rotate the complex phase so that component `comp` is real and positive."""
    c = v[comp]
    if abs(c) == 0:
        return v
    return v * (abs(c) / c)
