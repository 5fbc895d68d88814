"""The Davidson iteration, step by step (reading of SURVEY.md §8(c); the paper
says only "Lánczos or Davidson" with thresholds ε = 1e-5, 1e-7 — PAPER.md:60,
114, 118).  One pass of the loop = one "Davidson step" = exactly one H_eff apply.

    V=[x0/‖x0‖]; W=[H V0]; m=1
    repeat:  G = VᵀW ; G ← (G+Gᵀ)/2 ; (θ,y) = lowest eigenpair of G
             x = V y ; r = W y − θ x ; ρ = ‖r‖₂ ; if ρ ≤ tol: stop
             if m == m_max: V=[x], W=[W y], m=1            (collapse restart)
             t_i = r_i / (θ − d_i), |θ − d_i| < 1e-10 replaced by sign·1e-10
             t ← t − V(Vᵀt), twice ; if ‖t‖ < 1e-14‖r‖: t ← r orthogonalised
             v = t/‖t‖ ; w = H v ; append (v,w) ; m += 1

ε_Davidson is read as the residual 2-norm ‖Hx − θx‖ ≤ ε for normalised x (r10);
the preconditioner is the diagonal of H_eff, m_max = 16, collapse restart (r11).
"""
import numpy as np


def davidson(apply, diag, x0, tol=1e-9, m_max=16, max_iter=500, history=None):
    """Lowest eigenpair of the symmetric operator ``apply`` (flat vectors).
    Returns (θ, x, number of operator applications)."""
    x0 = np.asarray(x0, dtype=np.float64)
    V = [x0 / np.linalg.norm(x0)]
    W = [apply(V[0])]
    n_apply = 1
    theta, x = None, None
    for _ in range(max_iter):
        Vm, Wm = np.stack(V, axis=1), np.stack(W, axis=1)
        G = Vm.T @ Wm
        G = 0.5 * (G + G.T)
        w, Y = np.linalg.eigh(G)
        theta, y = float(w[0]), Y[:, 0]
        x = Vm @ y
        Wy = Wm @ y
        r = Wy - theta * x
        rho = float(np.linalg.norm(r))
        if history is not None:
            history.append((theta, rho))
        if rho <= tol:
            break
        if len(V) == m_max:
            V, W = [x], [Wy]
            Vm = np.stack(V, axis=1)
        den = theta - diag
        small = np.abs(den) < 1e-10
        den = np.where(small, np.where(den < 0, -1e-10, 1e-10), den)
        t = r / den
        for _ in range(2):
            t = t - Vm @ (Vm.T @ t)
        if np.linalg.norm(t) < 1e-14 * rho:
            t = r.copy()
            for _ in range(2):
                t = t - Vm @ (Vm.T @ t)
        v = t / np.linalg.norm(t)
        V.append(v)
        W.append(apply(v))
        n_apply += 1
    return theta, x, n_apply
