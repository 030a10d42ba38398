"""Block Davidson-Liu eigensolver for the lowest roots of the TDA operator (oracle side).

Test infrastructure only (see oracle/__init__.py).

The paper says only "The diagonalization is carried out iteratively using the Davidson
method" and cites ref. 85.  The algorithm below is reading
A11 of DESIGN.md, step by step:
  start   V = orthonormalised P_c-projected start vectors (x0)
  loop    W = A V (new columns only);  H = (V^T W + W^T V)/2;  H y = theta y (ascending)
          r_i = W y_i - theta_i V y_i  for the lowest nroots;  converged when ||r_i|| <= tol
          t_i(G) = r_i(G) / d,  d = |G|^2/2 - eps_v - theta_i,  |d| floored at 1e-2 keeping sign
          t_i <- P_c t_i;  two passes of classical Gram-Schmidt against V, then P_c once more; if what is left has
          norm < 1e-10 ||t_i|| (the correction lies in span V, which happens when the preconditioner
          is exact) use the plain residual r_i instead; drop if that collapses too
          append;  if the basis would exceed max_subspace: restart from the Ritz vectors
All inner products are the Gamma-point inner product of the half-sphere storage.
The small dense eigenproblem uses numpy.linalg.eigh (a library primitive serving as a step).
Only eigenvalues are compared with the CUDA path (eigenvectors are not unique).
Pins: tests/test_oracle_davidson.py (D-only closed form; dense diagonalisation of the
operator matrix on a tiny cell).
"""
import numpy as np

from .liouville import SPIN_CONSERVING


def _gs2(problem, t, V, mode):
    """Two passes of classical Gram-Schmidt of t against the orthonormal columns V, then P_c again.

    The final projection keeps rounding noise out of the occupied space: without it the noise is
    amplified by ||t|| / ||t_perp|| at every step and the basis drifts out of range(P_c)."""
    for _ in range(2):
        if V:
            coef = [problem.vdot(v, t) for v in V]
            for c, v in zip(coef, V):
                t = t - c * v
    t = problem.project_vector(t, mode)
    return t, np.sqrt(max(problem.vdot(t, t), 0.0))


def davidson(problem, nroots, x0, mode=SPIN_CONSERVING, tol=1e-6, max_iter=200,
             max_subspace=None, guard=0):
    if max_subspace is None:
        max_subspace = 12 * nroots
    diag = problem.precond_diag(mode)
    V, W = [], []
    for x in np.asarray(x0, dtype=np.complex128):
        t = problem.project_vector(x, mode)
        t, nrm = _gs2(problem, t, V, mode)
        if nrm > 1e-10:
            V.append(t / nrm)
    history = []
    for it in range(1, max_iter + 1):
        if len(W) < len(V):
            W.extend(list(problem.apply(np.stack(V[len(W):]), mode)))
        m = len(V)
        H = np.array([[problem.vdot(V[i], W[j]) for j in range(m)] for i in range(m)])
        H = 0.5 * (H + H.T)
        theta, Y = np.linalg.eigh(H)
        nr = min(nroots, m)
        X = [sum(Y[j, i] * V[j] for j in range(m)) for i in range(nr)]
        R = [sum(Y[j, i] * W[j] for j in range(m)) - theta[i] * X[i] for i in range(nr)]
        res = np.array([np.sqrt(problem.vdot(r, r)) for r in R])
        history.append((it, m, theta[:nr].copy(), res.copy()))
        if np.all(res <= tol) and nr == nroots:
            return theta[:nroots], np.stack(X), it, res
        new = []
        for i in range(nr):
            if res[i] <= tol:
                continue
            d = diag - theta[i]
            d = np.where(np.abs(d) < 1e-2, np.where(d < 0, -1e-2, 1e-2), d)
            new.append((problem.project_vector(R[i] / d, mode), R[i]))
        if m + len(new) > max_subspace:
            # restart: keep the lowest nroots (+guard) Ritz vectors and their images
            keep = min(nroots + guard, m)
            Xk = [sum(Y[j, i] * V[j] for j in range(m)) for i in range(keep)]
            Wk = [sum(Y[j, i] * W[j] for j in range(m)) for i in range(keep)]
            V, W = [], []
            for xk, wk in zip(Xk, Wk):     # Ritz vectors are orthonormal up to rounding
                V.append(xk); W.append(wk)
        for t, r in new:
            n0 = np.sqrt(problem.vdot(t, t))
            t, nrm = _gs2(problem, t, V, mode)
            if nrm <= 1e-10 * n0:
                n0 = np.sqrt(problem.vdot(r, r))
                t, nrm = _gs2(problem, problem.project_vector(r, mode), V, mode)
            if nrm > 1e-10 * n0:
                V.append(t / nrm)
        if len(V) == len(W):
            break   # nothing could be added
    return theta[:nr], np.stack(X), it, res
