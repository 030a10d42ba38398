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
Reading A11b (precond="projector", the default of the CUDA path): the diagonal correction ignores that D = P_c (T - eps_v) P_c
is not diagonal in the plane-wave basis when the occupied orbitals are not eigenfunctions of T.  The projector-aware correction
solves  P_c (T - lambda) P_c t = r  on range(P_c) exactly, block by block (lambda = eps_v + theta_i, the same floor on |d|):
          t = M^-1 (r - Phi c),   c = S^-1 Phi^T M^-1 r,   S = Phi^T M^-1 Phi,   M = diag(|G|^2/2 - lambda)
(Phi = occupied orbitals of the target spin; Phi^T t = 0 by construction).  It changes the path, not the converged eigenvalues.
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


def _blocks(problem, mode):
    """(occupied spin, target spin, number of functions) of each spin block of a trial vector."""
    if mode == SPIN_CONSERVING:
        return [(s, s, problem.nocc[s]) for s in range(problem.nspin)]
    so = 0 if mode == 1 else 1
    return [(so, 1 - so, problem.nocc[so])]


def precond_projector(problem, r, theta, mode):
    """Reading A11b: t with P_c (T - eps_v - theta) P_c t = r on range(P_c), for every function of the trial vector r."""
    out = []
    xs = problem.split(r, mode)
    for (so, st, n), blk in zip(_blocks(problem, mode), xs):
        Phi = problem.psi[st]
        for v in range(n):
            d = 0.5 * problem.g2 - problem.eig[so][v] - theta
            d = np.where(np.abs(d) < 1e-2, np.where(d < 0, -1e-2, 1e-2), d)
            w = 2.0 / d
            w[0] = 1.0 / d[0]                                   # Gamma inner product weighted by M^-1
            S = np.real((np.conj(Phi) * w) @ Phi.T)             # S_uu' = <phi_u| M^-1 |phi_u'>
            b = np.real((np.conj(Phi) * w) @ blk[v])            # <phi_u| M^-1 |r>
            c = np.linalg.solve(S, b)
            out.append((blk[v] - c @ Phi) / d)
    return np.concatenate(out)


def d_start_vectors(problem, nstart, mode=SPIN_CONSERVING, per_spin=4):
    """Reading A11c: start vectors = the nstart lowest eigenvectors of D alone (Eq. 3).  D is block diagonal in the
    occupied index v, D_v = P_c T P_c - eps_v on range(P_c), so its eigenvectors are u_m (x) e_v with u_m the eigenfunctions of
    P_c T P_c (eigenvalue mu_m) of the target spin.  Here the u_m come from a dense diagonalisation of P_c T P_c written in the
    real coordinates (1, sqrt2 cos, sqrt2 sin) of the half-sphere storage; the `per_spin` lowest are used.
    Returns complex [nstart, vector_len]."""
    r2 = np.sqrt(2.0)
    cands, funcs = [], {}
    off = 0
    for b, (so, st, n) in enumerate(_blocks(problem, mode)):
        if st not in funcs:
            c = problem.psi[st]
            U = np.concatenate([c[:, :1].real, r2 * c[:, 1:].real, r2 * c[:, 1:].imag], axis=1)      # orthonormal rows
            kin = 0.5 * np.concatenate([problem.g2, problem.g2[1:]])
            P = np.eye(U.shape[1]) - U.T @ U
            w, v = np.linalg.eigh(P @ (kin[:, None] * P))
            keep = np.where(w > 1e-8)[0][:per_spin]              # the null space is span(Phi)
            npwh = problem.npwh
            fs = []
            for k in keep:
                f = np.zeros(npwh, dtype=np.complex128)
                f[0] = v[0, k]
                f[1:] = (v[1:npwh, k] + 1j * v[npwh:, k]) / r2
                fs.append(f)
            funcs[st] = (w[keep], fs)
        mu, fs = funcs[st]
        for m in range(len(mu)):
            for vv in range(n):
                cands.append((mu[m] - problem.eig[so][vv], off + vv * problem.npwh, st, m))
        off += n * problem.npwh
    cands.sort(key=lambda t: t[0])
    x0 = np.zeros((nstart, problem.vector_len(mode)), dtype=np.complex128)
    for i, (_, o, st, m) in enumerate(cands[:nstart]):
        x0[i, o:o + problem.npwh] = funcs[st][1][m]
    return x0


def davidson(problem, nroots, x0, mode=SPIN_CONSERVING, tol=1e-6, max_iter=200,
             max_subspace=None, guard=0, precond="diagonal", block=None, history_out=None):
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
        if history_out is not None:
            history_out.append(history[-1])
        if np.all(res <= tol) and nr == nroots:
            return theta[:nroots], np.stack(X), it, res
        new = []
        for i in range(nr):
            if res[i] <= tol:
                continue
            if block is not None and len(new) >= block:
                break
            if precond == "projector":
                t = precond_projector(problem, R[i], theta[i], mode)
            else:
                d = diag - theta[i]
                d = np.where(np.abs(d) < 1e-2, np.where(d < 0, -1e-2, 1e-2), d)
                t = R[i] / d
            new.append((problem.project_vector(t, mode), R[i]))
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
