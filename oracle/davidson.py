"""ORACLE Davidson (test infrastructure).  Single-root Davidson, reading 11
(the paper cites only Ref. 74):

  x0 normalised; iteration k: w_k = H b_k; G_ik = b_i.w_k; lowest eigenpair (theta, y) of
  the m x m matrix G; x = sum y_i b_i; r = sum y_i w_i - theta x; stop if |r| <= tol;
  t = r * den/(den^2 + delta^2), den = theta - Hd, delta = 1e-3; orthogonalise t against
  b_1..b_m by MODIFIED Gram-Schmidt (one basis vector at a time, each projection taken
  from the already-updated t) applied twice; normalise -> b_{m+1}.
  When m reaches max_space the basis collapses to {x}.  One iteration = one H psi.
"""
import numpy as np


def davidson(sigma_fn, hdiag, x0, max_iter, max_space, tol, delta=1e-3):
    n = x0.shape[0]
    b = [x0 / np.linalg.norm(x0)]
    w = []
    G = np.zeros((max_space, max_space))
    thetas = []
    theta, rn, x = None, None, b[0]
    it = 0
    while it < max_iter:
        w.append(sigma_fn(b[-1]))
        it += 1
        m = len(b)
        for i in range(m):
            G[i, m - 1] = G[m - 1, i] = float(np.dot(b[i], w[m - 1]))
        ev, evec = np.linalg.eigh(G[:m, :m])
        theta, y = ev[0], evec[:, 0]
        x = sum(y[i] * b[i] for i in range(m))
        hx = sum(y[i] * w[i] for i in range(m))
        r = hx - theta * x
        rn = float(np.linalg.norm(r))
        thetas.append(float(theta))
        if rn <= tol or it >= max_iter:
            break
        if m >= max_space:
            nx = np.linalg.norm(x)
            b, w = [x / nx], []
            G[:] = 0.0
            # re-evaluate H x on the collapsed basis (costs one H psi, counted)
            continue
        den = theta - hdiag
        t = r * den / (den * den + delta * delta)
        for _ in range(2):
            for bi in b:
                t = t - np.dot(bi, t) * bi
        nt = np.linalg.norm(t)
        b.append(t / nt)
    return {"energy": float(theta), "resid": rn, "iters": it, "x": x / np.linalg.norm(x), "thetas": thetas}
