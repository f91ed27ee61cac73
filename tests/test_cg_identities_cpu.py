"""The two CG identities the CUDA path leans on, checked in numpy on a small mesh (no GPU, no library code).

1. Hestenes-Stiefel: preconditioned CG started from x0 raises the energy E(x) = 2 b.x - x.Lx by exactly
   alpha_j rho_j per iteration (rho_j = r_j.z_j), so  E(x_k) = b.x0 + x0.r0 + sum_{j<k} alpha_j rho_j  and its
   distance to b.L^+ b is the SQUARE of the energy-norm error, whatever x0 was -- the form the bump / load
   diagonals Z[s,s] are taken from (csrc/guess.cuh, k_finish_term_guess).
2. The residual norm after an update is a quadratic in alpha whose coefficients do not depend on it,
   ||r - alpha q||^2 = ||r||^2 - 2 alpha r.q + alpha^2 ||q||^2  (csrc/stencil3.cuh k_pq3_last, csrc/pcg.cuh
   k_scal_estimate), with a cancellation error far below what a convergence check needs.
"""
import numpy as np


def mesh_laplacian(n, rng, jitter):
    """n x n mesh, segment conductance 1 / U[1 - jitter, 1 + jitter]; dense Laplacian."""
    N = n * n
    L = np.zeros((N, N))
    for y in range(n):
        for x in range(n):
            i = y * n + x
            for j in ((i + 1) if x + 1 < n else None, (i + n) if y + 1 < n else None):
                if j is not None:
                    g = 1.0 / rng.uniform(1.0 - jitter, 1.0 + jitter)
                    L[i, i] += g; L[j, j] += g; L[i, j] -= g; L[j, i] -= g
    return L


def pcg(L, M, b, x0, iters):
    """Textbook PCG; returns the iterates' scalars and vectors needed by the checks."""
    x = x0.copy()
    r = b - L @ x
    z = M @ r
    p = z.copy()
    rho = r @ z
    hist = []
    for _ in range(iters):
        q = L @ p
        alpha = rho / (p @ q)
        hist.append(dict(alpha=alpha, rho=rho, r=r.copy(), q=q.copy(), x=x.copy()))
        x = x + alpha * p
        r = r - alpha * q
        z = M @ r
        rho_new = r @ z
        p = z + (rho_new / rho) * p
        rho = rho_new
    return x, r, hist


def setup(seed=0, n=12):
    rng = np.random.default_rng(seed)
    L = mesh_laplacian(n, rng, 0.1)          # the tier
    Lm = mesh_laplacian(n, rng, 0.0)         # its mean mesh: the closed-form guess comes from this one
    N = n * n
    s = rng.integers(N)
    b = -np.ones(N) / N
    b[s] += 1.0
    x0 = np.linalg.pinv(Lm) @ b              # guess: ||b - L x0|| ~ 0.1 ||b||
    # a fixed SPD preconditioner that is good but not exact (a V-cycle stands here): pinv of a slightly different mesh
    M = np.linalg.pinv(mesh_laplacian(n, rng, 0.03))
    M = 0.5 * (M + M.T)
    ztrue = b @ np.linalg.pinv(L) @ b
    return L, M, b, x0, ztrue


def test_energy_gain_per_iteration_is_alpha_rho():
    L, M, b, x0, ztrue = setup()
    r0 = b - L @ x0
    for k in range(1, 5):
        x, r, hist = pcg(L, M, b, x0, k)
        energy = 2 * b @ x - x @ L @ x
        scalars = b @ x0 + x0 @ r0 + sum(h["alpha"] * h["rho"] for h in hist)
        assert abs(energy - scalars) <= 1e-12 * abs(energy)
        # the same through the residual: E(x_k) = b.x_k + x_k.r_k
        assert abs(energy - (b @ x + x @ r)) <= 1e-12 * abs(energy)


def test_energy_form_is_second_order_from_a_guess_and_the_plain_form_is_not():
    L, M, b, x0, ztrue = setup(seed=3)
    r0 = b - L @ x0
    x, r, hist = pcg(L, M, b, x0, 2)
    e = np.linalg.pinv(L) @ b - x
    e -= e.mean()
    err2 = e @ L @ e                                        # squared energy norm of the error
    scalars = b @ x0 + x0 @ r0 + sum(h["alpha"] * h["rho"] for h in hist)
    assert abs((ztrue - scalars) - err2) <= 1e-10 * ztrue   # E(x) - E(x_k) = ||x - x_k||_L^2 exactly
    assert err2 < 1e-6 * ztrue
    plain = b @ x                                           # first order in the error once x0 != 0
    assert abs(ztrue - plain) > 30 * err2


def test_residual_norm_after_the_update_from_sums():
    L, M, b, x0, _ = setup(seed=5)
    _, _, hist = pcg(L, M, b, x0, 4)
    for h in hist:
        r, q, a = h["r"], h["q"], h["alpha"]
        exact = np.sum((r - a * q) ** 2)
        terms = (r @ r, 2 * a * (r @ q), a * a * (q @ q))
        est = (terms[0] - terms[1]) + terms[2]
        noise = 1e-13 * sum(abs(t) for t in terms)          # k_scal_estimate's bound
        assert abs(est - exact) <= noise
        assert exact > 100 * noise                          # i.e. the estimate would have been trusted
        assert abs(est - exact) <= 1e-6 * exact
