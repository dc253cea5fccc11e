"""Oracle of the solver rows of SURVEY.md section 8(f)2-3: the linear-Jacobian preconditioner
(App. B, App. C, section 4.2), right-preconditioned GMRES
(section 4.1) and the damped Newton iteration (eqs. (2), (3) L41-45).

TEST INFRASTRUCTURE, like everything under oracle/: plain numpy in FP64, dense matrices, the
formulas of the paper written out entry by entry, no blocking and no reordering.  It shares
nothing with the CUDA path.  The residual E(u) and the Jacobian action J(u) v it drives are
the C oracle's (`Oracle.residual`, `Oracle.jv_exact`).

Indexing (0-based in the arrays; k, l, n, m are the paper's 1-based indices in comments):
  unknown  phi_{1,m}      -> column (m-1)(N+1)              eq. (18)
           (phi_x)_{n,m}  -> column (m-1)(N+1) + n
           zeta block     -> the same + (N+1)M
  equation E3_l, E4_l     -> rows (l-1)(N+1), (l-1)(N+1)+1  App. A
           E1_{k,l}       -> row  (l-1)(N+1) + 1 + k
           E5, E6, E2     -> the same + (N+1)M

Pins (tests/test_oracle_jfnk.py): the dense linear Jacobian against the complex-step Jacobian
of the NONLINEAR residual at the flat state with eps = 0 (every column, tiny mesh); the App. C
block solve against numpy.linalg.solve on the assembled P; GMRES against numpy.linalg.solve
and scipy.sparse.linalg.gmres on explicit matrices; Newton against the root of a problem with
a known solution and against Newton with the explicit dense Jacobian.
"""
from __future__ import annotations

import numpy as np


# ---------------------------------------------------------------------------------------
# App. B: the linear Jacobian
def _mesh(p: dict):
    N, M = int(p["N"]), int(p["M"])
    x = p["x1"] + p["dx"] * np.arange(N)
    y = p["y1"] + p["dy"] * np.arange(M)
    return N, M, x, y


def midpoint_coefficients(N: int, dx: float) -> np.ndarray:
    """T[k-1, c]: coefficient of unknown c (c = 0: f_1, c = n: (f_x)_n) in the half-mesh value
    f*_k = (f_k + f_{k+1}) / 2, k = 1..N-1, with f_k the trapezoid expansion L446-450.
    Entries exactly as printed in (B.2) L458-460: Delta x/4 (n=1,k=1), Delta x/2 (n=1,k>1),
    Delta x (1<n<k), 3 Delta x/4 (n=k), Delta x/4 (n=k+1) and 1 for f_1 (reading Q8 for B.4)."""
    T = np.zeros((N - 1, N + 1))
    for k in range(1, N):
        T[k - 1, 0] = 1.0
        for n in range(1, N + 1):
            if n == 1 and k == 1:
                c = dx / 4
            elif n == 1 and k > 1:
                c = dx / 2
            elif n < k:
                c = dx
            elif n == k:
                c = 3 * dx / 4
            elif n == k + 1:
                c = dx / 4
            else:
                c = 0.0
            T[k - 1, n] = c
    return T


def k3(x, y, xs, ys):
    """K3 of eq. (17) L139 (direct + image)."""
    return 1.0 / np.sqrt((x - xs) ** 2 + (y - ys) ** 2) + 1.0 / np.sqrt((x - xs) ** 2 + (y + ys) ** 2)


def trapezoid_weights(p: dict) -> np.ndarray:
    """w(i, j) = dx dy c_i c_j, c = 1/2 on the first/last index (reading Q4); [M, N]."""
    N, M = int(p["N"]), int(p["M"])
    cx = np.ones(N); cx[[0, -1]] = 0.5
    cy = np.ones(M); cy[[0, -1]] = 0.5
    return p["dx"] * p["dy"] * np.outer(cy, cx)


def linear_I(p: dict, xs: float, ys: float, box_integral) -> float:
    """I = int int K3 dx dy over the truncated rectangle (L440): the closed form of eq. (23)
    with A = C = 1, B = 0 (reading Q5), direct box + image box.  `box_integral` is the pinned
    C-oracle routine (pin P5)."""
    N, M, x, y = _mesh(p)
    s1, s2 = x[0] - xs, x[-1] - xs
    return (box_integral(1.0, 0.0, 1.0, s1, s2, y[0] - ys, y[-1] - ys)
            + box_integral(1.0, 0.0, 1.0, s1, s2, -(y[-1] + ys), -(y[0] + ys)))


def linear_jacobian(p: dict, box_integral) -> np.ndarray:
    """The dense linear Jacobian P = [A B; C D] of App. B (B.3)-(B.6) L472-503 with the radiation
    rows of (B.2) L462-468, ordered by eq. (18) / App. A.  Independent of u and of eps."""
    N, M, x, y = _mesh(p)
    n1, H = N + 1, (N + 1) * M
    dx, F2, nr, x1 = p["dx"], p["froude"] ** 2, p["n_rad"], p["x1"]
    P = np.zeros((2 * H, 2 * H))
    T = midpoint_coefficients(N, dx)
    w = trapezoid_weights(p)
    xs = 0.5 * (x[:-1] + x[1:])
    X, Y = np.meshgrid(x, y)                       # [M, N]
    for l in range(M):
        r0, c0 = l * n1, l * n1
        # radiation rows E3, E4 (phi block) and E5, E6 (zeta block), (B.2) L462-468
        for off in (0, H):
            P[off + r0, off + c0] = nr
            P[off + r0, off + c0 + 1] = x1
            P[off + r0 + 1, off + c0 + 1] = nr - x1 / dx
            P[off + r0 + 1, off + c0 + 2] = x1 / dx
        for k in range(1, N):
            r = r0 + 1 + k
            # (B.3): dE1/d(phi_x)_{n,l} = 1/2 for n = k, k+1
            P[r, c0 + k] = 0.5
            P[r, c0 + k + 1] = 0.5
            # (B.4): dE1/d(zeta unknowns of line l) = (1/F^2) d zeta*_k
            P[r, H + c0:H + c0 + n1] = T[k - 1] / F2
            # (B.5): dE2/d(phi unknowns of line l) = 2 pi d phi*_k
            P[H + r, c0:c0 + n1] = 2 * np.pi * T[k - 1]
            # (B.6): dE2/d(zeta_x)_{n,m} = -w(n,m) K3 (+ (sum w K3 - I)/2 for n = k,k+1, m = l)
            K = k3(X, Y, xs[k - 1], y[l])           # [M, N]
            wK = w * K
            for m in range(M):
                P[H + r, H + m * n1 + 1:H + m * n1 + 1 + N] = -wK[m]
            corr = 0.5 * (wK.sum() - linear_I(p, xs[k - 1], y[l], box_integral))
            P[H + r, H + c0 + k] += corr
            P[H + r, H + c0 + k + 1] += corr
    return P


def band_truncate(P: np.ndarray, p: dict, b: int) -> np.ndarray:
    """Section 4.2: keep the lower-right submatrix D only within block bandwidth b
    (blocks (N+1) x (N+1); b = 1 block diagonal, b = 3 block tridiagonal, ...: |l - m| <= (b-1)/2)."""
    N, M = int(p["N"]), int(p["M"])
    n1, H = N + 1, (N + 1) * M
    if b % 2 != 1 or b < 1:
        raise ValueError("block bandwidth b must be odd and >= 1")
    hb = (b - 1) // 2
    Q = P.copy()
    for l in range(M):
        for m in range(M):
            if abs(l - m) > hb:
                Q[H + l * n1:H + (l + 1) * n1, H + m * n1:H + (m + 1) * n1] = 0.0
    return Q


def precond_solve_blocks(P: np.ndarray, rhs: np.ndarray) -> np.ndarray:
    """Solve P r = rhs by the block factorisation of App. C:
    t2 = b2 - C A^-1 b1; s1 = A^-1 b1; s2 = (D - C A^-1 B)^-1 t2; r1 = s1 - A^-1 B s2; r2 = s2."""
    H = P.shape[0] // 2
    A, B, C, D = P[:H, :H], P[:H, H:], P[H:, :H], P[H:, H:]
    b1, b2 = rhs[:H], rhs[H:]
    s1 = np.linalg.solve(A, b1)
    t2 = b2 - C @ s1
    S = D - C @ np.linalg.solve(A, B)
    s2 = np.linalg.solve(S, t2)
    r1 = s1 - np.linalg.solve(A, B @ s2)
    return np.concatenate([r1, s2])


# ---------------------------------------------------------------------------------------
# Section 4.1: right-preconditioned GMRES (Saad & Schultz [47]) and the damped Newton iteration
def gmres_right(apply_J, apply_Pinv, rhs, tol: float, restart: int, maxit: int):
    """Solve J d = rhs with GMRES(restart) on J P^-1 (right preconditioning, L209-215): the
    iterate after m steps is d = P^-1 V_m y_m with y_m minimising ||rhs - J P^-1 V_m y||_2 over
    the Krylov space K_m(J P^-1, rhs) (L213).  Textbook form: modified Gram-Schmidt Arnoldi,
    Givens rotations on the Hessenberg matrix, zero initial guess, stop when the residual
    estimate is <= tol * ||rhs||_2 or after maxit matrix-vector products in total.
    Returns (d, history) with history[i] = ||residual||_2 / ||rhs||_2 after i+1 products."""
    n = rhs.size
    d = np.zeros(n)
    bnorm = float(np.linalg.norm(rhs))
    hist = []
    if bnorm == 0.0:
        return d, hist
    r = rhs.copy()
    its = 0
    while its < maxit:
        beta = float(np.linalg.norm(r))
        V = np.zeros((restart + 1, n))
        Hm = np.zeros((restart + 1, restart))
        cs, sn = np.zeros(restart), np.zeros(restart)
        g = np.zeros(restart + 1)
        g[0] = beta
        V[0] = r / beta
        j_done = 0
        for j in range(restart):
            wv = apply_J(apply_Pinv(V[j]))
            its += 1
            for i in range(j + 1):
                Hm[i, j] = float(wv @ V[i])
                wv = wv - Hm[i, j] * V[i]
            Hm[j + 1, j] = float(np.linalg.norm(wv))
            if Hm[j + 1, j] > 0.0:
                V[j + 1] = wv / Hm[j + 1, j]
            for i in range(j):
                t = cs[i] * Hm[i, j] + sn[i] * Hm[i + 1, j]
                Hm[i + 1, j] = -sn[i] * Hm[i, j] + cs[i] * Hm[i + 1, j]
                Hm[i, j] = t
            rho = float(np.hypot(Hm[j, j], Hm[j + 1, j]))
            cs[j], sn[j] = Hm[j, j] / rho, Hm[j + 1, j] / rho
            Hm[j, j], Hm[j + 1, j] = rho, 0.0
            g[j + 1] = -sn[j] * g[j]
            g[j] = cs[j] * g[j]
            j_done = j + 1
            hist.append(abs(g[j + 1]) / bnorm)
            if abs(g[j + 1]) <= tol * bnorm or its >= maxit:
                break
        yv = np.linalg.solve(np.triu(Hm[:j_done, :j_done]), g[:j_done])
        d = d + apply_Pinv(yv @ V[:j_done])
        if hist[-1] <= tol or its >= maxit:
            break
        r = rhs - apply_J(d)
    return d, hist


def newton(residual, jv, apply_Pinv, u0, *, ftol: float, eta: float, restart: int, gmres_maxit: int,
           max_newton: int = 30, alpha: float = 1e-4, max_halvings: int = 20, forcing: int = 0,
           eta_max: float = 0.5):
    """Damped Newton iteration (2), (3) L41-45 with the simple line search of L209: lambda = 1,
    1/2, 1/4, ... until ||E(u + lambda du)||_2 < (1 - alpha lambda) ||E(u)||_2 (reading Q14: the
    paper only asks for a sufficient decrease; it used KINSOL's line search, L255).  The Newton
    correction solves J(u_k) du = -E(u_k) approximately (inexact Newton, L223) by `gmres_right`
    to the relative tolerance eta.  Stops when ||E||_inf <= ftol.
    forcing = 1: the tolerance of step k follows the nonlinear progress (the forcing term "choice 2" of
    Eisenstat & Walker as stated in the survey the paper cites for its inexact Newton method, [21] L223,
    L372): eta_0 = eta_max, eta_k = 0.9 (||E_k|| / ||E_{k-1}||)^2, raised to 0.9 eta_{k-1}^2 when that
    exceeds 0.1 (safeguard), then clipped to [eta, eta_max].
      residual(u) -> E(u);   jv(u, v) -> J(u) v.
    Returns (u, log) with one log entry per Newton step."""
    u = np.array(u0, dtype=np.float64)
    E = residual(u)
    log = []
    eta_k = eta_max if forcing == 1 else eta
    for it in range(max_newton):
        fn = float(np.linalg.norm(E))
        if float(np.abs(E).max()) <= ftol:
            break
        du, hist = gmres_right(lambda v: jv(u, v), apply_Pinv, -E, eta_k, restart, gmres_maxit)
        lam, ok = 1.0, False
        for _ in range(max_halvings + 1):
            Et = residual(u + lam * du)
            if float(np.linalg.norm(Et)) < (1.0 - alpha * lam) * fn:
                ok = True
                break
            lam *= 0.5
        log.append({"newton": it, "fnorm": fn, "finf": float(np.abs(E).max()), "gmres_its": len(hist),
                    "gmres_rel": hist[-1] if hist else 0.0, "lambda": lam if ok else 0.0})
        if not ok:
            break
        u = u + lam * du
        E = Et
        if forcing == 1:
            fnt = float(np.linalg.norm(E))
            e = 0.9 * (fnt / fn) ** 2
            sg = 0.9 * eta_k * eta_k
            if sg > 0.1:
                e = max(e, sg)
            eta_k = min(eta_max, max(e, eta))
    log.append({"newton": len(log), "fnorm": float(np.linalg.norm(E)), "finf": float(np.abs(E).max()),
                "gmres_its": 0, "gmres_rel": 0.0, "lambda": 0.0})
    return u, log


# ---------------------------------------------------------------------------------------
# Enlarged (block) GMRES: a Krylov method that uses b > 1 Jacobian-vector products per iteration
# ("block/s-step Krylov that actually uses b>1"; the paper's own solver is plain GMRES,
# section 4.1).  Plain restatement of the enlarged Krylov idea: the right-hand side is split by a
# partition of the unknowns into t vectors that sum to it,
#     R0 = [T_1 r, ..., T_t r],   r = R0 1,
# the BLOCK Krylov space K_m(J P^-1, R0) is built by block Arnoldi - ONE application of J to t vectors per
# iteration - and the iterate is d = P^-1 V y with y minimising ||r - J P^-1 V y||_2 over that space, which
# contains K_m(J P^-1, r) (so m block iterations are at least as good as m plain GMRES iterations).
def line_partition(p: dict, t: int) -> np.ndarray:
    """group[idx] in 0..t-1 for every unknown idx of eq. (18): the y-lines are cut into t contiguous
    groups, line l (0-based) belongs to group floor(l t / M); the phi and the zeta unknowns of a line go
    together."""
    N, M = int(p["N"]), int(p["M"])
    line = np.tile(np.repeat(np.arange(M), N + 1), 2)
    return (line * t) // M


def _mgs_qr(W: np.ndarray):
    """W [t, n] (rows are vectors) = R^T-combination of orthonormal rows Q: modified Gram-Schmidt, column by
    column, positive diagonal.  Returns (Q [t, n], R [t, t] upper triangular) with W^T = Q^T R."""
    t = W.shape[0]
    Q = np.zeros_like(W)
    R = np.zeros((t, t))
    for c in range(t):
        w = W[c].copy()
        for i in range(c):
            R[i, c] = float(Q[i] @ w)
            w = w - R[i, c] * Q[i]
        R[c, c] = float(np.linalg.norm(w))
        if R[c, c] == 0.0:
            raise np.linalg.LinAlgError("enlarged GMRES: rank-deficient block (breakdown)")
        Q[c] = w / R[c, c]
    return Q, R


def egmres_right(apply_J_block, apply_Pinv, rhs, group, t: int, tol: float, max_blocks: int):
    """Solve J d = rhs by enlarged GMRES with t right-hand-side pieces (no restart), right preconditioned.
      apply_J_block(Z) -> J Z for Z [t, n] (rows are vectors): the ONE batched product per iteration.
      group: partition of the unknowns (line_partition).
    Block Arnoldi with block modified Gram-Schmidt; the (m+1)t x mt band Hessenberg least-squares problem
    min ||e_1 (x) (B 1) - H y||_2 is solved by numpy.linalg.lstsq from scratch after every block (plain).
    Returns (d, history): history[j] = ||rhs - J d_j||_2 / ||rhs||_2 after j+1 block iterations."""
    n = rhs.size
    bnorm = float(np.linalg.norm(rhs))
    hist = []
    d = np.zeros(n)
    if bnorm == 0.0:
        return d, hist
    R0 = np.stack([np.where(group == i, rhs, 0.0) for i in range(t)])         # [t, n], rows sum to rhs
    V = np.zeros(((max_blocks + 1) * t, n))
    Hh = np.zeros(((max_blocks + 1) * t, max_blocks * t))
    V[:t], B = _mgs_qr(R0)
    g0 = B @ np.ones(t)                                                        # rhs = V_1^T (B 1)
    for j in range(max_blocks):
        Z = np.stack([apply_Pinv(V[j * t + c]) for c in range(t)])
        W = apply_J_block(Z)                                                   # t products at once
        for i in range(j + 1):                                                 # block modified Gram-Schmidt
            Vi = V[i * t:(i + 1) * t]
            Hij = Vi @ W.T                                                     # [t, t]: (V_i^T W)
            Hh[i * t:(i + 1) * t, j * t:(j + 1) * t] = Hij
            W = W - Hij.T @ Vi
        Q, R = _mgs_qr(W)
        V[(j + 1) * t:(j + 2) * t] = Q
        Hh[(j + 1) * t:(j + 2) * t, j * t:(j + 1) * t] = R
        rows, cols = (j + 2) * t, (j + 1) * t
        g = np.zeros(rows)
        g[:t] = g0
        y, *_ = np.linalg.lstsq(Hh[:rows, :cols], g, rcond=None)
        hist.append(float(np.linalg.norm(g - Hh[:rows, :cols] @ y)) / bnorm)
        if hist[-1] <= tol or j == max_blocks - 1:
            d = apply_Pinv(y @ V[:cols])
            break
    return d, hist
