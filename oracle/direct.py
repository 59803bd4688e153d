"""Direct (non-iterative) solutions of the unconstrained fixed-waypoint minimum-jerk/snap problem.

TEST INFRASTRUCTURE ONLY (part of oracle/): these are the plain definitions of the LIMIT that the
CADMM iteration must reach ("Optimality Conditions"; Eq. 2a-2c):

  closed_form_rest_to_rest  N = 1 textbook polynomials                                   (pin P1)
  dense_kkt                 min sum c_i'Q(T_i)c_i  s.t. waypoints, C^{s-1} continuity,
                            end states -- one dense KKT solve per dimension                (pin P3)
  banded_optimality         the optimality conditions themselves: degree 2s-1 pieces, C^{2s-2}
                            at junctions, s boundary rows at each end -- a square banded
                            2sN system per dimension (scipy.linalg.solve_banded)           (pin P4')

The last two are different formulations (a constrained minimisation vs. a linear system that never
mentions the cost) and are checked against each other and against the closed form in tests/.
Both work in normalised time (c^_k = c_k T^k) for conditioning and return coefficients in the
paper's basis (Eq. 18: ascending powers of t - t_{i-1}, physical seconds), shape [N][m][n].
"""
from __future__ import annotations

import math

import numpy as np
import scipy.linalg


def beta(n: int, k: int, t: float) -> np.ndarray:
    """[beta_k(t)]_j = j!/(j-k)! t^(j-k) (j >= k), else 0."""
    row = np.zeros(n)
    for j in range(k, n):
        row[j] = math.factorial(j) / math.factorial(j - k) * t ** (j - k)
    return row


def Q_unit(s: int) -> np.ndarray:
    """Q(1) = int_0^1 beta^(s) beta^(s)' dtau."""
    n = 2 * s
    Q = np.zeros((n, n))
    for j in range(s, n):
        for l in range(s, n):
            Q[j, l] = (math.factorial(j) / math.factorial(j - s)) * (math.factorial(l) / math.factorial(l - s)) \
                      / (j + l - 2 * s + 1)
    return Q


def closed_form_rest_to_rest(s: int, L: float, T: float):
    """N=1, rest to rest over length L in time T.  Returns (coeffs[n] in physical time, cost).

    jerk: sigma = L(10 tau^3 - 15 tau^4 + 6 tau^5),            cost 720 L^2 / T^5
    snap: sigma = L(35 tau^4 - 84 tau^5 + 70 tau^6 - 20 tau^7), cost 100800 L^2 / T^7
    """
    if s == 3:
        chat, cost = np.array([0, 0, 0, 10.0, -15.0, 6.0]), 720.0 * L * L / T ** 5
    elif s == 4:
        chat, cost = np.array([0, 0, 0, 0, 35.0, -84.0, 70.0, -20.0]), 100800.0 * L * L / T ** 7
    else:
        raise ValueError(s)
    return L * chat / T ** np.arange(2 * s), cost


def _to_physical(chat: np.ndarray, T: np.ndarray) -> np.ndarray:
    """chat [N][n][m] normalised-time coefficients -> [N][m][n] physical-time coefficients."""
    N, n, m = chat.shape
    scale = T[:, None] ** np.arange(n)[None, :]
    return np.transpose(chat / scale[:, :, None], (0, 2, 1)).copy()


def _end_states(s, m, start_derivs, end_derivs):
    sd = np.zeros((s - 1, m)) if start_derivs is None else np.asarray(start_derivs, dtype=np.float64)
    ed = np.zeros((s - 1, m)) if end_derivs is None else np.asarray(end_derivs, dtype=np.float64)
    return sd, ed


def dense_kkt(waypoints, durations, s, start_derivs=None, end_derivs=None):
    """Pin P3: dense KKT solve of the equality-constrained QP, per dimension."""
    P = np.asarray(waypoints, dtype=np.float64)
    T = np.asarray(durations, dtype=np.float64)
    N, m, n = T.size, P.shape[1], 2 * s
    sd, ed = _end_states(s, m, start_derivs, end_derivs)
    Q1 = Q_unit(s)
    nv = N * n
    Qbig = np.zeros((nv, nv))
    for i in range(N):
        Qbig[i * n:(i + 1) * n, i * n:(i + 1) * n] = Q1 * T[i] ** (1 - 2 * s)   # cost in normalised time
    rows, rhs = [], []
    def add(i_list, vecs, b):
        r = np.zeros(nv)
        for i, v in zip(i_list, vecs):
            r[i * n:(i + 1) * n] += v
        rows.append(r); rhs.append(np.asarray(b, dtype=np.float64))
    for i in range(N):                         # 2N position rows
        add([i], [beta(n, 0, 0.0)], P[i])
        add([i], [beta(n, 0, 1.0)], P[i + 1])
    for i in range(N - 1):                     # continuity of orders 1..s-1 (physical derivatives)
        for k in range(1, s):
            add([i, i + 1], [beta(n, k, 1.0) / T[i] ** k, -beta(n, k, 0.0) / T[i + 1] ** k], np.zeros(m))
    for k in range(1, s):                      # end states
        add([0], [beta(n, k, 0.0) / T[0] ** k], sd[k - 1])
        add([N - 1], [beta(n, k, 1.0) / T[N - 1] ** k], ed[k - 1])
    A = np.array(rows); B = np.array(rhs)      # [nc][nv], [nc][m]
    nc = A.shape[0]
    KKT = np.zeros((nv + nc, nv + nc))
    KKT[:nv, :nv] = 2 * Qbig; KKT[:nv, nv:] = A.T; KKT[nv:, :nv] = A
    sol = np.linalg.solve(KKT, np.vstack([np.zeros((nv, m)), B]))
    chat = sol[:nv].reshape(N, n, m)
    return _to_physical(chat, T)


def banded_optimality(waypoints, durations, s, start_derivs=None, end_derivs=None):
    """Pin P4': the optimality conditions as one square banded system per dimension."""
    P = np.asarray(waypoints, dtype=np.float64)
    T = np.asarray(durations, dtype=np.float64)
    N, m, n = T.size, P.shape[1], 2 * s
    sd, ed = _end_states(s, m, start_derivs, end_derivs)
    nv = N * n
    entries = []                               # (row, col, value)
    B = np.zeros((nv, m))
    r = 0
    def put(row, i, vec):
        for j in range(n):
            if vec[j] != 0.0:
                entries.append((row, i * n + j, vec[j]))
    put(r, 0, beta(n, 0, 0.0)); B[r] = P[0]; r += 1
    for k in range(1, s):                      # start derivatives, scaled by T^k to stay O(1)
        put(r, 0, beta(n, k, 0.0)); B[r] = sd[k - 1] * T[0] ** k; r += 1
    for i in range(N - 1):
        put(r, i, beta(n, 0, 1.0)); B[r] = P[i + 1]; r += 1          # end position of piece i
        for k in range(0, 2 * s - 1):          # C^{2s-2}: orders 0..2s-2 continuous (in units of T_i^k)
            put(r, i, beta(n, k, 1.0))
            put(r, i + 1, -beta(n, k, 0.0) * (T[i] / T[i + 1]) ** k)
            r += 1
    put(r, N - 1, beta(n, 0, 1.0)); B[r] = P[N]; r += 1
    for k in range(1, s):
        put(r, N - 1, beta(n, k, 1.0)); B[r] = ed[k - 1] * T[N - 1] ** k; r += 1
    assert r == nv
    lower = max(e[0] - e[1] for e in entries); upper = max(e[1] - e[0] for e in entries)
    ab = np.zeros((lower + upper + 1, nv))
    for (row, col, v) in entries:
        ab[upper + row - col, col] += v
    sol = scipy.linalg.solve_banded((lower, upper), ab, B)
    chat = sol.reshape(N, n, m)
    return _to_physical(chat, T)


def objective(coeffs, durations, s):
    """J = sum_i sum_d c' Q(T_i) c  for coeffs [N][m][n] in physical time (Eq. 2a, W = I)."""
    coeffs = np.asarray(coeffs, dtype=np.float64)
    T = np.asarray(durations, dtype=np.float64)
    n = 2 * s
    Q1 = Q_unit(s)
    J = 0.0
    for i in range(T.size):
        chat = coeffs[i] * (T[i] ** np.arange(n))[None, :]
        J += T[i] ** (1 - 2 * s) * np.einsum("da,ab,db->", chat, Q1, chat)
    return float(J)
