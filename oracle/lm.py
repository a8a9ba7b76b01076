"""CPU ORACLE (test infrastructure, NOT the product) -- O10: the moment-damped LM solve.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs may import this module.  It never
imports the CUDA package and shares no code with it.  Plain numpy, fp64, one Gaussian's systems written out
entry by entry (vectorised over the Gaussians only).

What it computes (Sec. 3.9 Eq. 14; App. A Eq. 19; Alg. 1 step 9):

  per Gaussian, two parameter blocks
      geometry    g in R^10 = (position 3, scale 3, rotation 4)
      appearance  a in R^4  = (RGB DC 3, opacity 1)
  each solved independently:
      (J^T J + diag(sqrt(v) + eps)) Delta = -m                                   (Eq. 14 = Eq. 19 left)
  by Cholesky decomposition, and every higher SH coefficient by Adam:
      Delta = -eta m_hat / (sqrt(v_hat) + eps)                                    (Eq. 19 right)

Readings (R30-R35; the paper leaves these open):
  R31  J_g ("the local Jacobian estimated from the accumulated gradients"): the V x d matrix whose
       row i is this Gaussian's gradient of the block from view i of the iteration's V views (Alg. 1 step 2
       selects K_t views per iteration), so J^T J = sum_i g_i g_i^T.            PARITY UNPINNED (a reading, no
       printed example or definition to hold it against); everything after J is pinned (tests/test_lm_pins.py).
  R32  the accumulated gradient is gbar = sum_i g_i; the Adam moments are updated with it BEFORE the solve,
       m <- beta1 m + (1 - beta1) gbar,  v <- beta2 v + (1 - beta2) gbar^2; Eq. 14 takes m and v as printed (no bias
       correction); Eq. 19 right takes m_hat = m / (1 - beta1^t), v_hat = v / (1 - beta2^t), t >= 1 the iteration.
  R33  one eps for both halves of Eq. 19 (the paper prints the same symbol).
  R34  `update` (nullable mask): a Gaussian with update == 0 received no gradient this iteration; its moments
       are left unchanged and its Delta is 0 (the sparse-Adam convention of Tab. 5).
  R35  Alg. 1 step 10 G <- G + Delta G is `apply`.
  R36  `view_touched` (nullable [V, N] mask): view i's gradient of Gaussian n counts as ZERO where the mask is 0 (the
       sparse raster backward left those rows unwritten, whatever they hold); a Gaussian touched in no view is
       treated like update == 0.  Pure input handling: the arithmetic after it is unchanged.
Layouts mirror the parameters: a "parameter set" is a dict with keys means3D [N,3], scales [N,3], quats [N,4],
opacities [N], sh [N,K,3]; gradients carry a leading view axis [V, ...]; moments m / v are parameter sets, the
moments of the RGB DC live in sh[:, 0, :].
"""
from __future__ import annotations

import numpy as np

KEYS = ("means3D", "scales", "quats", "opacities", "sh")


def cholesky_solve(A: np.ndarray, b: np.ndarray) -> np.ndarray:
    """Solve A x = b for a batch of symmetric positive definite A [N,d,d], b [N,d] by Cholesky decomposition
    A = L L^T (Cholesky-Banachiewicz, row by row), forward substitution L y = b, back substitution L^T x = y.
    PAPER.md:239 "Each local formulation is solved via Cholesky decomposition"."""
    A = np.asarray(A, np.float64)
    b = np.asarray(b, np.float64)
    n, d = b.shape
    L = np.zeros((n, d, d))
    for i in range(d):
        for j in range(i + 1):
            s = A[:, i, j].copy()
            for k in range(j):
                s -= L[:, i, k] * L[:, j, k]
            if i == j:
                if np.any(s <= 0.0):
                    raise np.linalg.LinAlgError("matrix not positive definite")
                L[:, i, i] = np.sqrt(s)
            else:
                L[:, i, j] = s / L[:, j, j]
    y = np.zeros((n, d))
    for i in range(d):
        s = b[:, i].copy()
        for k in range(i):
            s -= L[:, i, k] * y[:, k]
        y[:, i] = s / L[:, i, i]
    x = np.zeros((n, d))
    for i in range(d - 1, -1, -1):
        s = y[:, i].copy()
        for k in range(i + 1, d):
            s -= L[:, k, i] * x[:, k]
        x[:, i] = s / L[:, i, i]
    return x


def lm_system(J: np.ndarray, v: np.ndarray, eps: float) -> np.ndarray:
    """A = J^T J + diag(sqrt(v) + eps) of Eq. 14 for a batch: J [N,V,d] (rows = per-view gradients, R31), v [N,d]."""
    J = np.asarray(J, np.float64)
    n, V, d = J.shape
    A = np.zeros((n, d, d))
    for a in range(d):
        for c in range(d):
            for i in range(V):
                A[:, a, c] += J[:, i, a] * J[:, i, c]
    for a in range(d):
        A[:, a, a] += np.sqrt(v[:, a]) + eps
    return A


def moments(m: np.ndarray, v: np.ndarray, gbar: np.ndarray, beta1: float, beta2: float):
    """Adam moment update with the accumulated gradient (R32)."""
    return beta1 * m + (1.0 - beta1) * gbar, beta2 * v + (1.0 - beta2) * gbar * gbar


def _block(ps, geometry: bool) -> np.ndarray:
    """[..., N, d]: the geometry (d = 10) or appearance (d = 4) block of a parameter set."""
    if geometry:
        return np.concatenate([ps["means3D"], ps["scales"], ps["quats"]], axis=-1)
    return np.concatenate([ps["sh"][..., 0, :], ps["opacities"][..., None]], axis=-1)


def _unblock(out, x: np.ndarray, geometry: bool) -> None:
    if geometry:
        out["means3D"][...] = x[:, 0:3]
        out["scales"][...] = x[:, 3:6]
        out["quats"][...] = x[:, 6:10]
    else:
        out["sh"][:, 0, :] = x[:, 0:3]
        out["opacities"][...] = x[:, 3]


def lm_solve(grads, m, v, update=None, beta1=0.9, beta2=0.999, eps=1e-8, eta_sh=2.5e-3 / 20.0, t=1, params=None,
             view_touched=None):
    """One call of Alg. 1 step 9 (and step 10 when `params` is given).

    grads: parameter set with a leading view axis [V, N, ...]; m, v: parameter sets [N, ...] (not modified).
    Returns (delta, m_new, v_new, params_new or None), all fp64 parameter sets."""
    g = {k: np.asarray(grads[k], np.float64) for k in KEYS}
    m0 = {k: np.asarray(m[k], np.float64) for k in KEYS}
    v0 = {k: np.asarray(v[k], np.float64) for k in KEYS}
    V, N = g["opacities"].shape
    upd = np.ones(N, bool) if update is None else (np.asarray(update) != 0)
    if view_touched is not None:                            # R36
        vt = np.asarray(view_touched) != 0
        assert vt.shape == (V, N)
        for k in KEYS:
            mask = vt.reshape(vt.shape + (1,) * (g[k].ndim - 2))
            g[k] = np.where(mask, g[k], 0.0)
        upd = upd & vt.any(axis=0)
    m1 = {k: m0[k].copy() for k in KEYS}
    v1 = {k: v0[k].copy() for k in KEYS}
    delta = {k: np.zeros_like(m0[k]) for k in KEYS}

    # ---- the two LM blocks (Eq. 14) ----
    for geometry in (True, False):
        J = np.moveaxis(_block(g, geometry), 0, 1)         # [N, V, d]: row i = view i's gradient (R31)
        gbar = J.sum(axis=1)                                # accumulated gradient (R32)
        mb, vb = moments(_block(m0, geometry), _block(v0, geometry), gbar, beta1, beta2)
        A = lm_system(J, vb, eps)
        x = cholesky_solve(A, -mb)
        keep = ~upd
        x[keep] = 0.0
        mb[keep] = _block(m0, geometry)[keep]
        vb[keep] = _block(v0, geometry)[keep]
        _unblock(delta, x, geometry)
        _unblock(m1, mb, geometry)
        _unblock(v1, vb, geometry)

    # ---- higher SH coefficients: Adam (Eq. 19 right) ----
    K = g["sh"].shape[2]
    if K > 1:
        gbar = g["sh"][:, :, 1:, :].sum(axis=0)
        ms, vs = moments(m0["sh"][:, 1:, :], v0["sh"][:, 1:, :], gbar, beta1, beta2)
        m_hat = ms / (1.0 - beta1 ** t)
        v_hat = vs / (1.0 - beta2 ** t)
        d = -eta_sh * m_hat / (np.sqrt(v_hat) + eps)
        delta["sh"][upd, 1:, :] = d[upd]
        m1["sh"][upd, 1:, :] = ms[upd]
        v1["sh"][upd, 1:, :] = vs[upd]

    new = None
    if params is not None:                                  # Alg. 1 step 10
        new = {k: np.asarray(params[k], np.float64) + delta[k] for k in KEYS}
    return delta, m1, v1, new
