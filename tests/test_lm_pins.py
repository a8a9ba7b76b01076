"""Pins of the LM-solve oracle (oracle/lm.py, O10) against things other than itself:
numpy's LU solver, closed forms (Sherman-Morrison, J = 0, the first Adam step), torch.optim.Adam as a library
routine, invariants (view order, block independence, mask).  CPU only.

What stays unpinned is the READING of J (R31: rows = per-view gradients); every step after J is held here."""
import numpy as np
import pytest

import workloads
from oracle import lm

B1, B2, EPS, ETA = 0.9, 0.999, 1e-8, 1.25e-4


def _rand_spd_inputs(rng, n, V, d, scale=1.0):
    J = rng.standard_normal((n, V, d)) * scale
    v = rng.random((n, d)) * scale ** 2
    m = rng.standard_normal((n, d)) * scale
    return J, v, m


@pytest.mark.parametrize("d", [4, 10])
@pytest.mark.parametrize("V", [1, 2, 5, 12])
def test_cholesky_matches_numpy_solve(d, V):
    """the 10 x 10 and 4 x 4 systems of Eq. 14 against numpy.linalg.solve (LAPACK LU)."""
    rng = np.random.default_rng(100 * d + V)
    J, v, m = _rand_spd_inputs(rng, 64, V, d)
    A = lm.lm_system(J, v, EPS)
    x = lm.cholesky_solve(A, -m)
    ref = np.stack([np.linalg.solve(A[i], -m[i]) for i in range(len(A))])
    np.testing.assert_allclose(x, ref, rtol=1e-9, atol=1e-12)
    # residual of Eq. 14
    r = np.einsum("nij,nj->ni", A, x) + m
    assert np.abs(r).max() < 1e-10


def test_system_is_the_definition():
    """lm_system against J^T J + diag(sqrt(v) + eps) formed with numpy's matmul."""
    rng = np.random.default_rng(1)
    J, v, _ = _rand_spd_inputs(rng, 16, 3, 10)
    A = lm.lm_system(J, v, 1e-3)
    for i in range(16):
        ref = J[i].T @ J[i] + np.diag(np.sqrt(v[i]) + 1e-3)
        np.testing.assert_allclose(A[i], ref, rtol=1e-13, atol=1e-15)
        assert np.array_equal(A[i], A[i].T)


def test_spd_for_any_J():
    """sqrt(v) + eps > 0 makes the system positive definite whatever J is: rank-deficient, zero, huge, repeated rows.
    The Cholesky must go through and all eigenvalues are >= min(sqrt(v)) + eps."""
    rng = np.random.default_rng(2)
    n, d = 32, 10
    cases = [np.zeros((n, 1, d)), rng.standard_normal((n, 1, d)) * 1e3,
             np.repeat(rng.standard_normal((n, 1, d)), 4, axis=1),
             rng.standard_normal((n, 3, d)) * np.array([1e-6, 1, 1e4])[None, :, None]]
    for J in cases:
        v = rng.random((n, d)) * 1e-4
        v[:, 3] = 0.0  # a parameter that never saw a gradient: damping eps alone
        A = lm.lm_system(J, v, EPS)
        x = lm.cholesky_solve(A, -np.ones((n, d)))
        assert np.all(np.isfinite(x))
        for i in range(n):
            assert np.linalg.eigvalsh(A[i]).min() >= (np.sqrt(v[i]).min() + EPS) * (1 - 1e-9) - 1e-12 * np.abs(A[i]).max()


def test_J_zero_gives_damped_moment_step():
    """J = 0  =>  Delta = -m / (sqrt(v) + eps) elementwise (a diagonal system)."""
    rng = np.random.default_rng(3)
    _, v, m = _rand_spd_inputs(rng, 20, 1, 10)
    x = lm.cholesky_solve(lm.lm_system(np.zeros((20, 2, 10)), v, EPS), -m)
    np.testing.assert_allclose(x, -m / (np.sqrt(v) + EPS), rtol=1e-12)


@pytest.mark.parametrize("d", [4, 10])
def test_single_view_is_sherman_morrison(d):
    """V = 1: (D + g g^T)^-1 m = D^-1 m - D^-1 g (g^T D^-1 m) / (1 + g^T D^-1 g), D = diag(sqrt(v) + eps)."""
    rng = np.random.default_rng(4 + d)
    J, v, m = _rand_spd_inputs(rng, 50, 1, d)
    x = lm.cholesky_solve(lm.lm_system(J, v, EPS), -m)
    g = J[:, 0, :]
    Dinv = 1.0 / (np.sqrt(v) + EPS)
    ref = -(Dinv * m - Dinv * g * ((g * Dinv * m).sum(1) / (1.0 + (g * Dinv * g).sum(1)))[:, None])
    np.testing.assert_allclose(x, ref, rtol=1e-9, atol=1e-12)


def _as64(ps):
    return {k: np.asarray(a, np.float64) for k, a in ps.items()}


def test_full_call_blocks_and_layout():
    """lm_solve end to end against numpy.linalg.solve on hand-assembled blocks: the geometry block is (means, scales,
    quats), the appearance block (sh DC rgb, opacity); moments follow R32; results land in the
    parameter layouts."""
    grads, m, v, upd = workloads.lm_state(0, 40, 3, views=3)
    upd[:] = 1
    delta, m1, v1, _ = lm.lm_solve(grads, m, v, None, B1, B2, EPS, ETA, t=7)
    g, m, v = _as64(grads), _as64(m), _as64(v)
    for i in range(40):
        Jg = np.concatenate([g["means3D"][:, i], g["scales"][:, i], g["quats"][:, i]], axis=1)   # [V, 10]
        Ja = np.concatenate([g["sh"][:, i, 0, :], g["opacities"][:, i, None]], axis=1)            # [V, 4]
        for J, mo, vo, got in (
                (Jg, np.concatenate([m["means3D"][i], m["scales"][i], m["quats"][i]]),
                 np.concatenate([v["means3D"][i], v["scales"][i], v["quats"][i]]),
                 np.concatenate([delta["means3D"][i], delta["scales"][i], delta["quats"][i]])),
                (Ja, np.concatenate([m["sh"][i, 0], [m["opacities"][i]]]),
                 np.concatenate([v["sh"][i, 0], [v["opacities"][i]]]),
                 np.concatenate([delta["sh"][i, 0], [delta["opacities"][i]]]))):
            gb = J.sum(0)
            mn = B1 * mo + (1 - B1) * gb
            vn = B2 * vo + (1 - B2) * gb ** 2
            ref = np.linalg.solve(J.T @ J + np.diag(np.sqrt(vn) + EPS), -mn)
            np.testing.assert_allclose(got, ref, rtol=1e-9, atol=1e-14)
    gb = g["means3D"].sum(0)
    np.testing.assert_allclose(m1["means3D"], B1 * m["means3D"] + (1 - B1) * gb, rtol=1e-14)
    np.testing.assert_allclose(v1["quats"], B2 * v["quats"] + (1 - B2) * g["quats"].sum(0) ** 2, rtol=1e-14)


def test_adam_branch_first_step_closed_form():
    """Eq. 19 right, t = 1 from zero moments: m_hat = g, v_hat = g^2  =>  Delta = -eta g / (|g| + eps)."""
    grads, m, v, upd = workloads.lm_state(1, 30, 2, views=1, warm=False)
    delta, _, _, _ = lm.lm_solve(grads, m, v, None, B1, B2, EPS, ETA, t=1)
    g = np.asarray(grads["sh"][0, :, 1:, :], np.float64)
    np.testing.assert_allclose(delta["sh"][:, 1:, :], -ETA * g / (np.abs(g) + EPS), rtol=1e-9, atol=1e-18)


def test_adam_branch_and_moments_match_torch_adam():
    """Five iterations of the SH branch against torch.optim.Adam (a library routine): same parameter trajectory,
    and the oracle's moments equal torch's exp_avg / exp_avg_sq -- also for the LM blocks' moments, which are the
    same Adam recursion fed with the accumulated gradient (R32)."""
    import torch
    n, D = 12, 3
    K = (D + 1) ** 2
    rng = np.random.default_rng(5)
    p_sh = rng.standard_normal((n, K, 3))
    p_mu = rng.standard_normal((n, 3))
    tp_sh = torch.tensor(p_sh, dtype=torch.float64, requires_grad=True)
    tp_mu = torch.tensor(p_mu, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([tp_sh, tp_mu], lr=ETA, betas=(B1, B2), eps=EPS)
    _, m, v, _ = workloads.lm_state(6, n, D, views=1, warm=False)
    m, v = _as64(m), _as64(v)
    params = {"means3D": p_mu.copy(), "scales": np.ones((n, 3)), "quats": np.ones((n, 4)), "opacities": np.ones(n),
              "sh": p_sh.copy()}
    for t in range(1, 6):
        grads, _, _, _ = workloads.lm_state(10 + t, n, D, views=2, p_update=1.0)
        delta, m, v, params = lm.lm_solve(grads, m, v, None, B1, B2, EPS, ETA, t=t, params=params)
        tp_sh.grad = torch.tensor(np.asarray(grads["sh"], np.float64).sum(0))
        tp_mu.grad = torch.tensor(np.asarray(grads["means3D"], np.float64).sum(0))
        opt.step()
        np.testing.assert_allclose(params["sh"][:, 1:, :], tp_sh.detach().numpy()[:, 1:, :], rtol=1e-10, atol=1e-14)
        st = opt.state[tp_sh]
        np.testing.assert_allclose(m["sh"], st["exp_avg"].numpy(), rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(v["sh"], st["exp_avg_sq"].numpy(), rtol=1e-12, atol=1e-300)
        st = opt.state[tp_mu]
        np.testing.assert_allclose(m["means3D"], st["exp_avg"].numpy(), rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(v["means3D"], st["exp_avg_sq"].numpy(), rtol=1e-12, atol=1e-300)
    # the DC band is NOT an Adam step: it belongs to the appearance LM block
    assert np.abs(params["sh"][:, 0, :] - tp_sh.detach().numpy()[:, 0, :]).max() > 1e-6


def test_invariants_view_order_block_independence_mask():
    grads, m, v, upd = workloads.lm_state(2, 64, 3, views=4)
    d0, m0, v0, _ = lm.lm_solve(grads, m, v, upd, B1, B2, EPS, ETA, t=3)
    # J^T J and the accumulated gradient do not depend on the order of the views
    perm = {k: a[[2, 0, 3, 1]] for k, a in grads.items()}
    d1, _, _, _ = lm.lm_solve(perm, m, v, upd, B1, B2, EPS, ETA, t=3)
    for k in lm.KEYS:
        np.testing.assert_allclose(d1[k], d0[k], rtol=1e-9, atol=1e-16)
    # the blocks are solved independently: changing the appearance gradients leaves the geometry update alone, and
    # changing a higher SH gradient leaves both LM blocks alone
    g2 = {k: a.copy() for k, a in grads.items()}
    g2["opacities"] *= 3.0
    g2["sh"][:, :, 0, :] += 0.01
    g2["sh"][:, :, 5, :] -= 0.02
    d2, _, _, _ = lm.lm_solve(g2, m, v, upd, B1, B2, EPS, ETA, t=3)
    for k in ("means3D", "scales", "quats"):
        assert np.array_equal(d2[k], d0[k])
    assert np.abs(d2["opacities"] - d0["opacities"]).max() > 0
    g3 = {k: a.copy() for k, a in grads.items()}
    g3["sh"][:, :, 5, :] -= 0.02
    d3, _, _, _ = lm.lm_solve(g3, m, v, upd, B1, B2, EPS, ETA, t=3)
    assert np.array_equal(d3["opacities"], d0["opacities"]) and np.array_equal(d3["sh"][:, 0], d0["sh"][:, 0])
    # R34: masked Gaussians keep their moments and do not move
    off = upd == 0
    assert off.any()
    for k in lm.KEYS:
        assert not d0[k][off].any()
        assert np.array_equal(m0[k][off], np.asarray(m[k], np.float64)[off])
        assert np.array_equal(v0[k][off], np.asarray(v[k], np.float64)[off])
        assert d0[k][~off].any()
    # the geometry block couples its parameters: with J != 0 the update differs from the diagonal (J = 0) step
    gb = np.asarray(grads["means3D"], np.float64).sum(0)
    mn = B1 * np.asarray(m["means3D"], np.float64) + (1 - B1) * gb
    vn = B2 * np.asarray(v["means3D"], np.float64) + (1 - B2) * gb ** 2
    diag_step = -mn / (np.sqrt(vn) + EPS)
    on = ~off
    assert np.abs(d0["means3D"][on] - diag_step[on]).max() > 1e-3 * np.abs(diag_step[on]).max()


def test_apply_is_step_10():
    grads, m, v, upd = workloads.lm_state(3, 16, 1, views=1)
    params = {k: np.asarray(a[0], np.float64) * 0 + 1.5 for k, a in grads.items()}
    d, _, _, new = lm.lm_solve(grads, m, v, upd, B1, B2, EPS, ETA, t=2, params=params)
    for k in lm.KEYS:
        assert np.array_equal(new[k], params[k] + d[k])


def test_sh_degree_0_has_no_adam_branch():
    grads, m, v, upd = workloads.lm_state(4, 8, 0, views=2)
    d, m1, v1, _ = lm.lm_solve(grads, m, v, None, B1, B2, EPS, ETA, t=1)
    assert d["sh"].shape == (8, 1, 3) and np.all(np.isfinite(d["sh"]))


def test_view_touched_is_zeroed_rows():
    """R36: per-view masks are the same as zero gradient rows (whatever the masked rows hold) and a Gaussian touched in no
    view keeps its moments."""
    grads, m, v, upd = workloads.lm_state(7, 50, 2, views=3, p_update=1.0)
    rng = np.random.default_rng(8)
    vt = (rng.random((3, 50)) < 0.6).astype(np.int32)
    vt[:, 0] = 0                                            # touched in no view
    zeroed = {k: np.where(vt.reshape(vt.shape + (1,) * (a.ndim - 2)) != 0, a, 0.0).astype(np.float32) for k, a in grads.items()}
    garbage = {k: np.where(vt.reshape(vt.shape + (1,) * (a.ndim - 2)) != 0, a, np.nan).astype(np.float32) for k, a in grads.items()}
    d0, m0, v0, _ = lm.lm_solve(zeroed, m, v, vt.any(0).astype(np.int32), B1, B2, EPS, ETA, t=2)
    d1, m1, v1, _ = lm.lm_solve(garbage, m, v, None, B1, B2, EPS, ETA, t=2, view_touched=vt)
    for k in lm.KEYS:
        assert np.array_equal(d0[k], d1[k]) and np.array_equal(m0[k], m1[k]) and np.array_equal(v0[k], v1[k])
        assert not d1[k][0].any() and np.array_equal(m1[k][0], np.asarray(m[k], np.float64)[0])
