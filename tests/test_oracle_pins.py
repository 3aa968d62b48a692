"""Pins of the fp64 oracle against what the paper and the mathematics fix (no GPU, no CUDA code).

The paper prints no worked numeric example for this path, so every pin is a
closed form, an invariant, a special case reducing to a textbook routine, or brute force:

  P1  finite-difference Jacobians of every factor and of the re-anchoring map
  P2  noise-free inputs: zero GN step, estimates == ground truth (all factor types)
  P3  pure-translation odometry chain: closed-form covariance / log-det, through marginalization
      (values also stored in tests/golden/chain_logdet.txt, cited there)
  P4  odometry-only runs (all of BASELINE config 0): dead reckoning + EKF covariance recursion
  P5  noise-free runs with loop closures / landmarks: fixed-lag marginal == last block of the
      inverse of the GLOBAL full-trajectory Hessian (tests/fullbatch.py, independent numpy code)
  P6  linear-Gaussian mode, arbitrary noise: fixed-lag mean and covariance == brute-force full-batch
      least squares (pins the gradient path: b sign, Lam d + g, g' of the Schur complement)
  P7  invariants: covariances SPD and symmetric, prior PSD, log-det monotone on odometry-only runs,
      Gauss-Newton decreases the cost, constant problem size
  P8  noisy nonlinear runs: loose agreement with full-batch GN, NEES ~ chi^2_3
"""
import os

import numpy as np
import pytest

import oracle
from oracle import Oracle
from harness import synth
from tests import fullbatch
from tests.helpers import drive, rb_inputs, step_inputs

SIG = np.array(oracle.DEFAULT_SIGMAS)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def fd_jac(f, x, eps=1e-6):
    x = np.asarray(x, float)
    f0 = f(x)
    J = np.zeros((f0.size, x.size))
    for i in range(x.size):
        xp, xm = x.copy(), x.copy()
        xp[i] += eps
        xm[i] -= eps
        J[:, i] = (f(xp) - f(xm)) / (2 * eps)
    return J


# ----------------------------------------------------------------------------- P1
def test_between_factor_jacobians_fd():
    rng = np.random.default_rng(1)
    for _ in range(20):
        ei, ej = rng.normal(size=3), rng.normal(size=3)
        z = rng.normal(size=3) * 0.3
        r, Ji, Jj = oracle.between_factor(ei, ej, z)
        Ji_fd = fd_jac(lambda x: oracle.between_factor(x, ej, z)[0], ei)
        Jj_fd = fd_jac(lambda x: oracle.between_factor(ei, x, z)[0], ej)
        assert np.allclose(Ji, Ji_fd, atol=1e-7)
        assert np.allclose(Jj, Jj_fd, atol=1e-7)
        # frame case: pose i is the identity, not a variable
        r0, Ji0, Jj0 = oracle.between_factor(ei, ej, z, i_is_frame=True)
        assert np.allclose(r0, oracle.between_factor(np.zeros(3), ej, z)[0])
        assert np.allclose(Ji0, 0) and np.allclose(Jj0, np.eye(3))
    # definition (R2): z = between(p, q) gives r = 0
    p, q = np.array([0.3, -0.2, 0.7]), np.array([1.0, 0.5, -0.4])
    z = synth.between(p[:, None], q[:, None])[:, 0]
    assert np.allclose(oracle.between_factor(p, q, z)[0], 0, atol=1e-15)


def test_rb_factor_jacobians_fd():
    rng = np.random.default_rng(2)
    for _ in range(20):
        a = rng.normal(size=3) * [5, 5, 1]
        ek = rng.normal(size=3)
        x = synth.compose(a[:, None], ek[:, None])[:, 0]                 # global observing pose
        gl = x[:2] + rng.uniform(0.5, 8.0) * np.array([np.cos(1.3), np.sin(1.3)]) + rng.normal(size=2) * 0.1
        z = np.array([rng.uniform(0.5, 8), rng.uniform(-3, 3)])
        r, Ja, Jp, Jg = oracle.rb_factor(a, ek, gl, z)
        assert np.allclose(Ja, fd_jac(lambda q: oracle.rb_factor(q, ek, gl, z)[0], a), atol=1e-6)
        assert np.allclose(Jp, fd_jac(lambda q: oracle.rb_factor(a, q, gl, z)[0], ek), atol=1e-6)
        assert np.allclose(Jg, fd_jac(lambda q: oracle.rb_factor(a, ek, q, z)[0], gl), atol=1e-6)
        # the anchor slot observes from x = a: no e block
        r0, Ja0, Jp0, Jg0 = oracle.rb_factor(a, ek, gl, z, k_is_frame=True)
        assert np.allclose(r0, oracle.rb_factor(a, np.zeros(3), gl, z)[0]) and np.allclose(Jp0, 0)
        assert np.allclose(Ja0, fd_jac(lambda q: oracle.rb_factor(q, ek, gl, z, True)[0], a), atol=1e-6)
    # definition (R4): a landmark at range 2, bearing 0.5 from the global pose (1,2,0.3)
    p = np.array([1.0, 2.0, 0.3])
    l = p[:2] + 2.0 * np.array([np.cos(0.8), np.sin(0.8)])
    assert np.allclose(oracle.rb_factor(p, np.zeros(3), l, [2.0, 0.5], True)[0], 0, atol=1e-14)
    a, e = np.array([0.4, -0.3, 0.9]), np.array([0.2, 0.1, -0.5])
    x = synth.compose(a[:, None], e[:, None])[:, 0]
    l = x[:2] + 3.0 * np.array([np.cos(x[2] - 0.7), np.sin(x[2] - 0.7)])
    assert np.allclose(oracle.rb_factor(a, e, l, [3.0, -0.7])[0], 0, atol=1e-14)


def _random_window(W=6, L=3, seed=3):
    rng = np.random.default_rng(seed)
    o = Oracle(W, L)
    o.reset([0.5, -1.0, 0.8])
    if L:
        o.observe_first(np.ones(L, np.int32), np.stack([rng.uniform(1, 5, L), rng.uniform(-3, 3, L)], 1))
    for k in range(1, W):
        o.push(rng.normal(size=3) * [0.3, 0.1, 0.4], lc_back=(k if k % 2 == 0 else 0), lc_meas=rng.normal(size=3) * 0.2,
               rb_valid=np.ones(L, np.int32) if L else None,
               rb_meas=np.stack([rng.uniform(1, 5, L), rng.uniform(-3, 3, L)], 1) if L else None)
    v = o.state()
    o.set_state(v + rng.normal(size=v.size) * 0.05)
    return o


def test_reanchor_jacobian_fd():
    o = _random_window()
    v = o.state()
    M = o.reanchor_jac()
    M_fd = fd_jac(o.reanchor_map, v)
    assert np.allclose(M, M_fd, atol=1e-6)
    # re-anchoring preserves every global quantity: a' (+) e'_k == a (+) e_k
    u = o.reanchor_map(v)
    a2 = u[:3]
    for k in range(2, o.W):
        g_old = synth.compose(v[:3, None], v[3 * k:3 * k + 3, None])[:, 0]
        g_new = synth.compose(a2[:, None], u[3 * k:3 * k + 3, None])[:, 0]
        assert np.allclose(g_old, g_new, atol=1e-12)
    assert np.array_equal(u[3 * o.W:], v[3 * o.W:])        # landmarks are global: untouched (R17b)


def test_gradient_and_hessian_of_cost_fd():
    """b == -grad(cost) exactly; H == Gauss-Newton Hessian (J'Omega J + Lam): checked through the
    cost function by finite differences (H only approximately: GN drops second-order terms, so use a
    state at which all residuals vanish)."""
    o = _random_window(W=5, L=2, seed=4)
    v = o.state()
    H, b = o.assemble()

    def cost_at(x):
        o.set_state(x)
        return np.array([o.cost()])

    g_fd = fd_jac(cost_at, v, eps=1e-6)[0]
    o.set_state(v)
    assert np.allclose(-b, g_fd, rtol=1e-5, atol=1e-4 * np.abs(b).max())
    assert np.allclose(H, H.T)
    assert np.linalg.eigvalsh(H).min() > 0


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("W,L,p_lc,T", [(10, 0, 0.0, 40), (8, 0, 0.5, 60), (6, 5, 0.3, 40), (20, 24, 0.0, 45)])
def test_noise_free_exact_recovery(W, L, p_lc, T):
    cfg = synth.Config("nf", N=3, W=W, L=L, iters=3, T=T, p_lc=p_lc, seed=5)
    data = synth.generate(cfg, noise_scale=0.0, dtype=np.float64)
    for env in range(cfg.N):
        recs = drive(Oracle(W, L), data, env, iters=2)
        for rec in recs:
            assert rec["step"] < 1e-11, (rec["t"], rec["step"])
            c = rec["count"]
            gt = data["gt"][rec["t"] - c + 1: rec["t"] + 1, :, env]
            err = rec["poses"][:c] - gt
            err[:, 2] = fullbatch.wrap(err[:, 2])
            assert np.abs(err).max() < 1e-10


# ----------------------------------------------------------------------------- P3
def chain_cov_closed_form(k, d, P0, Q):
    px, py, pt = P0
    qx, qy, qt = Q
    S = np.zeros((3, 3))
    S[0, 0] = px + k * qx
    S[1, 1] = py + k * k * d * d * pt + k * qy + d * d * qt * (k - 1) * k * (2 * k - 1) / 6.0
    S[1, 2] = S[2, 1] = k * d * pt + d * qt * k * (k - 1) / 2.0
    S[2, 2] = pt + k * qt
    return S


@pytest.mark.parametrize("W", [2, 3, 5, 12])
def test_pure_translation_chain_closed_form(W):
    d = 0.2
    P0, Q = SIG[0:3] ** 2, SIG[3:6] ** 2
    o = Oracle(W, 0)
    o.reset()
    golden = {}
    with open(os.path.join(GOLDEN, "chain_logdet.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, val = line.split()
                golden[int(k)] = float(val)
    for k in range(1, 41):
        o.push([d, 0.0, 0.0])
        assert o.solve(3) < 1e-12
        S, ld = o.cov()
        ref = chain_cov_closed_form(k, d, P0, Q)
        assert np.allclose(S, ref, rtol=1e-9, atol=1e-15), (k, S, ref)
        assert abs(ld - np.log(np.linalg.det(ref))) < 1e-9
        if k in golden:
            assert abs(ld - golden[k]) < 5e-7, (k, ld, golden[k])
        if o.count == W:
            o.marginalize()


# ----------------------------------------------------------------------------- P4
def ekf_recursion(odom, P0, Q):
    """Dead reckoning + EKF prediction covariance; independent of any SLAM code."""
    x = np.zeros(3)
    S = np.diag(P0)
    out = []
    for z in odom:
        c, s = np.cos(x[2]), np.sin(x[2])
        xn = np.array([x[0] + c * z[0] - s * z[1], x[1] + s * z[0] + c * z[1], x[2] + z[2]])
        F = np.array([[1, 0, -(xn[1] - x[1])], [0, 1, xn[0] - x[0]], [0, 0, 1.0]])
        R = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1.0]])
        S = F @ S @ F.T + R @ np.diag(Q) @ R.T
        x = xn
        out.append((x.copy(), S.copy()))
    return out


def test_config0_equals_ekf_recursion():
    cfg = synth.CONFIGS[0]
    data = synth.generate(cfg)          # float32 inputs: exactly what the library and bench consume
    res = oracle.run_batch(data, cfg.iters)
    assert res["bad"] == 0
    assert res["step"].max() < 1e-10    # dead reckoning is already the optimum of an odometry tree
    for env in range(cfg.N):
        ref = ekf_recursion(data["odom"][:, :, env].astype(np.float64), SIG[0:3] ** 2, SIG[3:6] ** 2)
        prev = -np.inf
        for t, (x, S) in enumerate(ref):
            c = min(t + 2, cfg.W)
            got = res["poses"][t, env, c - 1]
            err = got - x
            err[2] = fullbatch.wrap(err[2])
            assert np.abs(err).max() < 1e-10 * max(1.0, np.abs(x).max())
            assert np.allclose(res["cov"][t, env], S, rtol=1e-8, atol=1e-14)
            ld = np.log(np.linalg.det(S))
            assert abs(res["logdet"][t, env] - ld) < 1e-8
            assert res["logdet"][t, env] >= prev - 1e-9   # P7: non-decreasing on odometry-only runs
            prev = res["logdet"][t, env]


# ----------------------------------------------------------------------------- P5
@pytest.mark.parametrize("W,L,p_lc,T", [(6, 0, 0.5, 40), (5, 6, 0.4, 30), (10, 24, 0.0, 30)])
def test_noise_free_fixed_lag_equals_global_full_batch(W, L, p_lc, T):
    cfg = synth.Config("nf", N=2, W=W, L=L, iters=2, T=T, p_lc=p_lc, seed=7)
    data = synth.generate(cfg, noise_scale=0.0, dtype=np.float64)
    for env in range(cfg.N):
        fb = fullbatch.FullBatch(SIG, L)
        if L:
            fb.observe_first(*rb_inputs(data, 0, env))
        o = Oracle(W, L)
        o.reset()
        if L:
            o.observe_first(*rb_inputs(data, 0, env))
        for t in range(1, T + 1):
            odom, back, zlc, valid, zrb = step_inputs(data, t, env)
            fb.push(odom, back, zlc, valid, zrb)
            o.push(odom, back, zlc, valid, zrb)
            o.solve(2)
            S, ld = o.cov()
            ref = fb.last_cov()
            scale = np.sqrt(np.outer(np.diag(ref), np.diag(ref)))
            assert np.abs(S - ref).max() / scale.max() < 1e-8 and np.all(np.abs(S - ref) <= 1e-7 * scale), (t, S, ref)
            assert abs(ld - np.log(np.linalg.det(ref))) < 1e-7
            if o.count == W:
                o.marginalize()


# ----------------------------------------------------------------------------- P6
def test_linear_gaussian_fixed_lag_equals_brute_force_full_batch():
    rng = np.random.default_rng(11)
    W, T = 4, 25
    P0 = SIG[0:3] ** 2
    om_odo, om_lc = 1.0 / SIG[3:6] ** 2, 1.0 / SIG[6:9] ** 2
    x0 = np.array([0.3, -0.2, 0.1])
    o = Oracle(W, 0, linear=True)
    o.reset(x0)
    # brute force: stack every factor as a row block of a weighted least-squares problem
    rows, rhs, wts = [], [], []

    def add(i, j, z, om, nvar_hint):
        rows.append((i, j))
        rhs.append(np.asarray(z, float))
        wts.append(om)

    gt = [x0.copy()]
    for t in range(1, T + 1):
        u = rng.normal(size=3) * 0.3
        gt.append(gt[-1] + u)
        z = u + rng.normal(size=3) * SIG[3:6]
        add(t - 1, t, z, om_odo, t)
        c_old = min(t, W - 1)
        back = int(rng.integers(1, c_old + 1)) if rng.uniform() < 0.6 else 0
        zl = np.zeros(3)
        if back:
            zl = gt[t] - gt[t - back] + rng.normal(size=3) * SIG[6:9] * 3.0
            add(t - back, t, zl, om_lc, t)
        o.push(z, back, zl)
        o.solve(1)                     # linear problem: one GN iteration is the exact optimum
        assert o.solve(1) < 1e-9       # ... so a second one must not move
        S, ld = o.cov()
        n = 3 * (t + 1)
        A = np.zeros((n, n))
        rv = np.zeros(n)
        A[:3, :3] += np.diag(1.0 / P0)
        rv[:3] += x0 / P0
        for (i, j), zz, om in zip(rows, rhs, wts):
            for k in range(3):
                a = np.zeros(n)
                a[3 * j + k], a[3 * i + k] = 1.0, -1.0
                A += om[k] * np.outer(a, a)
                rv += om[k] * a * zz[k]
        P = np.linalg.inv(A)
        xhat = P @ rv
        got = o.poses()[o.count - 1]
        assert np.allclose(got, xhat[-3:], rtol=1e-8, atol=1e-9), (t, got, xhat[-3:])
        assert np.allclose(S, P[-3:, -3:], rtol=1e-7, atol=1e-14)
        # every pose still in the window must match the full-batch smoothed estimate
        c = o.count
        for s in range(c):
            assert np.allclose(o.poses()[s], xhat[3 * (t - c + 1 + s):3 * (t - c + 2 + s)], rtol=1e-8, atol=1e-9)
        if o.count == W:
            # A quadratic problem is marginalized exactly at ANY expansion point: move the state off the
            # optimum first, so that the gradient terms of the Schur complement (g' = g_r - H_rw H_ww^-1 g_w)
            # are non-zero and a wrong sign or index in them shows up at the next step.
            o.set_state(o.state() + rng.normal(size=o.n) * 0.1)
            o.marginalize()


# ----------------------------------------------------------------------------- P7
def test_invariants_noisy_loops_and_landmarks():
    for cfg in (synth.Config("a", N=3, W=8, L=0, iters=3, T=80, p_lc=0.3, seed=2),
                synth.Config("b", N=2, W=6, L=8, iters=2, T=60, p_lc=0.2, seed=3)):
        data = synth.generate(cfg)
        for env in range(cfg.N):
            o = Oracle(cfg.W, cfg.L)

            def check(rec, orc):
                S = rec["cov"]
                assert np.allclose(S, S.T, atol=0)
                assert np.linalg.eigvalsh(S).min() > 0
                Lam, g, vb = orc.prior()
                assert np.allclose(Lam, Lam.T, atol=0)
                assert np.linalg.eigvalsh(Lam).min() > -1e-9 * np.abs(Lam).max()
                assert rec["poses"].shape == (cfg.W, 3)       # bounded memory

            drive(o, data, env, cfg.iters, on_step=check)


def test_gauss_newton_decreases_cost():
    cfg = synth.Config("c", N=1, W=8, L=4, iters=1, T=30, p_lc=0.5, seed=9)
    data = synth.generate(cfg)
    o = Oracle(cfg.W, cfg.L)
    o.reset()
    o.observe_first(*rb_inputs(data, 0, 0))
    for t in range(1, cfg.T + 1):
        o.push(*step_inputs(data, t, 0))
        c0 = o.cost()
        o.solve(1)
        c1 = o.cost()
        o.solve(3)
        c2 = o.cost()
        assert c1 <= c0 * (1 + 1e-9) + 1e-12 and c2 <= c1 * (1 + 1e-9) + 1e-12
        # at the (near-)optimum the gradient vanishes
        _, b = o.assemble()
        H, _ = o.assemble()
        assert np.abs(np.linalg.solve(H, b)).max() < 1e-6
        if o.count == cfg.W:
            o.marginalize()


# ----------------------------------------------------------------------------- P8
def test_noisy_fixed_lag_close_to_full_batch_and_nees():
    cfg = synth.Config("d", N=48, W=10, L=0, iters=3, T=60, p_lc=0.2, seed=4)
    data = synth.generate(cfg)
    res = oracle.run_batch(data, cfg.iters)
    assert res["bad"] == 0
    # loose agreement with a converged global full-batch solve (differs only by linearization points)
    for env in range(2):
        fb = fullbatch.FullBatch(SIG, 0)
        for t in range(1, cfg.T + 1):
            fb.push(*step_inputs(data, t, env)[:3])
        fb.gauss_newton()
        S_fb = fb.last_cov()
        S = res["cov"][-1, env]
        assert np.abs(S - S_fb).max() < 2e-2 * np.abs(S_fb).max()
        x = res["poses"][-1, env, cfg.W - 1]
        assert np.abs(x[:2] - fb.x[-1][:2]).max() < 5e-2
    # NEES of the newest pose ~ chi^2 with 3 dof (mean 3)
    nees = []
    for t in range(10, cfg.T):
        c = min(t + 2, cfg.W)
        err = res["poses"][t, :, c - 1] - data["gt"][t + 1].T
        err[:, 2] = fullbatch.wrap(err[:, 2])
        Sinv = np.linalg.inv(res["cov"][t])
        nees.append(np.einsum("ni,nij,nj->n", err, Sinv, err))
    m = float(np.mean(nees))
    assert 2.0 < m < 4.5, m


def test_run_batch_matches_single_env_driver_and_is_env_independent():
    cfg = synth.Config("e", N=5, W=6, L=4, iters=2, T=25, p_lc=0.3, seed=6)
    data = synth.generate(cfg)
    res = oracle.run_batch(data, cfg.iters, envs=[3, 1])
    recs = drive(Oracle(cfg.W, cfg.L), data, 3, cfg.iters)
    for t, rec in enumerate(recs):
        assert np.allclose(res["cov"][t, 0], rec["cov"], rtol=1e-12, atol=0)
        assert np.allclose(res["poses"][t, 0], rec["poses"], rtol=1e-12, atol=1e-14)
    # environment i's trajectory does not depend on which other environments are generated
    sub = synth.generate(cfg, env_ids=[1])
    res1 = oracle.run_batch(sub, cfg.iters)
    assert np.array_equal(res1["logdet"][:, 0], res["logdet"][:, 1])


# ----------------------------------------------------------------------------- NEXT-1: unary absolute-pose factor
def _random_spd(rng, scale):
    A = rng.normal(size=(3, 3))
    return (A @ A.T + 0.5 * np.eye(3)) * scale


def test_unary_factor_jacobians_fd():
    rng = np.random.default_rng(21)
    for _ in range(10):
        a, ek, z = rng.normal(size=3) * [4, 4, 1], rng.normal(size=3), rng.normal(size=3) * [4, 4, 1]
        r, Ja, Je = oracle.unary_factor(a, ek, z)
        assert np.allclose(Ja, fd_jac(lambda q: oracle.unary_factor(q, ek, z)[0], a), atol=1e-6)
        assert np.allclose(Je, fd_jac(lambda q: oracle.unary_factor(a, q, z)[0], ek), atol=1e-6)
        r0, Ja0, Je0 = oracle.unary_factor(a, ek, z, k_is_frame=True)
        assert np.allclose(Ja0, np.eye(3)) and np.allclose(Je0, 0)
    # definition: measuring the pose itself gives r = 0
    a, e = np.array([1.0, -2.0, 0.4]), np.array([0.3, 0.2, -0.1])
    x = synth.compose(a[:, None], e[:, None])[:, 0]
    assert np.allclose(oracle.unary_factor(a, e, x)[0], 0, atol=1e-15)


def test_unary_factor_is_the_kalman_update():
    """One odometry step then an absolute-pose measurement of the predicted pose (zero residual):
    the posterior covariance is the textbook information-form update (P^-1 + Omega)^-1."""
    rng = np.random.default_rng(22)
    P0, Q = SIG[0:3] ** 2, SIG[3:6] ** 2
    for W in (2, 4):
        o = Oracle(W, 0)
        o.reset()
        Sig = np.diag(P0)
        for k in range(1, 7):
            o.push([0.2, 0.0, 0.0])
            F = np.array([[1, 0, 0], [0, 1, 0.2], [0, 0, 1.0]])
            Sig = F @ Sig @ F.T + np.diag(Q)
            Om = _random_spd(rng, 50.0)
            o.add_unary(o.poses()[o.count - 1], Om)
            assert o.solve(2) < 1e-12
            Sig = np.linalg.inv(np.linalg.inv(Sig) + Om)
            S, ld = o.cov()
            assert np.allclose(S, Sig, rtol=1e-9, atol=1e-15), (W, k)
            assert abs(ld - np.log(np.linalg.det(Sig))) < 1e-9
            if o.count == W:
                o.marginalize()


@pytest.mark.parametrize("W,L,p_lc", [(6, 0, 0.4), (5, 6, 0.3)])
def test_unary_noise_free_recovery_and_full_batch_equality(W, L, p_lc):
    cfg = synth.Config("un", N=2, W=W, L=L, iters=2, T=35, p_lc=p_lc, seed=13, p_unary=0.5)
    data = synth.generate(cfg, noise_scale=0.0, dtype=np.float64)
    assert data["un_valid"].sum() > 10
    from tests.helpers import unary_inputs
    for env in range(cfg.N):
        fb = fullbatch.FullBatch(SIG, L)
        o = Oracle(W, L)
        o.reset()
        if L:
            fb.observe_first(*rb_inputs(data, 0, env))
            o.observe_first(*rb_inputs(data, 0, env))
        for t in range(1, cfg.T + 1):
            odom, back, zlc, valid, zrb = step_inputs(data, t, env)
            fb.push(odom, back, zlc, valid, zrb)
            o.push(odom, back, zlc, valid, zrb)
            un = unary_inputs(data, t, env)
            if un is not None:
                fb.add_unary(*un)
                o.add_unary(*un)
            assert o.solve(2) < 1e-10
            c = o.count
            err = o.poses()[:c] - data["gt"][t - c + 1: t + 1, :, env]
            err[:, 2] = fullbatch.wrap(err[:, 2])
            assert np.abs(err).max() < 1e-9
            S, ld = o.cov()
            ref = fb.last_cov()
            scale = np.sqrt(np.outer(np.diag(ref), np.diag(ref)))
            assert np.all(np.abs(S - ref) <= 1e-7 * scale), (t, S, ref)
            if o.count == W:
                o.marginalize()


def test_unary_linear_gaussian_equals_brute_force():
    rng = np.random.default_rng(23)
    W, T = 4, 20
    P0 = SIG[0:3] ** 2
    om_odo = 1.0 / SIG[3:6] ** 2
    x0 = np.array([0.1, 0.2, -0.1])
    o = Oracle(W, 0, linear=True)
    o.reset(x0)
    facs = []       # (A_rows [m x n later], rhs, weight matrix)
    gt = [x0.copy()]
    for t in range(1, T + 1):
        u = rng.normal(size=3) * 0.3
        gt.append(gt[-1] + u)
        z = u + rng.normal(size=3) * SIG[3:6]
        facs.append(("b", t - 1, t, z, np.diag(om_odo)))
        o.push(z)
        if rng.uniform() < 0.6:
            Om = _random_spd(rng, 30.0)
            zu = gt[t] + rng.normal(size=3) * 0.2
            facs.append(("u", t, t, zu, Om))
            o.add_unary(zu, Om)
        o.solve(1)
        assert o.solve(1) < 1e-9
        n = 3 * (t + 1)
        A = np.zeros((n, n))
        rv = np.zeros(n)
        A[:3, :3] += np.diag(1.0 / P0)
        rv[:3] += x0 / P0
        for kind, i, j, zz, Om in facs:
            Jm = np.zeros((3, n))
            Jm[:, 3 * j:3 * j + 3] = np.eye(3)
            if kind == "b":
                Jm[:, 3 * i:3 * i + 3] = -np.eye(3)
            A += Jm.T @ Om @ Jm
            rv += Jm.T @ Om @ zz
        P = np.linalg.inv(A)
        xhat = P @ rv
        assert np.allclose(o.poses()[o.count - 1], xhat[-3:], rtol=1e-8, atol=1e-9)
        assert np.allclose(o.cov()[0], P[-3:, -3:], rtol=1e-7, atol=1e-14)
        if o.count == W:
            o.set_state(o.state() + rng.normal(size=o.n) * 0.1)
            o.marginalize()


# ----------------------------------------------------------------------------- NEXT-2: per-environment episode reset
def test_reset_restarts_the_estimator_like_a_fresh_run():
    """A reset at step t0 at the true pose must give exactly what a fresh estimator started there gives
    (the batch driver's reset path against single-environment runs), and noise-free recovery must
    survive resets."""
    cfg = synth.Config("rs", N=3, W=6, L=4, iters=2, T=40, p_lc=0.3, seed=19, p_reset=0.08)
    data = synth.generate(cfg)
    assert data["reset"].sum() >= 3
    res = oracle.run_batch(data, cfg.iters)
    for env in range(cfg.N):
        recs = drive(Oracle(cfg.W, cfg.L), data, env, cfg.iters)
        for t, rec in enumerate(recs):
            assert np.allclose(res["cov"][t, env], rec["cov"], rtol=1e-12, atol=0)
        # after the LAST reset the run equals a fresh estimator initialised at that pose
        ts = np.where(data["reset"][:, env])[0]
        if len(ts) == 0:
            continue
        t0 = ts[-1]                                   # reset before the push of step t0+1
        o = Oracle(cfg.W, cfg.L)
        o.reset(data["reset_pose"][t0, :, env].astype(np.float64))
        for t in range(t0 + 1, cfg.T + 1):
            o.push(*step_inputs(data, t, env))
            o.solve(cfg.iters)
            S, ld = o.cov()
            assert np.allclose(S, res["cov"][t - 1, env], rtol=1e-12, atol=0)
            if o.count == cfg.W:
                o.marginalize()
    nf = synth.generate(cfg, noise_scale=0.0, dtype=np.float64)
    for env in range(cfg.N):
        for rec in drive(Oracle(cfg.W, cfg.L), nf, env, 2):
            c = rec["count"]
            gt = nf["gt"][rec["t"] - c + 1: rec["t"] + 1, :, env]
            err = rec["poses"][:c] - gt
            err[:, 2] = fullbatch.wrap(err[:, 2])
            assert rec["step"] < 1e-10 and np.abs(err).max() < 1e-9
