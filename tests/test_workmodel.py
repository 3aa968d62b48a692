"""The roofline work model replays the kernels' window bookkeeping on the event arrays; here its
envelope (`first`) is checked against the sparsity pattern of the ORACLE's dense H (independent code),
permuted into the kernels' elimination order, and its flop formula against brute force."""
import numpy as np

from oracle import Oracle
from harness import synth, workmodel
from tests.helpers import rb_inputs, step_inputs


def _mask(data, t, env):
    m = 0
    for q in range(data["rb_mask"].shape[1]):
        m |= int(data["rb_mask"][t, q, env]) << (32 * q)
    return m


def test_envelope_matches_oracle_sparsity_pattern():
    for cfg in (synth.Config("a", N=2, W=8, L=0, iters=2, T=60, p_lc=0.4, seed=1),
                synth.Config("b", N=2, W=6, L=7, iters=2, T=40, p_lc=0.3, seed=2)):
        W, L, n = cfg.W, cfg.L, 3 * cfg.W + 2 * cfg.L
        data = synth.generate(cfg)
        for env in range(cfg.N):
            o = Oracle(W, L)
            o.reset()
            ws = workmodel.WindowStructure(W, L)
            if L:
                o.observe_first(*rb_inputs(data, 0, env))
                ws.observe_first(_mask(data, 0, env))
            for t in range(1, cfg.T + 1):
                o.push(*step_inputs(data, t, env))
                ws.push(int(data["lc_back"][t - 1, env]), _mask(data, t, env) if L else 0)
                c = o.count
                assert c == ws.c
                H, _ = o.assemble()
                # natural index -> elimination offset
                perm = np.full(n, -1)
                perm[0:3] = 3 * (W - 2) + 2 * L + 3 + np.arange(3)
                for k in range(1, c):
                    perm[3 * k:3 * k + 3] = ws.off_slot(k) + np.arange(3)
                _, act = o.landmarks()
                for l in range(L):
                    if act[l]:
                        perm[3 * W + 2 * l:3 * W + 2 * l + 2] = ws.off_lm(l) + np.arange(2)
                live = np.where(perm >= 0)[0]
                first_true = {}
                for i in live:
                    cols = [perm[j] for j in live if abs(H[i, j]) > 1e-9 * np.sqrt(H[i, i] * H[j, j]) and perm[j] <= perm[i]]
                    first_true[perm[i]] = min(cols)
                first = ws.first()
                # block granularity: every structural non-zero lies inside the model's envelope, and the
                # envelope of each block starts exactly at the first coupled block
                blocks = {}
                for pi, f in first_true.items():
                    assert first[pi] <= f
                    blocks.setdefault(first[pi], []).append(f)
                for i in live:
                    pi = perm[i]
                    blk = [first_true[perm[j]] for j in live if first[perm[j]] == first[pi] and abs(perm[j] - pi) <= 2]
                    assert min(blk) - first[pi] <= 2, (t, pi, first[pi], min(blk))
                o.solve(cfg.iters)
                if c == W:
                    o.marginalize()
                    ws.marginalize()
                    Lam, _, _ = o.prior()
                    # the model's support == the non-zero pattern of the oracle's new prior
                    # (dense congruence leaves round-off dust, ~1e-16 relative, outside the true support)
                    sup_true = {i for i in range(n) if np.abs(Lam[i]).max() > 1e-9 * np.abs(Lam).max()}
                    sup_model = {0, 1, 2}
                    for k in range(1, W):
                        if (ws.ps >> k) & 1:
                            sup_model |= {3 * k, 3 * k + 1, 3 * k + 2}
                    for l in range(L):
                        if (ws.ls >> l) & 1:
                            sup_model |= {3 * W + 2 * l, 3 * W + 2 * l + 1}
                    assert sup_true == sup_model


def test_envelope_flops_brute_force():
    rng = np.random.default_rng(0)
    n = 17
    first = np.minimum(np.arange(n), rng.integers(0, n, n))
    f_chol, f_fwd, f_back, words = workmodel.envelope_flops(first)
    brute = 0
    for i in range(n):
        for j in range(first[i], i + 1):
            brute += 1
            for k in range(max(first[i], first[j]), j):
                brute += 2
    assert f_chol == brute
    assert f_fwd == sum(2 * (j - first[j]) + 1 for j in range(n)) == f_back
    assert words == sum(i - first[i] + 1 for i in range(n)) + n + 1
    # dense case: n^3/3 leading term
    d = workmodel.envelope_flops(np.zeros(60, np.int64))[0]
    assert abs(d - 60 ** 3 / 3) / (60 ** 3 / 3) < 0.05


def test_step_work_orders_of_magnitude():
    cfg = synth.Config("w", N=4, W=20, L=0, iters=3, T=60, p_lc=0.1, seed=0)
    data = synth.generate(cfg)
    w = workmodel.step_work(data, cfg.iters, envs=[0, 1, 2, 3])
    steady = w["flops"][30:].mean()
    assert 1.5e4 < steady < 1.5e5          # ~3.3e4 flop per env-step for config 1
    assert 5e2 < w["bytes"][30:].mean() < 5e3
    assert (np.diff(w["flops"][:15]) > 0).all()   # window-fill phase grows
