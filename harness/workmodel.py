"""Algorithmic work model of one environment step (host logic, numpy only, no method arithmetic).

``bench.py`` needs the ALGORITHMIC flops and bytes of the hot path to report a roofline fraction
(DESIGN.md "Roofline accounting").  They depend on the per-environment structure
(live loop closures, landmark visibility, prior support), so this module replays the window
bookkeeping of the kernels on the generator's event arrays -- no floating-point state -- and counts

  F_alg = (iters+1) (F_lin + F_chol) + iters (F_fwd + F_back) + F_cov + F_marg
  B_alg = step inputs + outputs + state r/w + live factor data + prior on its support r/w

with the envelope (skyline) of H in the kernel's elimination order
[passive landmarks | e_1..e_{W-2} | observed landmarks | newest pose | anchor]
(passive = no live range-bearing factor in the window):

  F_chol = sum_{i<n} sum_{j=first_i..i} (2 (j - max(first_i, first_j)) + 1)
  F_fwd  = sum_{j<n} (2 (j - first_j) + 1)         (the rhs row that rides along the factorisation)
  F_back = sum_{i<n} (2 (i - first_i) + 1)
  F_lin  = 230 #between + 140 #range-bearing + 3 s^2   (s = prior support dimension)
  F_cov  = 500,  F_marg = 12 s'^2                      (s' = support of the marginalised sub-problem)

Structural zeros are never counted: a kernel that multiplies them gets no credit.
"""
from __future__ import annotations

import numpy as np

F_BETWEEN, F_RB, F_COV = 230.0, 140.0, 500.0


def _popcount(x: int) -> int:
    return bin(int(x)).count("1")


class WindowStructure:
    """Structure-only replay of one environment's window (mirrors the kernels' bookkeeping)."""

    def __init__(self, W: int, L: int):
        self.W, self.L, self.n = W, L, 3 * W + 2 * L
        self.c = 1
        self.lct = [-1] * W            # loop-closure target slot per slot
        self.rbm = [0] * W             # visibility bit mask per slot
        self.ps = 0                    # prior support: pose slots (bit k)
        self.ls = 0                    # prior support: landmarks
        self.act = 0                   # active landmarks

    def observe_first(self, mask: int):
        self.rbm[0] = mask
        self.act |= mask

    def push(self, lc_back: int, mask: int):
        c = self.c
        self.lct[c] = c - lc_back if 1 <= lc_back <= c else -1
        self.rbm[c] = mask
        self.act |= mask
        self.c = c + 1

    # elimination offsets: [passive landmarks | chain poses | observed landmarks | newest | anchor]
    def obs(self):
        key = (self.c, tuple(self.rbm))          # (cached: first() asks for it hundreds of times per step)
        if getattr(self, "_obs_key", None) != key:
            m = 0
            for k in range(self.c):
                m |= self.rbm[k]
            self._obs_key, self._obs, self._npas = key, m, self.L - _popcount(m)
        return self._obs

    def npas(self):
        self.obs()
        return self._npas

    def off_slot(self, k):
        return 3 * (self.W - 2) + 2 * self.L if k == self.c - 1 else 2 * self.npas() + 3 * (k - 1)

    def off_lm(self, l):
        obs = self.obs()
        below = (1 << l) - 1
        if (obs >> l) & 1:
            return 2 * self.npas() + 3 * (self.W - 2) + 2 * _popcount(obs & below)
        return 2 * _popcount(~obs & below)

    def support_dim(self):
        return 3 + 3 * _popcount(self.ps) + 2 * _popcount(self.ls)

    def first(self) -> np.ndarray:
        """first[i] for the n rows of H (block granularity), as the symbolic phase computes it."""
        W, L, n, c = self.W, self.L, self.n, self.c
        oC = 2 * self.npas()
        oL, oN, oA = oC + 3 * (W - 2), 3 * (W - 2) + 2 * L, 3 * (W - 2) + 2 * L + 3
        first = np.empty(n, np.int64)
        idx = np.arange(n)
        first[:oC] = (idx[:oC] // 2) * 2
        first[oC:oL] = oC + ((idx[oC:oL] - oC) // 3) * 3
        first[oL:oN] = oL + ((idx[oL:oN] - oL) // 2) * 2
        first[oN:oA] = oN
        first[oA:] = oA
        for k in range(1, c):
            o = self.off_slot(k)
            f = o
            if k >= 2:
                f = min(f, self.off_slot(k - 1))
            if self.lct[k] >= 1:
                f = min(f, self.off_slot(self.lct[k]))
            if k == c - 1 and self.rbm[k]:
                low = (self.rbm[k] & -self.rbm[k]).bit_length() - 1
                f = min(f, self.off_lm(low))
            first[o:o + 3] = f
        for l in range(L):
            o = self.off_lm(l)
            for k in range(1, c - 1):
                if (self.rbm[k] >> l) & 1:
                    first[o:o + 2] = oC + 3 * (k - 1)
                    break
        sup = [self.off_slot(k) for k in range(1, c) if (self.ps >> k) & 1] + \
              [self.off_lm(l) for l in range(L) if (self.ls >> l) & 1]
        if sup:
            fs = min(sup)
            for o in sup:
                d = 3 if (oC <= o < oL or o >= oN) else 2
                first[o:o + d] = np.minimum(first[o:o + d], fs)
            first[oA:] = np.minimum(first[oA:], fs)
        # landmarks are global (R17b): every range-bearing factor also touches the anchor a, so a's rows
        # reach back to the first observing pose and the first observed landmark
        fa = oA
        for k in range(c):
            if self.rbm[k]:
                if k >= 1:
                    fa = min(fa, self.off_slot(k))
                low = (self.rbm[k] & -self.rbm[k]).bit_length() - 1
                fa = min(fa, self.off_lm(low))
        first[oA:] = np.minimum(first[oA:], fa)
        return first

    def counts(self):
        c = self.c
        n_between = (c - 1) + sum(1 for k in range(1, c) if self.lct[k] >= 0)
        n_rb = sum(_popcount(self.rbm[k]) for k in range(c))
        return n_between, n_rb

    def marginalize(self):
        """Returns the support dimension s' of the marginalised sub-problem, then shifts the window."""
        c = self.c
        lc0 = sum(1 << k for k in range(1, c) if self.lct[k] == 0)
        nps = self.ps | 2 | lc0
        nls = self.ls | self.rbm[0]
        s_sub = 3 + 3 * _popcount(nps) + 2 * _popcount(nls)
        self.ps = (nps & ~2) >> 1
        self.ls = nls
        for k in range(1, c):
            t = self.lct[k]
            self.lct[k - 1] = t - 1 if t >= 1 else -1
            self.rbm[k - 1] = self.rbm[k]
        self.lct[c - 1] = -1
        self.rbm[c - 1] = 0
        self.lct[0] = -1
        self.c = c - 1
        return s_sub


def envelope_flops(first: np.ndarray):
    """(F_chol, F_fwd, F_back, envelope words incl. the rhs row) for a given `first` array."""
    n = first.shape[0]
    idx = np.arange(n)
    live = (idx[None, :] >= first[:, None]) & (idx[None, :] <= idx[:, None])          # j in [first_i, i]
    f_chol = int(((2 * (idx[None, :] - np.maximum(first[:, None], first[None, :])) + 1) * live).sum())
    lens = np.arange(n) - first
    f_fwd = int((2 * lens + 1).sum())
    f_back = f_fwd
    words = int((lens + 1).sum()) + n + 1
    return f_chol, f_fwd, f_back, words


def step_work_parallel(data: dict, iters: int, envs, steps: int | None = None, procs: int = 8) -> dict:
    """step_work over `envs` split across `procs` forked processes (pure host logic; the structure replay is
    Python and takes ~1 ms per env-step)."""
    import multiprocessing as mp
    envs = np.asarray(envs)
    procs = max(1, min(procs, len(envs)))
    if procs == 1:
        return step_work(data, iters, envs, steps)
    chunks = [c for c in np.array_split(envs, procs) if len(c)]
    keys = ("cfg", "T", "lc_back", "rb_mask")
    slim = {k: data[k] for k in keys}
    with mp.get_context("fork").Pool(len(chunks)) as pool:
        parts = pool.starmap(step_work, [(slim, iters, c, steps) for c in chunks])
    return {k: sum(p[k] * len(c) for p, c in zip(parts, chunks)) / len(envs) for k in parts[0]}


def step_work(data: dict, iters: int, envs, steps: int | None = None) -> dict:
    """Per-step algorithmic flops/bytes, averaged over the sampled environments `envs`.

    Returns arrays of length T: ``flops``, ``bytes``, ``env_words`` (envelope words incl. rhs row),
    ``support`` (prior support dimension at solve time), ``n_between``, ``n_rb``."""
    cfg = data["cfg"]
    W, L = cfg.W, cfg.L
    T = data["T"] if steps is None else steps
    nw = (L + 31) // 32
    envs = np.asarray(envs)
    out = {k: np.zeros(T) for k in ("flops", "bytes", "env_words", "support", "n_between", "n_rb")}

    def mask_of(t, e):
        m = 0
        for q in range(nw):
            m |= int(data["rb_mask"][t, q, e]) << (32 * q)
        return m

    for e in envs:
        ws = WindowStructure(W, L)
        if L:
            ws.observe_first(mask_of(0, e))
        for t in range(1, T + 1):
            ws.push(int(data["lc_back"][t - 1, e]), mask_of(t, e) if L else 0)
            c = ws.c
            s = ws.support_dim()
            first = ws.first()
            f_chol, f_fwd, f_back, words = envelope_flops(first)
            nb, nrb = ws.counts()
            f_lin = F_BETWEEN * nb + F_RB * nrb + 3.0 * s * s
            s_sub = 0
            f_marg = 0.0
            prior_rw = 4.0 * (s * (s + 1) / 2 + 2 * s)          # read
            if c == W:
                s_sub = ws.marginalize()
                f_marg = 12.0 * s_sub * s_sub
                s_new = s_sub - 3
                prior_rw += 4.0 * (s_new * (s_new + 1) / 2 + 2 * s_new)   # write
            flops = (iters + 1) * (f_lin + f_chol) + iters * (f_fwd + f_back) + F_COV + f_marg
            io = 4.0 * (3 + 1 + 3 + nw + 2 * L) + 4.0 * 10
            state_rw = 2 * 4.0 * (3 + 3 * c + 2 * L)
            factors = 4.0 * (7 * c + nw * c) + 8.0 * nrb
            i = t - 1
            out["flops"][i] += flops
            out["bytes"][i] += io + state_rw + factors + prior_rw
            out["env_words"][i] += words
            out["support"][i] += s
            out["n_between"][i] += nb
            out["n_rb"][i] += nrb
    for k in out:
        out[k] /= len(envs)
    return out
