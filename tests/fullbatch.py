"""Independent global-coordinate, full-trajectory (no marginalization) pose-graph routines in numpy.

Used ONLY to pin the oracle (tests/test_oracle_pins.py): every pose x_0..x_t and every observed
landmark is a variable in GLOBAL coordinates, nothing is marginalized, the Hessian is dense.  This
is the textbook problem statement (eq. (5)); the fixed-lag oracle must agree with it where
mathematics says it must (noise-free inputs; linear-Gaussian inputs).  Shares no code with oracle/
or with the CUDA path.
"""
import numpy as np


def wrap(x):
    return np.arctan2(np.sin(x), np.cos(x))


def between_res_jac(xi, xj, z):
    c, s = np.cos(xi[2]), np.sin(xi[2])
    dx, dy = xj[0] - xi[0], xj[1] - xi[1]
    hx, hy = c * dx + s * dy, -s * dx + c * dy
    r = np.array([hx - z[0], hy - z[1], wrap(xj[2] - xi[2] - z[2])])
    Ji = np.array([[-c, -s, hy], [s, -c, -hx], [0, 0, -1.0]])
    Jj = np.array([[c, s, 0], [-s, c, 0], [0, 0, 1.0]])
    return r, Ji, Jj


def rb_res_jac(x, l, z):
    dx, dy = l[0] - x[0], l[1] - x[1]
    q = dx * dx + dy * dy
    rho = np.sqrt(q)
    r = np.array([rho - z[0], wrap(np.arctan2(dy, dx) - x[2] - z[1])])
    Jp = np.array([[-dx / rho, -dy / rho, 0], [dy / q, -dx / q, -1.0]])
    Jl = np.array([[dx / rho, dy / rho], [-dy / q, dx / q]])
    return r, Jp, Jl


class FullBatch:
    """Global full-batch Gauss-Newton problem built incrementally from the same step inputs."""

    def __init__(self, sig, L=0):
        self.sig = np.asarray(sig, float)
        self.x = [np.zeros(3)]          # poses, global
        self.lm = {}                    # landmark id -> position (global)
        self.fac = []                   # ('b', i, j, z, omega) / ('rb', k, l, z)
        self.L = L

    def _observe(self, k, valid, zrb):
        for l in range(self.L):
            if not valid[l]:
                continue
            if l not in self.lm:
                x = self.x[k]
                self.lm[l] = np.array([x[0] + zrb[l, 0] * np.cos(x[2] + zrb[l, 1]),
                                       x[1] + zrb[l, 0] * np.sin(x[2] + zrb[l, 1])])
            self.fac.append(("rb", k, l, np.array(zrb[l], float)))

    def observe_first(self, valid, zrb):
        self._observe(0, valid, zrb)

    def push(self, odom, lc_back=0, lc_meas=None, valid=None, zrb=None):
        p = self.x[-1]
        c, s = np.cos(p[2]), np.sin(p[2])
        self.x.append(np.array([p[0] + c * odom[0] - s * odom[1], p[1] + s * odom[0] + c * odom[1],
                                wrap(p[2] + odom[2])]))
        t = len(self.x) - 1
        self.fac.append(("b", t - 1, t, np.array(odom, float), 1.0 / self.sig[3:6] ** 2))
        if lc_back > 0:
            self.fac.append(("b", t - lc_back, t, np.array(lc_meas, float), 1.0 / self.sig[6:9] ** 2))
        if self.L:
            self._observe(t, valid, zrb)

    def add_unary(self, z, Om):
        """absolute-pose factor on the newest pose, full 3x3 information"""
        self.fac.append(("un", len(self.x) - 1, np.array(z, float), np.array(Om, float).reshape(3, 3)))

    def system(self):
        T = len(self.x)
        lids = sorted(self.lm)
        lpos = {l: 3 * T + 2 * i for i, l in enumerate(lids)}
        n = 3 * T + 2 * len(lids)
        H, g = np.zeros((n, n)), np.zeros(n)
        om0 = 1.0 / self.sig[0:3] ** 2
        r0 = self.x[0].copy()
        r0[2] = wrap(r0[2])
        H[:3, :3] += np.diag(om0)
        g[:3] += om0 * r0
        om_rb = 1.0 / self.sig[9:11] ** 2
        for f in self.fac:
            if f[0] == "un":
                _, k, z, Om = f
                r = self.x[k] - z
                r[2] = wrap(r[2])
                H[3 * k:3 * k + 3, 3 * k:3 * k + 3] += Om
                g[3 * k:3 * k + 3] += Om @ r
                continue
            if f[0] == "b":
                _, i, j, z, om = f
                r, Ji, Jj = between_res_jac(self.x[i], self.x[j], z)
                blocks = [(3 * i, Ji), (3 * j, Jj)]
            else:
                _, k, l, z = f
                r, Jp, Jl = rb_res_jac(self.x[k], self.lm[l], z)
                om = om_rb
                blocks = [(3 * k, Jp), (lpos[l], Jl)]
            for ia, Ja in blocks:
                g[ia:ia + Ja.shape[1]] += Ja.T @ (om * r)
                for ib, Jb in blocks:
                    H[ia:ia + Ja.shape[1], ib:ib + Jb.shape[1]] += Ja.T @ (om[:, None] * Jb)
        return H, g, lpos

    def gauss_newton(self, iters=20):
        for _ in range(iters):
            H, g, lpos = self.system()
            d = np.linalg.solve(H, -g)
            T = len(self.x)
            for k in range(T):
                self.x[k] = self.x[k] + d[3 * k:3 * k + 3]
                self.x[k][2] = wrap(self.x[k][2])
            for l, p in lpos.items():
                self.lm[l] = self.lm[l] + d[p:p + 2]
            if np.abs(d).max() < 1e-13:
                break

    def last_cov(self):
        H, _, _ = self.system()
        T = len(self.x)
        P = np.linalg.inv(H)
        return P[3 * (T - 1):3 * T, 3 * (T - 1):3 * T]
