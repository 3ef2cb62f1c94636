"""A second, vectorised numpy statement of the C.1 model, used only by
the pins that need an ODE right-hand side independent of oracle/ (brute-force implicit Euler,
scipy cross-check).  libm exp/pow, no ordering contract -- agreement is to rounding only."""
import numpy as np

NA_MEV = 9.648533212331e17
RGAS = 8.31446261815324e7
ARAD = 7.565733250e-15


class RefModel:
    def __init__(self, net):
        self.net = net
        self.N = net.nspec
        self.K = net.nreac
        self.fac = NA_MEV / net.cv
        self.reac = [[int(r) for r in row if r >= 0] for row in net.reactant]
        self.sto = [[(int(i), float(d)) for i, d in zip(net.stoich_id[k], net.stoich_dy[k]) if i >= 0]
                    for k in range(self.K)]
        self.sym = []
        for r in self.reac:
            s = 1.0
            for sp in set(r):
                s *= float(np.prod(np.arange(1, r.count(sp) + 1)))
            self.sym.append(1.0 / s)

    def lam(self, T):
        T9 = T * 1e-9
        n = self.net
        return n.rate_A * T9 ** n.rate_n * np.exp(-n.rate_B / np.cbrt(T9))

    def rho_factor(self, rho):
        e = getattr(self.net, "rate_rho_exp", None)
        return 1.0 if e is None else rho ** np.asarray(e)

    def rate(self, k, rho, Y, lam):
        r = self.reac[k]
        mag = lam[k] * rho ** (len(r) - 1) * self.sym[k] * np.prod([abs(Y[a]) for a in r])
        return -mag if any(Y[a] < 0 for a in r) else mag      # reading s19 (odd extension)

    def f(self, rho, y):
        lam = self.lam(y[self.N]) * self.rho_factor(rho)
        out = np.zeros(self.N + 1)
        for k in range(self.K):
            R = self.rate(k, rho, y, lam)
            for i, d in self.sto[k]:
                out[i] += d * R
            out[self.N] += self.net.q_mev[k] * R
        out[self.N] *= NA_MEV / self.cv(rho, y)
        return out

    def cv(self, rho, y):
        """Constant c_v, or the analytic EOS when the network carries charges."""
        z = getattr(self.net, "zion", None)
        if z is None:
            return self.net.cv
        ysum = getattr(self.net, "eos_extra", 0.0) + np.dot(1.0 + np.asarray(z), y[: self.N])
        return 1.5 * RGAS * ysum + 4.0 * ARAD * y[self.N] ** 3 / rho

    def jac_fd(self, rho, y, rel=1e-6):
        n = self.N + 1
        J = np.zeros((n, n))
        for j in range(n):
            h = rel * max(abs(y[j]), 1e-12 if j < self.N else 1.0)
            yp, ym = y.copy(), y.copy()
            yp[j] += h
            ym[j] -= h
            J[:, j] = (self.f(rho, yp) - self.f(rho, ym)) / (2 * h)
        return J
