"""Closed-form two-species Krook-Wu (BKW) solution, section 3.2, Eq. 19-23.
ORACLE -- test infrastructure.  Pins the whole operator against an exact right-hand side.

Constant collision kernel B_pq = lambda_pq / (4 pi n^(q)) (reading K-2): gamma = eta = 0
and beta_pq = lambda_pq / (4 pi n^(q)).
"""
from math import exp, pi

import numpy as np


class KrookWu:
    def __init__(self, m1, m2, n1=1.0, n2=1.0, lam11=1.0, lam22=1.0, lam12=0.5, lam21=0.5):
        self.m = (m1, m2)
        self.n = (n1, n2)
        self.lam = ((lam11, lam12), (lam21, lam22))
        mu = 4.0 * m1 * m2 / (m1 + m2) ** 2                               # Eq. 20
        self.mu = mu
        tau1 = lam22 - lam21 * mu * (3.0 - 2.0 * mu)
        tau2 = lam11 - lam12 * mu * (3.0 - 2.0 * mu)
        self.tau = (tau1, tau2)
        self.A = (lam11 + lam21 * mu * (3.0 - 2.0 * mu * tau2 / tau1)) / 6.0
        self.B = (lam11 * tau1 + lam21 * mu * (3.0 - 2.0 * mu) * tau2) / 3.0

    def condition(self):
        """Left-hand side of Eq. 21; must vanish."""
        t1, t2 = self.tau
        return (t1 - t2) * (2.0 * self.mu ** 2 * (self.lam[1][0] / t1 - self.lam[0][1] / t2) - 1.0)

    def Q(self, t):
        return self.A / (self.A * exp(self.A * t) - self.B)

    def dQ(self, t):                                                      # Eq. 23
        return -self.A ** 3 * exp(self.A * t) / (self.A * exp(self.A * t) - self.B) ** 2

    def K(self, t):
        n1, n2 = self.n
        s = n1 * self.tau[0] + n2 * self.tau[1]
        return (n1 + n2) / ((n1 + n2) + 2.0 * s * self.Q(t))

    def dK(self, t):                                                      # Eq. 23
        n1, n2 = self.n
        s = n1 * self.tau[0] + n2 * self.tau[1]
        return -2.0 * (n1 + n2) * s / ((n1 + n2) + 2.0 * s * self.Q(t)) ** 2 * self.dQ(t)

    def f(self, p, t, v2):
        """Eq. 19: f^(p)(t, v) as a function of v2 = |v|^2."""
        m, n = self.m[p], self.n[p]
        K, Qp = self.K(t), self.tau[p] * self.Q(t)
        return n * (m / (2.0 * pi * K)) ** 1.5 * np.exp(-m * v2 / (2.0 * K)) * ((1.0 - 3.0 * Qp) + m / K * Qp * v2)

    def dfdt(self, p, t, v2):
        """Eq. 22: d/dt f^(p) = sum_q Q^(pq)(f^p, f^q)."""
        m, n = self.m[p], self.n[p]
        K, dK = self.K(t), self.dK(t)
        Qp, dQp = self.tau[p] * self.Q(t), self.tau[p] * self.dQ(t)
        Mx = n * (m / (2.0 * pi * K)) ** 1.5 * np.exp(-m * v2 / (2.0 * K))
        return self.f(p, t, v2) * (-1.5 / K * dK + m * v2 / (2.0 * K * K) * dK) \
            + Mx * (-3.0 * dQp + m / K * dQp * v2 - m / (K * K) * dK * Qp * v2)

    def beta(self):
        """beta_pq = lambda_pq / (4 pi n^(q))."""
        return [[self.lam[p][q] / (4.0 * pi * self.n[q]) for q in range(2)] for p in range(2)]
