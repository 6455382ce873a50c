"""Adaptive dynamic relaxation (ADR) on top of the CPU oracle's force -- quasi-static driver of the paper's Ex. 4
("solved by using an adaptive dynamic relaxation algorithm presented in [Underwood 1983; Kilic & Madenci
2010; Ni 2019]"; the paper does not restate the algorithm, SPEC.md:460 records the canonical formulation used here).

TEST INFRASTRUCTURE (same rule as pd_oracle.c).  Step by step, in the cited notation, pseudo time step Dt = 1:

    Lambda Udd + c Lambda Ud = F(U)           F = internal force density of Eq. 2.1 + external body force density
    n = 0:  Ud^{1/2} = Dt Lambda^{-1} F^0 / 2
    n > 0:  1K_ii^n = -(F_i^n - F_i^{n-1}) / (lambda_ii Dt Ud_i^{n-1/2})      (0 where Ud_i^{n-1/2} = 0)
            c^n     = 2 sqrt( (U^n . 1K^n U^n) / (U^n . U^n) )                (0 if the quotient is not positive)
            Ud^{n+1/2} = ((2 - c^n Dt) Ud^{n-1/2} + 2 Dt Lambda^{-1} F^n) / (2 + c^n Dt)
    U^{n+1} = U^n + Dt Ud^{n+1/2}
    clamped dofs keep U; dofs flagged "prescribed" advance by the fixed increment value[i,k] per iteration
    ("a gradually increasing ... displacement ... with a fix increment"), their Ud is that increment;
    after the update the failure check of the explicit scheme runs on U^{n+1} (every iteration, SPEC.md open question).
Lambda = lam * I (uniform fictitious density; stability needs lam >= Dt^2/4 * lambda_max(K), Underwood's bound; the
harness takes it from the explicit scheme's own stability literal: lambda_max(K) = rho (2 / dt_crit)^2).
Pins (tests/test_oracle_pins.py): 1-dof spring -> F/k; zero load -> 0; a small bar under end load and a prescribed end
displacement -> the direct dense solve of K U = F assembled from the (linear) oracle force, to 1e-6.
"""
from __future__ import annotations

import numpy as np


class ADROracle:
    def __init__(self, oracle, lam: float):
        self.o = oracle            # a PDOracle; its u is U^n, its flags / value give the boundary dofs
        self.lam = float(lam)
        n, d = oracle.n, oracle.dim
        self.ud = np.zeros((n, d))
        self.f_prev = np.zeros((n, d))
        self.it = 0
        self.c_hist = []
        self.near_total = 0        # bonds within 1e-9 relative of s_c at a failure check (reported, like PDOracle.near_total)
        fl = oracle.flags
        self.clamped = np.stack([(fl & (1 << k)) != 0 for k in range(d)], axis=1)
        self.presc = np.stack([(fl & (8 << k)) != 0 for k in range(d)], axis=1) & ~self.clamped
        self.body = ((fl & 64) != 0)[:, None] & ~self.clamped & ~self.presc

    def total_force(self):
        f = self.o.force_density().copy()
        return f + np.where(self.body, self.o.value, 0.0)

    def iterate(self, niter: int):
        o = self.o
        for _ in range(niter):
            F = self.total_force()
            free = ~self.clamped & ~self.presc
            if self.it == 0:
                c = 0.0
                ud = 0.5 * F / self.lam
            else:
                with np.errstate(divide="ignore", invalid="ignore"):
                    k1 = np.where(self.ud != 0.0, -(F - self.f_prev) / (self.lam * self.ud), 0.0)
                k1 = np.where(free, k1, 0.0)
                uu = np.where(free, o.u, 0.0)
                num, den = float(np.sum(uu * k1 * uu)), float(np.sum(uu * uu))
                c = 2.0 * np.sqrt(num / den) if (den > 0.0 and num / den > 0.0) else 0.0
                ud = ((2.0 - c) * self.ud + 2.0 * F / self.lam) / (2.0 + c)
            ud = np.where(self.clamped, 0.0, np.where(self.presc, o.value, ud))
            o.u += ud
            self.ud, self.f_prev = ud, F
            self.c_hist.append(c)
            self.it += 1
            if o.s_c > 0.0 and np.isfinite(o.s_c):
                self.near_total += o.break_bonds()[1]
        o.damage()
        return o.u


def dense_stiffness(oracle):
    """K with f(u) = -K u, column by column from the linear oracle force (small models only)"""
    n, d = oracle.n, oracle.dim
    K = np.zeros((n * d, n * d))
    for q in range(n * d):
        e = np.zeros(n * d)
        e[q] = 1.0
        K[:, q] = -oracle.force_density(e.reshape(n, d)).reshape(-1)
    return K
