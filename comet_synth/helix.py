"""Closed-form helix of a charged particle in a uniform B_z (truth generator only).

dT/ds = c (T x z_hat),  c = KAPPA q B_z / |p|   (Eq. (2)'s "0.3 B",
in cm: radius R = p_T / (KAPPA |q B_z|)).  This is the analytic solution the
input generator uses to make truth hits; the method under test integrates the
same equation numerically (RKN4) and never sees this file's formulas.
"""
import numpy as np

KAPPA = 2.99792458  # (MeV/c) / (T cm)


class Helix:
    def __init__(self, x0, p, charge: int, bz: float):
        self.x0 = np.asarray(x0, dtype=np.float64)
        p = np.asarray(p, dtype=np.float64)
        self.pmag = float(np.linalg.norm(p))
        self.T0 = p / self.pmag
        self.c = KAPPA * charge * bz / self.pmag
        self.charge = charge
        self.bz = bz

    @property
    def radius(self) -> float:
        return float(np.hypot(self.T0[0], self.T0[1]) / abs(self.c))

    @property
    def centre_xy(self):
        # x(s) = x0 + (Tx0 sin cs + Ty0 (1 - cos cs)) / c  => centre = x0 + (Ty0, -Tx0)/c
        return self.x0[0] + self.T0[1] / self.c, self.x0[1] - self.T0[0] / self.c

    def tangent(self, s):
        s = np.asarray(s, dtype=np.float64)
        cs, sn = np.cos(self.c * s), np.sin(self.c * s)
        tx = self.T0[0] * cs + self.T0[1] * sn
        ty = -self.T0[0] * sn + self.T0[1] * cs
        tz = np.broadcast_to(self.T0[2], s.shape)
        return np.stack([tx, ty, tz], axis=-1)

    def position(self, s):
        s = np.asarray(s, dtype=np.float64)
        if self.c == 0.0:
            return self.x0 + s[..., None] * self.T0
        cs, sn = np.cos(self.c * s), np.sin(self.c * s)
        # 1 - cos written as 2 sin^2(cs/2) to keep small-angle accuracy
        omc = 2.0 * np.sin(0.5 * self.c * s) ** 2
        x = self.x0[0] + (self.T0[0] * sn + self.T0[1] * omc) / self.c
        y = self.x0[1] + (-self.T0[0] * omc + self.T0[1] * sn) / self.c
        z = self.x0[2] + self.T0[2] * s
        return np.stack([x, y, z], axis=-1)
