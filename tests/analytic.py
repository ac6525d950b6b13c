"""Closed forms used as pins (test side only; nothing here is called by oracle/ or the CUDA path).

MacLaurin spheroid: PAPER.md:196-226 (Eq. 6-12) with the two corrections listed in DESIGN.md
("garbled" readings): Eq. 6 carries +A3(a3^2 - z^2); Eq. 10's second term carries 1/(2 a1 e).
Potentials are returned as physical (negative) values: Phi = -(magnitude).
"""
import numpy as np


def maclaurin_A(e):
    """Eq. 7-8."""
    A1 = np.sqrt(1 - e * e) / e ** 3 * np.arcsin(e) - (1 - e * e) / e ** 2
    A3 = 2 / e ** 2 - 2 * np.sqrt(1 - e * e) / e ** 3 * np.arcsin(e)
    return A1, A3


def maclaurin_interior(x, y, z, a1, e, rho=1.0, G=1.0):
    """Corrected Eq. 6: Phi = -pi G rho [2 A1 a1^2 - A1 (x^2+y^2) + A3 (a3^2 - z^2)]; x,y,z from the centre."""
    A1, A3 = maclaurin_A(e)
    a3 = a1 * np.sqrt(1 - e * e)
    return -np.pi * G * rho * (2 * A1 * a1 ** 2 - A1 * (x * x + y * y) + A3 * (a3 ** 2 - z * z))


def maclaurin_exterior(x, y, z, a1, e, rho=1.0, G=1.0):
    """Corrected Eq. 10-12 (lambda = positive root of Eq. 12, a quadratic because a1 = a2)."""
    a3 = a1 * np.sqrt(1 - e * e)
    R2 = x * x + y * y
    z2 = z * z
    # R2/(a1^2+lam) + z2/(a3^2+lam) = 1  ->  lam^2 + (a1^2+a3^2-R2-z2) lam + (a1^2 a3^2 - R2 a3^2 - z2 a1^2) = 0
    b = a1 ** 2 + a3 ** 2 - R2 - z2
    c = a1 ** 2 * a3 ** 2 - R2 * a3 ** 2 - z2 * a1 ** 2
    lam = 0.5 * (-b + np.sqrt(b * b - 4 * c))
    h = a1 * e / np.sqrt(a3 ** 2 + lam)
    at = np.arctan(h)
    mag = 2 * a3 / e ** 2 * np.pi * G * rho * (
        a1 * e * at - (1.0 / (2 * a1 * e)) * (R2 * (at - h / (1 + h * h)) + 2 * z2 * (h - at)))
    return -mag


def sphere_potential(r, R, rho=1.0, G=1.0):
    """Uniform sphere: -2 pi G rho (R^2 - r^2/3) inside, -G M / r outside."""
    r = np.asarray(r, dtype=np.float64)
    M = 4.0 / 3.0 * np.pi * R ** 3 * rho
    inside = -2 * np.pi * G * rho * (R * R - r * r / 3)
    outside = -G * M / np.maximum(r, 1e-300)
    return np.where(r <= R, inside, outside)


CUBE_SELF = 3 * np.log(2 + np.sqrt(3)) - np.pi / 2  # = 2.3800774...: -Phi at the centre of a uniform unit cube of unit mass
