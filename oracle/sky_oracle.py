"""sky_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Oracle of two small pieces of SURVEY.md section 8(f) NEXT-4, plain numpy in fp64.  Shares no code with
paper_2210_07912_b200 and never imports it.

1. Rotated detector-network-frame sky coordinates (section III): "a coordinate system for the sky where the
   nominal north pole corresponds to a vector connecting two of the interferometers".  The paper gives no formula; readings
   (F1-F2):
     F1  Earth-fixed unit vector of a sky position, as in the delay of step a3:
             n(ra, dec) = (cos dec cos(ra - gmst), cos dec sin(ra - gmst), sin dec).
     F2  frame (columns of R):  z' = (r_b - r_a) / |r_b - r_a|;  x' = (e_z x z') / |e_z x z'| (e_z the Earth's axis; if the
         baseline is parallel to it, x' = e_x);  y' = z' x x'.  Network coordinates (lambda, beta), beta the nominal
         declination:  n = R (cos beta cos lambda, cos beta sin lambda, sin beta).
   A rotation preserves solid angle, so an isotropic prior is cos(beta)/(4 pi) in the new coordinates as well.
2. rho_guess, Eq. (D7) under reading A14 of SURVEY.md (the printed ratio U / max|Q|^2 is inverted: maximising
   Eq. (D5) over the distance scale gives Q^2 / U):
             (2.3 rho_guess)^2 = sum_k sum_lm max_t |Q_{k,lm}(t)|^2 / |U_{k,lm,lm}|,   terms with U_{k,lm,lm} = 0 left out.

Pins: tests/test_next4_oracle_pins.py (P27 pole = baseline and orthonormal frame, P28 the a-b delay difference depends on
beta only and equals |r_b - r_a| sin(beta) / c, P29 round trip and solid angle, P30 a delayed noise-free single-mode signal
gives rho_guess = rho / 2.3, P31 brute force).
"""
from __future__ import annotations

import numpy as np

__all__ = ["sky_unit_vector", "network_frame", "network_to_radec", "radec_to_network", "rho_guess"]


def sky_unit_vector(ra, dec, gmst: float) -> np.ndarray:
    """F1: [n][3] Earth-fixed unit vectors."""
    ra, dec = np.asarray(ra, dtype=np.float64), np.asarray(dec, dtype=np.float64)
    return np.stack([np.cos(dec) * np.cos(ra - gmst), np.cos(dec) * np.sin(ra - gmst), np.sin(dec)], axis=-1)


def network_frame(loc_a, loc_b) -> np.ndarray:
    """F2: R [3][3], columns x', y', z' (z' along the baseline from detector a to detector b)."""
    a, b = np.asarray(loc_a, dtype=np.float64), np.asarray(loc_b, dtype=np.float64)
    z = (b - a) / np.linalg.norm(b - a)
    x = np.cross([0.0, 0.0, 1.0], z)
    if np.linalg.norm(x) < 1e-12:
        x = np.array([1.0, 0.0, 0.0])
    x = x / np.linalg.norm(x)
    y = np.cross(z, x)
    return np.stack([x, y, z], axis=1)


def network_to_radec(lam, beta, R, gmst: float):
    """(ra in [0, 2 pi), dec) of network coordinates (lambda, beta)."""
    lam, beta = np.asarray(lam, dtype=np.float64), np.asarray(beta, dtype=np.float64)
    v = np.stack([np.cos(beta) * np.cos(lam), np.cos(beta) * np.sin(lam), np.sin(beta)], axis=-1)
    n = v @ np.asarray(R, dtype=np.float64).T
    dec = np.arcsin(np.clip(n[..., 2], -1.0, 1.0))
    ra = np.mod(np.arctan2(n[..., 1], n[..., 0]) + gmst, 2.0 * np.pi)
    return ra, dec


def radec_to_network(ra, dec, R, gmst: float):
    """(lambda in [0, 2 pi), beta) of equatorial coordinates: the inverse of network_to_radec."""
    v = sky_unit_vector(ra, dec, gmst) @ np.asarray(R, dtype=np.float64)
    beta = np.arcsin(np.clip(v[..., 2], -1.0, 1.0))
    lam = np.mod(np.arctan2(v[..., 1], v[..., 0]), 2.0 * np.pi)
    return lam, beta


def rho_guess(Q, U) -> float:
    """Eq. (D7) with reading A14 for one intrinsic point: Q [K][M][n_t], U [K][M][M] complex128."""
    Q, U = np.asarray(Q, dtype=np.complex128), np.asarray(U, dtype=np.complex128)
    total = 0.0
    for k in range(Q.shape[0]):
        for a in range(Q.shape[1]):
            u = abs(U[k, a, a])
            if u > 0.0:
                total += float(np.max(np.abs(Q[k, a]) ** 2)) / u
    return float(np.sqrt(total) / 2.3)
