"""Helpers for the tests: closed forms from the MPC literature and brute-force numpy re-computations.
None of this is imported by the product or by oracle/."""
import numpy as np


def srd_viscosity(nbar, h, alpha_deg, kT=1.0, m=1.0, a=1.0, conserve_L=False):
    """Kinematic viscosity of the 3-D SRD fluid: kinetic + collisional part (refs [31],[32],[68] of the
    paper, review [1]); SURVEY.md section 8(c). Returns (nu_kin, nu_col)."""
    al = np.deg2rad(alpha_deg)
    fac = nbar - 1.0 + np.exp(-nbar)
    nu_kin = (kT * h / m) * (5.0 * nbar / (fac * (4.0 - 2.0 * np.cos(al) - 2.0 * np.cos(2 * al))) - 0.5)
    if conserve_L:
        nu_col = (a * a / h) * (1.0 - np.cos(al)) * (nbar - 7.0 / 5.0) / (36.0 * nbar)
    else:
        nu_col = (a * a / h) * (1.0 - np.cos(al)) * fac / (18.0 * nbar)
    return nu_kin, nu_col


def cell_sums(key, nkeys, *cols):
    """Brute-force per-key sums of the given per-particle columns (float64)."""
    return [np.bincount(key, weights=np.asarray(c, np.float64), minlength=nkeys) for c in cols]


def by_id(ids, *arrs):
    order = np.argsort(ids, kind="stable")
    return [np.asarray(a)[order] for a in arrs]


def poiseuille_startup(zc, t, g, nu, Lz, nmax=199):
    """v_x(z,t) of a fluid at rest at t=0 between no-slip walls at 0 and Lz under acceleration g."""
    v = g / (2 * nu) * zc * (Lz - zc)
    for n in range(1, nmax + 1, 2):
        v -= 4 * g * Lz**2 / (nu * n**3 * np.pi**3) * np.sin(n * np.pi * zc / Lz) * np.exp(-nu * n**2 * np.pi**2 * t / Lz**2)
    return v
