"""Pin P7 (north_star oracle check 4): the whole box run of
configs[0] (Golovin kernel, exponential initial spectrum) against the analytic solution of the
Smoluchowski equation at t = 1200, 2400, 3600 s, on the paper's 31 log-spaced radius bins
(PAPER.md:70-71).  The closed form is evaluated here with scipy (independent of oracle/)."""
import json
import math
import os

import numpy as np
from scipy.special import ive

import oracle
import sdm_workloads as W

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
RHO_W = 1000.0  # kg m^-3


def golovin_number_density(v, t, n0, v0, b):
    """n(v, t) [m^-3 per m^3 of droplet volume] for K = b (v + v'), n(v,0) = n0/v0 exp(-v/v0)."""
    x = v / v0
    tau = 1.0 - math.exp(-n0 * b * v0 * t)
    st = math.sqrt(tau)
    z = 2.0 * x * st
    # ive(1, z) = exp(-z) I1(z); scipy returns nan beyond z ~ 1e9, where the large-argument form
    # 1/sqrt(2 pi z) is exact to double precision.  exponent: z - (1+tau) x = -x (1 - sqrt(tau))^2.
    zs = np.minimum(z, 1e8)
    i1 = np.where(z > 1e8, 1.0 / np.sqrt(2.0 * math.pi * np.maximum(z, 1e-300)), ive(1, zs))
    return (n0 / v0) * (1.0 - tau) / (x * st) * i1 * np.exp(-x * (1.0 - st) ** 2)


def analytic_bin_mass_density(edges_r, t, n0, v0, b, sub=400):
    """bin-averaged g(ln r) = 3 rho v^2 n(v,t)  [kg m^-3 per unit ln r] on each bin."""
    out = np.zeros(len(edges_r) - 1)
    for i in range(len(out)):
        lr = np.linspace(math.log(edges_r[i]), math.log(edges_r[i + 1]), sub)
        r = np.exp(lr)
        v = 4.0 / 3.0 * math.pi * r ** 3
        g = 3.0 * RHO_W * v * v * golovin_number_density(v, t, n0, v0, b)
        out[i] = np.trapezoid(g, lr) / (lr[-1] - lr[0])
    return out


def test_closed_form_reproduces_printed_anchors():
    g = json.load(open(os.path.join(GOLDEN, "golovin_analytic.json")))
    n0, v0, b = W.N0_PER_M3, W.V0, 1500.0
    assert abs(n0 * b * v0 - g["n0_b_v0_per_s"]) < 2e-8
    for t, frac, rpk, gpk in zip(g["t_s"], g["number_fraction_N_over_n0"], g["mass_density_peak_radius_um"],
                                 g["mass_density_peak_g_per_m3_per_lnr"]):
        tau = 1.0 - math.exp(-n0 * b * v0 * t)
        assert abs((1.0 - tau) / frac - 1.0) < 2e-5
        # total number from integrating the closed-form density agrees with 1 - tau
        lr = np.linspace(math.log(1e-7), math.log(5e-2), 20000)
        v = 4.0 / 3.0 * math.pi * np.exp(lr) ** 3
        nd = golovin_number_density(v, t, n0, v0, b)
        assert abs(np.trapezoid(nd * 3.0 * v, lr) / n0 / (1.0 - tau) - 1.0) < 1e-3
        gl = 3.0 * RHO_W * v * v * nd * 1e3      # g m^-3 per ln r
        k = int(np.argmax(gl))
        assert abs(math.exp(lr[k]) * 1e6 / rpk - 1.0) < 5e-3
        assert abs(gl[k] / gpk - 1.0) < 5e-3


def test_box_run_against_golovin_solution():
    g = json.load(open(os.path.join(GOLDEN, "golovin_analytic.json")))
    tol = g["tolerances"]
    w = W.cfg0()                                     # n_sd = 2^13, dt = 1 s, dV = 1e6 m^3, b = 1500 /s
    assert w.n_sd == 2 ** 13 and w.n_cell == 1
    kp = oracle.golovin(w.b)
    edges = np.logspace(np.log10(10e-6), np.log10(5e3 * 1e-6), num=32)
    dlnr = np.diff(np.log(edges))
    n0, v0 = W.N0_PER_M3, W.V0
    mass0 = float(np.sum(w.xi.astype(np.float64) * w.v)) * RHO_W / w.dV
    assert abs(mass0 - 1.0e-3) / 1.0e-3 < 2e-3       # rho_w n0 v0 = 1.000 g m^-3
    step = 0
    n_sd = w.n_sd
    for t in g["t_s"]:
        n_sd = oracle.run(w.xi, w.v, w.cell_id, 1, w.dt, w.dV, kp, w.seed, step, t - step, n_sd=n_sd)
        step = t
        tau = 1.0 - math.exp(-n0 * w.b * v0 * t)
        n_sim = float(w.xi.sum()) / w.dV
        assert abs(n_sim / (n0 * (1.0 - tau)) - 1.0) < tol["number_ratio"], (t, n_sim / (n0 * (1 - tau)))
        r = (w.v / (4.0 / 3.0 * math.pi)) ** (1.0 / 3.0)
        mass = w.xi.astype(np.float64) * w.v * RHO_W / w.dV
        g_sim = np.histogram(r, bins=edges, weights=mass)[0] / dlnr
        g_ana = analytic_bin_mass_density(edges, t, n0, v0, w.b)
        assert abs(int(np.argmax(g_sim)) - int(np.argmax(g_ana))) <= tol["peak_bin"]
        f_sim = g_sim * dlnr / mass0
        f_ana = g_ana * dlnr / mass0
        assert np.abs(f_sim - f_ana).sum() < tol["l1_mass_fraction"], (t, np.abs(f_sim - f_ana).sum())
    # mass conserved over the whole run to rounding (R22)
    mass1 = float(np.sum(w.xi.astype(np.float64) * w.v)) * RHO_W / w.dV
    assert abs(mass1 - mass0) / mass0 < 1e-11
