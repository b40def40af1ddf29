"""Host-side formatting of what the kernels wrote: no propagation, no
reduction over trajectories that the device has not already done -- array arithmetic on records and summaries.

  scattering(...)      per-trajectory scattering angle and momentum transfer of the ATOM (Fig. 1):
                       chi = arccos(v_i . v_f / (|v_i| |v_f|)),  q = m_a |v_f - v_i|
  maps(...)            the three (theta, phi) images of Fig. 1: chi, log10(number of bounces), min(q, 0.015 a.u.)
  survival_curve(...)  fraction of complexes still alive after t (Fig. 2) from ia_summary.hist_tlife
  power_law_exponent() slope of log S against log t beyond t_min ("after about 20 us ... a power law")
  heating_scale_uK()   W0^3D of Eq. 3, the energy scale the paper's thresholds are quoted in
"""
from __future__ import annotations

import numpy as np

Q_CLIP_AU = 0.015   # Fig. 1(d) of the paper clips the momentum transfer at 0.015 a.u.


def heating_scale_uK(m_ion_u: float, m_atom_u: float, alpha_au: float, a_x: float, q_x: float,
                     omega_rf_au: float) -> float:
    """Eq. 3 of the paper: W0^3D = 8/(3 pi) (m_a/(m_i+m_a))^(5/3) (m_i^2 w^4 C4 / q_x^2)^(1/3) with the
    secular frequency w ~ Omega_rf/2 sqrt(a_x + q_x^2/2) and C4 = alpha/2, returned as W0/k_B in
    microkelvin.  A scale for reading results ("the threshold energy is consistently 2-3 times" W0);
    nothing in the propagation uses it."""
    me_per_u, kb_eh_per_k = 1822.888486283, 3.1668115634564e-6   # CODATA 2022
    m_i, m_a = m_ion_u * me_per_u, m_atom_u * me_per_u
    w = 0.5 * omega_rf_au * np.sqrt(a_x + 0.5 * q_x * q_x)
    w0 = 8.0 / (3.0 * np.pi) * (m_a / (m_i + m_a)) ** (5.0 / 3.0) * (m_i * m_i * w ** 4 * (0.5 * alpha_au) / (q_x * q_x)) ** (1.0 / 3.0)
    return float(w0 / kb_eh_per_k * 1e6)


def scattering(records: np.ndarray, ic: np.ndarray, m_atom_me: float):
    """records: ia_record array [n]; ic: the launch's ic_dump [n, 14] (or ia_generate's output); m_atom_me: atom mass in
    electron masses (ia_get_derived()['m_a']).  Returns (chi [rad], q [a.u.])."""
    v_i = np.asarray(ic)[:, 9:12]
    v_f = np.asarray(records["va_f"])
    ni, nf = np.linalg.norm(v_i, axis=1), np.linalg.norm(v_f, axis=1)
    cosang = np.clip(np.sum(v_i * v_f, axis=1) / (ni * nf), -1.0, 1.0)
    return np.arccos(cosang), m_atom_me * np.linalg.norm(v_f - v_i, axis=1)


def maps(records: np.ndarray, ic: np.ndarray, m_atom_me: float, n_theta: int, n_phi: int) -> dict:
    """The (theta, phi) images of a GRID launch (row = theta index, column = phi index)."""
    chi, q = scattering(records, ic, m_atom_me)
    shape = (int(n_theta), int(n_phi))
    n_coll = np.asarray(records["n_coll"]).astype(np.float64)
    return {"scattering_angle": chi.reshape(shape),
            "log10_bounces": np.log10(np.maximum(n_coll, 1.0)).reshape(shape),
            "momentum_transfer_clipped": np.minimum(q, Q_CLIP_AU).reshape(shape),
            "complex": (np.asarray(records["n_coll"]) >= 2).reshape(shape)}


def life_bin_edges(T_rf: float, nbins: int = 64) -> np.ndarray:
    """Lower edges of ia_summary.hist_tlife's bins 1..nbins-1 and the upper edge of the last regular bin, in a.u.:
    bin b holds 2^((b-8)/4) <= t_life/T_rf < 2^((b-7)/4); bin 0 also collects everything shorter, the last bin
    everything longer."""
    return T_rf * 2.0 ** ((np.arange(1, nbins + 1) - 8) / 4.0)


def survival_curve(summary, T_rf: float):
    """(t [a.u.], S): S[k] = fraction of the launch's complexes with t_life >= t[k], at the bin edges of hist_tlife."""
    h = np.asarray(summary["hist_tlife"], dtype=np.float64)
    total = h.sum()
    edges = life_bin_edges(T_rf, len(h))[:-1]          # lower edges of bins 1 .. nbins-1
    if total == 0:
        return edges, np.zeros(len(edges))
    alive = total - np.cumsum(h)[:-1]                  # complexes in bins above bin k
    return edges, alive / total


def power_law_exponent(t: np.ndarray, S: np.ndarray, t_min: float, t_max: float = np.inf) -> float:
    """Least-squares slope of log S against log t over t_min <= t <= t_max where S > 0."""
    t, S = np.asarray(t, dtype=np.float64), np.asarray(S, dtype=np.float64)
    m = (t >= t_min) & (t <= t_max) & (S > 0)
    if m.sum() < 2:
        return float("nan")
    return float(np.polyfit(np.log(t[m]), np.log(S[m]), 1)[0])
