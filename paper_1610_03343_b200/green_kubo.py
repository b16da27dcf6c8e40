"""Caller-side post-processing of md_nve_heat_run's J(t) series: heat-current autocorrelation and the running
Green-Kubo integral (the application of the paper's Ref. [27]).  Plain numpy on the few
numbers per sample the GPU path returns; nothing of the force path runs here.

    kappa(t) = 1 / (3 kB T^2 V) * integral_0^t <J(0) . J(t')> dt'        (isotropic average of the three components)
"""
from __future__ import annotations

import numpy as np

KB_EV_PER_K = 8.617333262e-5
# 1 eV / (fs A K) in W / (m K): 1.602176634e-19 J / (1e-15 s * 1e-10 m * K)
EV_PER_FS_A_K_IN_W_PER_M_K = 1.602176634e6


def hcacf(J, max_lag):
    """<J(0).J(t)> / 3 for lags 0..max_lag-1 from a series J[ns][3] (time-origin average)."""
    J = np.asarray(J, dtype=np.float64)
    ns = J.shape[0]
    out = np.zeros(max_lag)
    for lag in range(max_lag):
        out[lag] = (J[:ns - lag] * J[lag:]).sum() / (3.0 * (ns - lag))
    return out


def running_kappa(J, dt_sample_fs, T_K, volume_A3, max_lag):
    """Running thermal conductivity in W/(m K) from the total heat current series (eV A/fs)."""
    c = hcacf(J, max_lag)
    integral = np.concatenate([[0.0], np.cumsum(0.5 * (c[1:] + c[:-1]) * dt_sample_fs)])
    return integral / (KB_EV_PER_K * T_K ** 2 * volume_A3) * EV_PER_FS_A_K_IN_W_PER_M_K
