"""Seeded synthetic receiver gathers d_r(t) (an INPUT of the backward RTM phase): one smooth pulse
per receiver, delayed by the source-receiver distance, with a seeded amplitude.  Stands in for recorded data where a
test or a stored expected value must not depend on a forward run (the imaging arithmetic does not care where d_r
comes from).  Plain arrays only; none of the method's arithmetic."""
import numpy as np


def synthetic_gather(xr, x0, nsamp, dt, seed, f0=15.0, c0=2.0, t_shift=0.02):
    xr = np.asarray(xr, dtype=np.float64).reshape(-1, 3)
    rng = np.random.default_rng(seed)
    amp = rng.uniform(0.5, 1.5, xr.shape[0]) * rng.choice([-1.0, 1.0], xr.shape[0])
    delay = t_shift + np.linalg.norm(xr - np.asarray(x0, dtype=np.float64)[None, :], axis=1) / c0
    t = dt * np.arange(nsamp)
    a = (np.pi * f0 * (t[None, :] - delay[:, None])) ** 2
    return amp[:, None] * (1.0 - 2.0 * a) * np.exp(-a)
