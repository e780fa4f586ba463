"""Seeded synthetic material models: per-element density rho and phase velocity c (piecewise
constant per cell).  Plain arrays only."""
import numpy as np


def centroid_of_elements(etov, vx):
    return vx[etov].mean(axis=1)


def two_layer_model(etov, vx, z_interface, c_top, rho_top, c_bot, rho_bot):
    """Two half-spaces separated by the plane z = z_interface (z = depth), chosen by the element
    centroid (shape of the paper's validation model)."""
    zc = centroid_of_elements(etov, vx)[:, 2]
    top = zc < z_interface
    c = np.where(top, c_top, c_bot).astype(np.float64)
    rho = np.where(top, rho_top, rho_bot).astype(np.float64)
    return rho, c


def smooth_random_field(etov, vx, lengths, lo, hi, seed, grid=(48, 48, 24), sigma_cells=3.0):
    """Gaussian-filtered seeded noise on a regular grid, mapped affinely to [lo, hi] and sampled at
    the element centroids (nearest grid cell)."""
    from scipy.ndimage import gaussian_filter

    rng = np.random.default_rng(seed)
    gx, gy, gz = grid
    noise = rng.standard_normal((gz, gy, gx))
    f = gaussian_filter(noise, sigma=sigma_cells, mode="reflect")
    f = (f - f.min()) / (f.max() - f.min())
    cen = centroid_of_elements(etov, vx)
    ix = np.clip((cen[:, 0] / lengths[0] * gx).astype(np.int64), 0, gx - 1)
    iy = np.clip((cen[:, 1] / lengths[1] * gy).astype(np.int64), 0, gy - 1)
    iz = np.clip((cen[:, 2] / lengths[2] * gz).astype(np.int64), 0, gz - 1)
    return lo + (hi - lo) * f[iz, iy, ix]


def planted_reflector_model(etov, vx, lengths, c_background, depth0, dip_x, dip_y, factor):
    """`true` model for the observed data of config 4: the background velocity multiplied by
    `factor` below the gently dipping plane z = depth0 + dip_x*(x-Lx/2) + dip_y*(y-Ly/2)."""
    cen = centroid_of_elements(etov, vx)
    plane = depth0 + dip_x * (cen[:, 0] - 0.5 * lengths[0]) + dip_y * (cen[:, 1] - 0.5 * lengths[1])
    return np.where(cen[:, 2] > plane, c_background * factor, c_background)
