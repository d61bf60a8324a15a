"""Error measures shared by the GPU parity tests (test infrastructure; no method arithmetic)."""
import numpy as np

# velocity order of the 14 conserved moments: rho | rho u_i | U_ij | U_ijj | U_iijj
ORDER14 = np.array([0, 1, 1, 1, 2, 2, 2, 2, 2, 2, 3, 3, 3, 4])


def moment_errors(Ug, Uo):
    """R22: per moment, max |U_gpu - U_or| / max |U_or| over the given cells; a
    moment that is identically zero in the oracle must be identically zero on the GPU."""
    e = np.zeros(Uo.shape[0])
    for m in range(Uo.shape[0]):
        scale = np.abs(Uo[m]).max()
        if scale == 0.0:
            assert np.all(Ug[m] == 0.0), f"moment {m}: oracle identically 0, GPU not"
        else:
            e[m] = np.abs(Ug[m] - Uo[m]).max() / scale
    return e


def window_errors(Ug, Uo):
    """Per-moment error of a WINDOW of a 14-moment field, scaled by the window's own data only.
    The yardstick of moment m is the larger of its own maximum in the window and rho c^n, with rho the
    window's largest density, c^2 = max tr(U_ij)/(3 rho) (thermal + bulk speed) and n the moment's order
    in velocity: in gas at rest the odd moments are differences of O(rho c^n) fluxes and their own
    magnitude (1e-8 rho c in the perturbed background) says nothing about the arithmetic's accuracy."""
    rho = Uo[0].max()
    c = np.sqrt(((Uo[4] + Uo[7] + Uo[9]) / (3.0 * Uo[0])).max())
    e = np.zeros(14)
    for m in range(14):
        own = np.abs(Uo[m]).max()
        if own == 0.0:
            assert np.all(Ug[m] == 0.0), f"moment {m}: oracle identically 0, GPU not"
            continue
        e[m] = np.abs(Ug[m] - Uo[m]).max() / max(own, rho * c ** ORDER14[m])
    return e
