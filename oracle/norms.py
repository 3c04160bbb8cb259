"""The norm parity is measured in.  Test infrastructure."""
import numpy as np


def parity_errors(Ua, Ub, gamma):
    """Per-variable normalised max-norm difference."""
    rho = Ub[:, 0]
    m2 = Ub[:, 1] ** 2 + Ub[:, 2] ** 2 + Ub[:, 3] ** 2
    P = (gamma - 1.0) * (Ub[:, 4] - 0.5 * m2 / rho)
    cs = np.sqrt(gamma * np.abs(P) / rho)
    scale_m = (np.sqrt(m2) + rho * cs).max()
    scales = [np.abs(rho).max(), scale_m, scale_m, scale_m, np.abs(Ub[:, 4]).max()]
    return np.array([np.abs(Ua[:, v] - Ub[:, v]).max() / scales[v] for v in range(5)])
