"""Closed-form dam-break solutions (textbook: Stoker 1957, Ritter 1892; Toro 2001 ch. 6).

Independent of oracle/ and of the CUDA path: used to pin the oracle and to check the GPU path.
"""
import numpy as np


def stoker(hL, hR, g=9.81):
    """Plateau depth/velocity and wave speeds of the wet-wet dam break (hL > hR > 0)."""
    aL = np.sqrt(g * hL)

    def f(hm):  # rarefaction velocity minus shock velocity
        return 2.0 * (aL - np.sqrt(g * hm)) - (hm - hR) * np.sqrt(g * (hm + hR) / (2.0 * hm * hR))

    lo, hi = hR, hL
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if f(mid) > 0.0:
            lo = mid
        else:
            hi = mid
    hm = 0.5 * (lo + hi)
    um = 2.0 * (aL - np.sqrt(g * hm))
    s = hm * um / (hm - hR)
    return dict(hm=hm, um=um, shock=s, head=-aL, tail=um - np.sqrt(g * hm))


def stoker_profile(xi, hL, hR, g=9.81):
    """h, u at similarity coordinate xi = (x - x_dam) / t."""
    p = stoker(hL, hR, g)
    aL = np.sqrt(g * hL)
    xi = np.asarray(xi, dtype=np.float64)
    h = np.where(xi < p["head"], hL,
                 np.where(xi < p["tail"], (2.0 * aL - xi) ** 2 / (9.0 * g),
                          np.where(xi < p["shock"], p["hm"], hR)))
    u = np.where(xi < p["head"], 0.0,
                 np.where(xi < p["tail"], 2.0 / 3.0 * (aL + xi),
                          np.where(xi < p["shock"], p["um"], 0.0)))
    return h, u


def ritter_profile(xi, h0, g=9.81):
    a0 = np.sqrt(g * h0)
    xi = np.asarray(xi, dtype=np.float64)
    h = np.where(xi < -a0, h0, np.where(xi < 2.0 * a0, (2.0 * a0 - xi) ** 2 / (9.0 * g), 0.0))
    u = np.where(xi < -a0, 0.0, np.where(xi < 2.0 * a0, 2.0 / 3.0 * (a0 + xi), 0.0))
    return h, u
