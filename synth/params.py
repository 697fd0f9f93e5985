"""Per-region material parameters (a plain container, SI units; Fig. 1)."""
from dataclasses import dataclass, field
import numpy as np


def _arr(x, n, shape=()):
    a = np.zeros((n,) + shape, dtype=np.float64)
    a[...] = x
    return a


@dataclass
class Params:
    """Look-up tables indexed by region id + uniform applied field.

    exch_scale: None (S = 1 everywhere) or the lower-triangular table
    S[i(i+1)/2 + j], i >= j, of Eq. 9.
    """
    nregions: int = 1
    Msat: np.ndarray = None      # A/m
    Aex: np.ndarray = None       # J/m
    alpha: np.ndarray = None
    Ku1: np.ndarray = None       # J/m^3
    Ku2: np.ndarray = None
    anisU: np.ndarray = None     # (nregions, 3)
    Kc1: np.ndarray = None
    Kc2: np.ndarray = None
    Kc3: np.ndarray = None
    anisC1: np.ndarray = None    # (nregions, 3)
    anisC2: np.ndarray = None
    B_ext: np.ndarray = field(default_factory=lambda: np.zeros(3))
    exch_scale: np.ndarray = None
    gamma_LL: float = 1.7595e11  # rad/(T s)

    @staticmethod
    def uniform(nregions=1, Msat=0.0, Aex=0.0, alpha=0.0, Ku1=0.0, Ku2=0.0, anisU=(0, 0, 1),
                Kc1=0.0, Kc2=0.0, Kc3=0.0, anisC1=(1, 0, 0), anisC2=(0, 1, 0),
                B_ext=(0, 0, 0), exch_scale=None, gamma_LL=1.7595e11):
        n = nregions
        return Params(nregions=n, Msat=_arr(Msat, n), Aex=_arr(Aex, n), alpha=_arr(alpha, n),
                      Ku1=_arr(Ku1, n), Ku2=_arr(Ku2, n), anisU=_arr(anisU, n, (3,)),
                      Kc1=_arr(Kc1, n), Kc2=_arr(Kc2, n), Kc3=_arr(Kc3, n),
                      anisC1=_arr(anisC1, n, (3,)), anisC2=_arr(anisC2, n, (3,)),
                      B_ext=np.asarray(B_ext, dtype=np.float64),
                      exch_scale=None if exch_scale is None else np.asarray(exch_scale, dtype=np.float64),
                      gamma_LL=gamma_LL)
