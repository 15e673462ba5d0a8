"""Plain numpy / scipy (float64) definition of the detector-resolution broadening of a pulse-height spectrum
 -- test infrastructure only, like the rest of oracle/: the counts of every bin are spread as a
Gaussian centred on the bin middle with FWHM(E)^2 = a + b E + c E^2 (E in MeV); bin 0 also takes the mass below 0 and
the last slot the overflow counts and the mass above e_max, so the total is conserved."""
import numpy as np
from scipy.special import erf


def broaden(spectrum, e_max_mev, a, b=0.0, c=0.0):
    s = np.asarray(spectrum, dtype=np.float64)
    n = len(s) - 1
    de = e_max_mev / n
    centre = (np.arange(n) + 0.5) * de
    fwhm2 = a + b * centre + c * centre * centre
    sigma = np.sqrt(fwhm2) / 2.3548200450309493
    lo = np.concatenate([[-1e300], np.arange(1, n) * de, [e_max_mev]])          # lower edges of the n + 1 outputs
    hi = np.concatenate([np.arange(1, n + 1) * de, [1e300]])
    out = np.zeros(n + 1)
    out[n] = s[n]
    for i in np.nonzero(s[:n])[0]:
        z = sigma[i] * np.sqrt(2.0)
        out += s[i] * 0.5 * (erf((hi - centre[i]) / z) - erf((lo - centre[i]) / z))
    return out
