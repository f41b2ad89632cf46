"""fp64 ORACLE for the Shockley-Ramo signal sum (section 3.4, Eq 3.13).

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as obem_ref.c): imports nothing from paper_2110_09214_b200 and
shares no code with the CUDA path.  Plain numpy; the definition written out.

    i(t) = sum_p q_p v_p(t) . E_w(r_p)                                                     (3.13)

E_w is the weighting field of one read-out electrode (that electrode at 1 V, all others grounded; units 1/m when the
potential is taken as dimensionless, V/m as the library returns it for 1 V), evaluated at the particle.  "the signals
created by each type are generated separately": the sum is returned per sign of q.
"""
from __future__ import annotations

import numpy as np


def ramo_current(q, vel, ew):
    """q [N] charges [C], vel [N,3] velocities [m/s], ew [K,N,3] weighting field of electrode k at particle p [V/m].
    Returns [K,2] float64: column 0 = the particles with q < 0 (electrons), column 1 = those with q > 0 (ions);
    amperes for a weighting potential of 1 V.  Plain left-to-right fp64 sums in index order."""
    q = np.asarray(q, dtype=np.float64)
    vel = np.asarray(vel, dtype=np.float64)
    ew = np.asarray(ew, dtype=np.float64)
    assert vel.shape == (q.shape[0], 3) and ew.shape[1:] == (q.shape[0], 3)
    out = np.zeros((ew.shape[0], 2), dtype=np.float64)
    for k in range(ew.shape[0]):
        for p in range(q.shape[0]):
            term = q[p] * (vel[p, 0] * ew[k, p, 0] + vel[p, 1] * ew[k, p, 1] + vel[p, 2] * ew[k, p, 2])
            if q[p] < 0.0:
                out[k, 0] += term
            elif q[p] > 0.0:
                out[k, 1] += term
    return out
