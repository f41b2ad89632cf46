"""fp64 ORACLE for the numerical integrators of the transport loop.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as obem_ref.c): imports nothing from paper_2110_09214_b200 and
shares no code with the CUDA path.  Plain numpy, one statement per sub-step, in the order of the published schemes.

PAPER.md:300-306, section 3.2.5: "Two stepper algorithms have been implemented": the basic Euler algorithm (one
field evaluation per time step) and PEFRL [18] (Omelyan, Mryglod, Folk, Comput. Phys. Commun. 146 (2002) 188:
the position-extended Forest-Ruth-like scheme, 4th order, symplectic, time reversible).

Equations of motion (non-relativistic; the paper transports eV-scale electrons and thermal ions):
    dx/dt = v,   dv/dt = (q/m) E(x)
`field(x)` is any callable x[n,3] float64 -> E[n,3] float64; the tests pass closed-form fields to pin the schemes
and the fp64 field oracle (oracle/ref.py) for parity with the GPU path.

DESIGN.md reading A17: the paper counts "5 field evaluations" per PEFRL step; the published scheme has 5 position
sub-steps and 4 velocity sub-steps, i.e. 4 force evaluations.  This oracle follows the published scheme.
"""
from __future__ import annotations

import numpy as np

# Omelyan et al. 2002, Eq. (20)-(22): the optimised parameters of the position-extended Forest-Ruth-like scheme
PEFRL_XI = 0.1786178958448091
PEFRL_LAMBDA = -0.2123418310626054
PEFRL_CHI = -0.6626458266981849e-1


def euler_step(x, v, q_over_m, h, field):
    """Basic (explicit, forward) Euler: both updates use the state at the START of the step.
        x_{n+1} = x_n + h v_n
        v_{n+1} = v_n + h (q/m) E(x_n)
    Returns (x_new, v_new, E(x_n))."""
    x = np.asarray(x, dtype=np.float64)
    v = np.asarray(v, dtype=np.float64)
    qm = np.asarray(q_over_m, dtype=np.float64).reshape(-1, 1)
    e = np.asarray(field(x), dtype=np.float64)
    x_new = x + h * v
    v_new = v + h * qm * e
    return x_new, v_new, e


def pefrl_step(x, v, q_over_m, h, field):
    """PEFRL, one step h (Omelyan et al. 2002, the velocity-Verlet-like ordering x v x v x v x v x):
        x += xi h v
        v += (1 - 2 lambda) h/2 a(x)
        x += chi h v
        v += lambda h a(x)
        x += (1 - 2 (chi + xi)) h v
        v += lambda h a(x)
        x += chi h v
        v += (1 - 2 lambda) h/2 a(x)
        x += xi h v
    with a(x) = (q/m) E(x).  Returns (x_new, v_new)."""
    x = np.array(x, dtype=np.float64)
    v = np.array(v, dtype=np.float64)
    qm = np.asarray(q_over_m, dtype=np.float64).reshape(-1, 1)
    xi, lam, chi = PEFRL_XI, PEFRL_LAMBDA, PEFRL_CHI
    x = x + xi * h * v
    v = v + (1.0 - 2.0 * lam) * 0.5 * h * qm * np.asarray(field(x), dtype=np.float64)
    x = x + chi * h * v
    v = v + lam * h * qm * np.asarray(field(x), dtype=np.float64)
    x = x + (1.0 - 2.0 * (chi + xi)) * h * v
    v = v + lam * h * qm * np.asarray(field(x), dtype=np.float64)
    x = x + chi * h * v
    v = v + (1.0 - 2.0 * lam) * 0.5 * h * qm * np.asarray(field(x), dtype=np.float64)
    x = x + xi * h * v
    return x, v
