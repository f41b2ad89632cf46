"""Error metrics of the GPU-vs-oracle parity tests (reading A6; BASELINE.json north_star).

For E:   rel-L2 = sqrt(sum_t ||dE_t||^2 / sum_t ||E_ref,t||^2)            bar 2e-5
         per-target max of ||dE_t|| / ||E_ref,t||                         bar 1e-3
For phi: rel-L2 over all phi                                              bar 2e-5
         per-target |dphi| / max(|phi_ref|, PHI_FLOOR * rms(phi_ref))     bar 1e-3,  PHI_FLOOR = 1e-2
(phi changes sign inside a neutral cloud: it is a small difference of two large sums, the electrons' and the
ions', so "relative to |phi_t|" is meaningless where phi_t crosses zero.  A target whose |phi| is below 1 % of the rms
is measured against 1 % of the rms.  Round 1 needed a floor of 10 % of the rms; the fp64 running sums and the short
fp32 phi chains of round 2 brought the measured worst case at a 1 % floor to 5e-4 (N-body part
of config 2).  SURVEY.md's first proposal, 0.1 % of the rms, asks for an absolute error of 1e-6 rms on sums whose
terms add up to ~50 rms in fp32: section 7 gives the bound that says why that is out of reach.)
"""
import numpy as np

TOL_REL_L2 = 2e-5
TOL_MAX_REL = 1e-3
PHI_FLOOR = 1e-2


def field_errors(got, ref):
    """got [T,4] (any float dtype), ref [T,4] float64 -> dict of the four numbers."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape and got.shape[1] == 4
    if got.shape[0] == 0:
        return {"E_rel_l2": 0.0, "E_max_rel": 0.0, "phi_rel_l2": 0.0, "phi_max_rel": 0.0}
    dE = got[:, :3] - ref[:, :3]
    nE = np.linalg.norm(ref[:, :3], axis=1)
    ndE = np.linalg.norm(dE, axis=1)
    e_l2 = float(np.sqrt((ndE ** 2).sum() / max((nE ** 2).sum(), 1e-300)))
    floor_e = 1e-6 * float(np.sqrt((nE ** 2).mean()))          # guards an exactly-zero reference field
    e_max = float((ndE / np.maximum(nE, max(floor_e, 1e-300))).max())
    dphi = got[:, 3] - ref[:, 3]
    rms = float(np.sqrt((ref[:, 3] ** 2).mean()))
    p_l2 = float(np.sqrt((dphi ** 2).sum() / max((ref[:, 3] ** 2).sum(), 1e-300)))
    p_max = float((np.abs(dphi) / np.maximum(np.abs(ref[:, 3]), max(PHI_FLOOR * rms, 1e-300))).max())
    return {"E_rel_l2": e_l2, "E_max_rel": e_max, "phi_rel_l2": p_l2, "phi_max_rel": p_max}


def assert_parity(got, ref, what=""):
    e = field_errors(got, ref)
    assert np.isfinite(np.asarray(got)).all(), "%s: non-finite GPU output" % what
    assert e["E_rel_l2"] <= TOL_REL_L2, "%s: E rel-L2 %.3e > %.1e" % (what, e["E_rel_l2"], TOL_REL_L2)
    assert e["E_max_rel"] <= TOL_MAX_REL, "%s: E per-target max rel %.3e > %.1e" % (what, e["E_max_rel"], TOL_MAX_REL)
    assert e["phi_rel_l2"] <= TOL_REL_L2, "%s: phi rel-L2 %.3e > %.1e" % (what, e["phi_rel_l2"], TOL_REL_L2)
    assert e["phi_max_rel"] <= TOL_MAX_REL, "%s: phi per-target max rel %.3e > %.1e" % (what, e["phi_max_rel"],
                                                                                      TOL_MAX_REL)
    return e
